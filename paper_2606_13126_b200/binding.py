"""Thin ctypes binding over libminipic.so - argument marshalling only.

Every function here has the name of the C entry point it forwards to (include/minipic.h); every
step of the hot path runs inside the library's CUDA kernels.  PyTorch appears only as the owner of
device memory and streams (``tensor.data_ptr()``, ``torch.cuda.current_stream()``).

There is no fallback: ``lib()`` raises if the shared library has not been built
(``python -m paper_2606_13126_b200.build``), and nothing here imports ``oracle/``.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libminipic.so")

MINIPIC_OK = 0
MINIPIC_ERR_INVALID_ARG = 1
MINIPIC_ERR_UNSUPPORTED = 2
MINIPIC_ERR_WORKSPACE_TOO_SMALL = 3
MINIPIC_ERR_CUDA = 4
MINIPIC_BF16, MINIPIC_F32 = 0, 1
MINIPIC_Q_PREROTATED, MINIPIC_K_PREROTATED, MINIPIC_FORCE_SIMT, MINIPIC_KEY_MASK = 1, 2, 4, 8

# every symbol include/minipic.h declares (tests check the library exports all of them)
EXPORTS = [
    "minipic_rope_table_bytes", "minipic_rope_table_build", "minipic_cache_write",
    "minipic_prefill_workspace_bytes", "minipic_prefill_attention",
    "minipic_decode_workspace_bytes", "minipic_decode_attention",
    "minipic_prefill_host_arena_bytes", "minipic_prefill_step_host",
    "minipic_decode_host_arena_bytes", "minipic_decode_step_host",
    "minipic_status_string", "minipic_last_cuda_error", "minipic_launch_count", "minipic_last_variant",
    "minipic_prefill_status", "minipic_preattn_fused", "minipic_block_rerotate",
    "minipic_block_hashes", "minipic_pool_create", "minipic_pool_destroy", "minipic_pool_admit", "minipic_pool_release",
    "minipic_pool_stats", "minipic_static_scratch_bytes", "minipic_decode_attention_static",
]


class minipic_config(C.Structure):
    _fields_ = [("num_q_heads", C.c_int32), ("num_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("block_size", C.c_int32), ("num_blocks", C.c_int32), ("dtype", C.c_int32),
                ("rope_theta", C.c_double), ("softmax_scale", C.c_float), ("flags", C.c_uint32),
                ("rope_table", C.c_void_p), ("rope_table_len", C.c_int32), ("reserved", C.c_int32)]


_lib = None


def lib() -> C.CDLL:
    """Load libminipic.so (once).  Fails loudly if it is missing - there is no CPU path."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not built: run `python -m paper_2606_13126_b200.build` "
                           "(the MiniPIC hot path has no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    P, I32, SZ, VP = C.POINTER(minipic_config), C.c_int32, C.c_size_t, C.c_void_p
    L.minipic_rope_table_bytes.restype = SZ
    L.minipic_rope_table_bytes.argtypes = [P, I32]
    L.minipic_rope_table_build.restype = C.c_int
    L.minipic_rope_table_build.argtypes = [P, I32, VP, VP]
    L.minipic_cache_write.restype = C.c_int
    L.minipic_cache_write.argtypes = [P, VP, VP, VP, I32, VP, VP, VP]
    L.minipic_prefill_workspace_bytes.restype = SZ
    L.minipic_prefill_workspace_bytes.argtypes = [P, I32, I32]
    L.minipic_prefill_attention.restype = C.c_int
    L.minipic_prefill_attention.argtypes = [P, VP, VP, VP, VP, I32, VP, VP, VP, VP, VP, VP, I32, I32, I32, VP, VP, VP, SZ, VP]
    L.minipic_decode_workspace_bytes.restype = SZ
    L.minipic_decode_workspace_bytes.argtypes = [P, I32, I32]
    L.minipic_decode_attention.restype = C.c_int
    L.minipic_static_scratch_bytes.restype = SZ
    L.minipic_static_scratch_bytes.argtypes = []
    L.minipic_decode_attention_static.restype = C.c_int
    L.minipic_decode_attention_static.argtypes = [P, VP, VP, VP, VP, I32, VP, VP, VP, VP, I32, I32, VP, VP, VP]
    L.minipic_decode_attention.argtypes = [P, VP, VP, VP, VP, I32, VP, VP, VP, VP, I32, I32, VP, VP, VP, SZ, VP]
    L.minipic_prefill_host_arena_bytes.restype = SZ
    L.minipic_prefill_host_arena_bytes.argtypes = [P, I32, I32, I32, I32, I32]
    L.minipic_prefill_step_host.restype = C.c_int
    L.minipic_prefill_step_host.argtypes = [P, VP, VP, VP, I32, VP, VP, VP, VP, I32, VP, VP, VP, VP, VP, VP,
                                            I32, I32, I32, VP, VP, VP, SZ, VP]
    L.minipic_decode_host_arena_bytes.restype = SZ
    L.minipic_decode_host_arena_bytes.argtypes = [P, I32, I32, I32, I32, I32]
    L.minipic_decode_step_host.restype = C.c_int
    L.minipic_decode_step_host.argtypes = [P, VP, VP, VP, I32, VP, VP, VP, VP, I32, VP, VP, VP, VP, I32, I32,
                                           VP, VP, VP, SZ, VP]
    L.minipic_status_string.restype = C.c_char_p
    L.minipic_status_string.argtypes = [C.c_int]
    L.minipic_last_cuda_error.restype = C.c_char_p
    L.minipic_launch_count.restype = C.c_uint64
    L.minipic_last_variant.restype = C.c_char_p
    L.minipic_prefill_status.restype = C.c_int
    L.minipic_prefill_status.argtypes = [VP, VP]
    L.minipic_preattn_fused.restype = C.c_int
    L.minipic_preattn_fused.argtypes = [P, VP, VP, VP, I32, VP, VP, VP, VP]
    L.minipic_block_rerotate.restype = C.c_int
    L.minipic_block_rerotate.argtypes = [P, VP, VP, VP, VP, VP, I32, VP]
    L.minipic_block_hashes.restype = C.c_int
    L.minipic_block_hashes.argtypes = [VP, I32, I32, I32, I32, C.c_uint64, VP]
    L.minipic_pool_create.restype = VP
    L.minipic_pool_create.argtypes = [I32, I32, I32, I32, C.c_uint64]
    L.minipic_pool_destroy.restype = None
    L.minipic_pool_destroy.argtypes = [VP]
    L.minipic_pool_admit.restype = C.c_int
    L.minipic_pool_admit.argtypes = [VP, VP, I32, VP, VP, VP, VP, VP]
    L.minipic_pool_release.restype = C.c_int
    L.minipic_pool_release.argtypes = [VP, VP, I32]
    L.minipic_pool_stats.restype = None
    L.minipic_pool_stats.argtypes = [VP, VP, VP, VP, VP]
    _lib = L
    return L


class MinipicError(RuntimeError):
    def __init__(self, status: int):
        L = lib()
        self.status = status
        msg = L.minipic_status_string(status).decode()
        if status == MINIPIC_ERR_CUDA:
            msg += ": " + L.minipic_last_cuda_error().decode()
        super().__init__(msg)


def _check(status: int) -> None:
    if status != MINIPIC_OK:
        raise MinipicError(status)


def _ptr(x) -> Optional[int]:
    """Address of a torch tensor / numpy array / raw int; None -> NULL."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    return x.ctypes.data  # numpy (host entry points)


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream if isinstance(stream, int) else stream.cuda_stream


def make_config(*, num_q_heads, num_kv_heads, head_dim, num_blocks, dtype, rope_theta, block_size=16,
                softmax_scale=0.0, flags=0, rope_table=None, rope_table_len=0) -> minipic_config:
    return minipic_config(num_q_heads, num_kv_heads, head_dim, block_size, num_blocks,
                          MINIPIC_BF16 if dtype in ("bf16", MINIPIC_BF16) else MINIPIC_F32,
                          float(rope_theta), float(softmax_scale), int(flags), _ptr(rope_table), int(rope_table_len), 0)


# ----------------------------------------------------------------------------- forwarding calls
def minipic_rope_table_bytes(cfg, num_positions: int) -> int:
    return lib().minipic_rope_table_bytes(C.byref(cfg), num_positions)


def minipic_rope_table_build(cfg, num_positions: int, table, stream=None) -> None:
    _check(lib().minipic_rope_table_build(C.byref(cfg), num_positions, _ptr(table), _stream(stream)))


def minipic_cache_write(cfg, k_new, v_new, slot_mapping, num_tokens, k_cache, v_cache, stream=None) -> None:
    _check(lib().minipic_cache_write(C.byref(cfg), _ptr(k_new), _ptr(v_new), _ptr(slot_mapping), num_tokens,
                                     _ptr(k_cache), _ptr(v_cache), _stream(stream)))


def minipic_preattn_fused(cfg, qkv, slot_mapping, positions, num_tokens, q_out, k_cache, v_cache, stream=None) -> None:
    _check(lib().minipic_preattn_fused(C.byref(cfg), _ptr(qkv), _ptr(slot_mapping), _ptr(positions), num_tokens,
                                       _ptr(q_out), _ptr(k_cache), _ptr(v_cache), _stream(stream)))


def minipic_block_rerotate(cfg, k_cache, v_cache, src_blocks, dst_blocks, delta, num_pairs, stream=None) -> None:
    _check(lib().minipic_block_rerotate(C.byref(cfg), _ptr(k_cache), _ptr(v_cache), _ptr(src_blocks), _ptr(dst_blocks),
                                        _ptr(delta), num_pairs, _stream(stream)))


def minipic_prefill_workspace_bytes(cfg, num_reqs: int, num_q_tokens: int) -> int:
    return lib().minipic_prefill_workspace_bytes(C.byref(cfg), num_reqs, num_q_tokens)


def minipic_prefill_attention(cfg, q, k_cache, v_cache, block_tables, max_blocks_per_req, cu_q_lens, kv_lens,
                              cu_kv_lens, kv_positions, q_seq_idx, q_vis_lo, num_reqs, num_q_tokens, max_kv_len,
                              out, lse, workspace, workspace_bytes, stream=None) -> None:
    _check(lib().minipic_prefill_attention(
        C.byref(cfg), _ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(block_tables), max_blocks_per_req, _ptr(cu_q_lens),
        _ptr(kv_lens), _ptr(cu_kv_lens), _ptr(kv_positions), _ptr(q_seq_idx), _ptr(q_vis_lo), num_reqs, num_q_tokens,
        max_kv_len, _ptr(out), _ptr(lse), _ptr(workspace), workspace_bytes, _stream(stream)))


def minipic_decode_workspace_bytes(cfg, num_seqs: int, max_kv_len: int) -> int:
    return lib().minipic_decode_workspace_bytes(C.byref(cfg), num_seqs, max_kv_len)


def minipic_decode_attention(cfg, q, k_cache, v_cache, block_tables, max_blocks_per_req, kv_lens, cu_kv_lens,
                             kv_positions, q_vis_lo, num_seqs, max_kv_len, out, lse, workspace, workspace_bytes,
                             stream=None) -> None:
    _check(lib().minipic_decode_attention(
        C.byref(cfg), _ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(block_tables), max_blocks_per_req, _ptr(kv_lens),
        _ptr(cu_kv_lens), _ptr(kv_positions), _ptr(q_vis_lo), num_seqs, max_kv_len, _ptr(out), _ptr(lse),
        _ptr(workspace), workspace_bytes, _stream(stream)))


def minipic_static_scratch_bytes() -> int:
    return lib().minipic_static_scratch_bytes()


def minipic_decode_attention_static(cfg, q, k_cache, v_cache, block_tables, max_blocks_per_req, kv_lens, cu_kv_lens,
                                    kv_positions, q_vis_lo, num_seqs, max_kv_len, out, lse, stream=None) -> None:
    """minipic_decode_attention with the split-KV partials in the library's static device array: allocates nothing."""
    _check(lib().minipic_decode_attention_static(
        C.byref(cfg), _ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(block_tables), max_blocks_per_req, _ptr(kv_lens),
        _ptr(cu_kv_lens), _ptr(kv_positions), _ptr(q_vis_lo), num_seqs, max_kv_len, _ptr(out), _ptr(lse), _stream(stream)))


def minipic_prefill_host_arena_bytes(cfg, num_reqs, num_q_tokens, num_new_tokens, max_blocks_per_req, total_kv_len) -> int:
    return lib().minipic_prefill_host_arena_bytes(C.byref(cfg), num_reqs, num_q_tokens, num_new_tokens,
                                                  max_blocks_per_req, total_kv_len)


def minipic_prefill_step_host(cfg, k_new_host, v_new_host, slot_mapping_host, num_new_tokens, q_host, k_cache, v_cache,
                              block_tables_host, max_blocks_per_req, cu_q_lens_host, kv_lens_host, cu_kv_lens_host,
                              kv_positions_host, q_seq_idx_host, q_vis_lo_host, num_reqs, num_q_tokens, max_kv_len,
                              out_host, lse_host, arena, arena_bytes, stream=None) -> None:
    _check(lib().minipic_prefill_step_host(
        C.byref(cfg), _ptr(k_new_host), _ptr(v_new_host), _ptr(slot_mapping_host), num_new_tokens, _ptr(q_host),
        _ptr(k_cache), _ptr(v_cache), _ptr(block_tables_host), max_blocks_per_req, _ptr(cu_q_lens_host),
        _ptr(kv_lens_host), _ptr(cu_kv_lens_host), _ptr(kv_positions_host), _ptr(q_seq_idx_host), _ptr(q_vis_lo_host),
        num_reqs, num_q_tokens, max_kv_len, _ptr(out_host), _ptr(lse_host), _ptr(arena), arena_bytes, _stream(stream)))


def minipic_decode_host_arena_bytes(cfg, num_seqs, num_new_tokens, max_blocks_per_req, total_kv_len, max_kv_len) -> int:
    return lib().minipic_decode_host_arena_bytes(C.byref(cfg), num_seqs, num_new_tokens, max_blocks_per_req,
                                                 total_kv_len, max_kv_len)


def minipic_decode_step_host(cfg, k_new_host, v_new_host, slot_mapping_host, num_new_tokens, q_host, k_cache, v_cache,
                             block_tables_host, max_blocks_per_req, kv_lens_host, cu_kv_lens_host, kv_positions_host,
                             q_vis_lo_host, num_seqs, max_kv_len, out_host, lse_host, arena, arena_bytes,
                             stream=None) -> None:
    _check(lib().minipic_decode_step_host(
        C.byref(cfg), _ptr(k_new_host), _ptr(v_new_host), _ptr(slot_mapping_host), num_new_tokens, _ptr(q_host),
        _ptr(k_cache), _ptr(v_cache), _ptr(block_tables_host), max_blocks_per_req, _ptr(kv_lens_host),
        _ptr(cu_kv_lens_host), _ptr(kv_positions_host), _ptr(q_vis_lo_host), num_seqs, max_kv_len, _ptr(out_host),
        _ptr(lse_host), _ptr(arena), arena_bytes, _stream(stream)))


def minipic_status_string(status: int) -> str:
    return lib().minipic_status_string(status).decode()


def minipic_launch_count() -> int:
    return int(lib().minipic_launch_count())


def minipic_last_variant() -> str:
    return lib().minipic_last_variant().decode()


def minipic_prefill_status(workspace, stream=None) -> None:
    """Synchronises the stream and raises if the last tcgen05 prefill call on `workspace` recorded a barrier timeout."""
    _check(lib().minipic_prefill_status(_ptr(workspace), _stream(stream)))


# ---- f3: host-side block hasher / pool (numpy arrays in host memory; argument marshalling only)
def _np_ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def minipic_block_hashes(tokens, block_size: int, ssep_id: int, pdep_id: int, seed: int = 0):
    import numpy as np
    tokens = np.ascontiguousarray(tokens, dtype=np.int32)
    out = np.zeros((len(tokens) // block_size, 32), np.uint8)
    _check(lib().minipic_block_hashes(_np_ptr(tokens), len(tokens), block_size, ssep_id, pdep_id, seed, _np_ptr(out)))
    return out


class Pool:
    """Thin handle on a minipic_pool (Eq. 1 block pool); all logic lives in csrc/hasher.cu."""

    def __init__(self, num_blocks: int, block_size: int, ssep_id: int, pdep_id: int, seed: int = 0):
        self.block_size = block_size
        self.h = lib().minipic_pool_create(num_blocks, block_size, ssep_id, pdep_id, seed)
        if not self.h:
            raise MinipicError(1)

    def admit(self, tokens):
        import numpy as np
        tokens = np.ascontiguousarray(tokens, dtype=np.int32)
        n, nb = len(tokens), -(-len(tokens) // self.block_size)
        table, hit = np.zeros(nb, np.int32), np.zeros(nb, np.uint8)
        slots, lo, n_new = np.zeros(n, np.int64), np.zeros(n, np.int32), C.c_int32(0)
        _check(lib().minipic_pool_admit(self.h, _np_ptr(tokens), n, _np_ptr(table), _np_ptr(hit), _np_ptr(slots), _np_ptr(lo),
                                        C.byref(n_new)))
        return table, hit, slots, lo, int(n_new.value)

    def release(self, table):
        import numpy as np
        table = np.ascontiguousarray(table, dtype=np.int32)
        _check(lib().minipic_pool_release(self.h, _np_ptr(table), len(table)))

    def stats(self):
        h, m, e, f = C.c_uint64(0), C.c_uint64(0), C.c_uint64(0), C.c_int32(0)
        lib().minipic_pool_stats(self.h, C.byref(h), C.byref(m), C.byref(e), C.byref(f))
        return dict(hits=h.value, misses=m.value, evictions=e.value, free_blocks=f.value)

    def close(self):
        if self.h:
            lib().minipic_pool_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
