"""Device-side plumbing around the binding: upload a ``workloads.Workload``, own the caches /
workspaces as torch tensors, and call the C ABI.  No arithmetic of the method happens here.
Used by tests, bench.py and __graft_entry__.smoke()."""
from __future__ import annotations

import numpy as np
import torch

from . import binding as mp
from .workloads import Workload


def _dev(a: np.ndarray, device) -> torch.Tensor:
    """numpy -> device tensor, bit for bit (uint16 bf16 bits travel as int16)."""
    a = np.ascontiguousarray(a)
    if a.dtype == np.uint16:
        a = a.view(np.int16)
    return torch.from_numpy(a).to(device, non_blocking=False)


def _pinned(a: np.ndarray) -> torch.Tensor:
    a = np.ascontiguousarray(a)
    if a.dtype == np.uint16:
        a = a.view(np.int16)
    t = torch.from_numpy(a)
    return t.pin_memory() if torch.cuda.is_available() else t


class DeviceWorkload:
    """A workload resident on one GPU: caches, inputs, outputs, workspaces."""

    def __init__(self, w: Workload, device="cuda:0", flags: int = 0, rope_table_positions: int | None = None,
                 cache_fill: int | None = None, upload_resident: bool = True):
        self.w = w
        self.device = torch.device(device)
        self.itemsize = w.itemsize
        el = torch.int16 if w.dtype == "bf16" else torch.float32
        shape = (w.num_blocks, w.num_kv_heads, w.block_size, w.head_dim)
        if cache_fill is None:
            self.k_cache = torch.zeros(shape, dtype=el, device=self.device)
            self.v_cache = torch.zeros(shape, dtype=el, device=self.device)
        else:
            self.k_cache = torch.full(shape, cache_fill, dtype=el, device=self.device)
            self.v_cache = torch.full(shape, cache_fill, dtype=el, device=self.device)
        self.table = None
        self.table_len = 0
        self.flags = flags
        self.cfg = self._cfg()
        if rope_table_positions:
            nbytes = mp.minipic_rope_table_bytes(self.cfg, rope_table_positions)
            self.table = torch.empty(nbytes // 4, dtype=torch.float32, device=self.device)
            mp.minipic_rope_table_build(self.cfg, rope_table_positions, self.table)
            self.table_len = rope_table_positions
            self.cfg = self._cfg()
        d = self.device
        self.q = _dev(w.q, d)
        self.block_tables = _dev(w.block_tables, d)
        self.cu_q_lens = _dev(w.cu_q_lens, d)
        self.kv_lens = _dev(w.kv_lens, d)
        self.cu_kv_lens = _dev(w.cu_kv_lens, d)
        self.kv_positions = _dev(w.kv_positions, d)
        self.q_seq_idx = _dev(w.q_seq_idx, d)
        self.q_vis_lo = _dev(w.q_vis_lo, d)
        self.out = torch.zeros_like(self.q)
        self.lse = torch.zeros(self.q.shape[:2], dtype=torch.float32, device=d)
        self.new_dev = [(_dev(b.k, d), _dev(b.v, d), _dev(b.slots, d)) for b in w.new]
        if w.kind == "prefill":
            self.ws_bytes = mp.minipic_prefill_workspace_bytes(self.cfg, w.num_reqs, w.num_q_tokens)
        else:
            self.ws_bytes = mp.minipic_decode_workspace_bytes(self.cfg, w.num_reqs, w.max_kv_len)
        self.workspace = torch.empty(max(self.ws_bytes, 256), dtype=torch.uint8, device=d)
        if upload_resident:
            self.write_resident()

    def _cfg(self, flags=None):
        w = self.w
        return mp.make_config(num_q_heads=w.num_q_heads, num_kv_heads=w.num_kv_heads, head_dim=w.head_dim,
                              num_blocks=w.num_blocks, dtype=w.dtype, rope_theta=w.rope_theta,
                              flags=self.flags if flags is None else flags,
                              rope_table=self.table, rope_table_len=self.table_len)

    def set_flags(self, flags: int):
        self.flags = flags
        self.cfg = self._cfg()

    # ---- a1
    def write_resident(self):
        """Cached spans enter the cache through the library's own cache_write (one call per batch;
        aliased source arrays are uploaded once)."""
        seen = {}
        for b in self.w.resident:
            key = (id(b.k), id(b.v))
            if key not in seen:
                seen[key] = (_dev(b.k, self.device), _dev(b.v, self.device))
            k, v = seen[key]
            slots = _dev(b.slots, self.device)
            mp.minipic_cache_write(self.cfg, k, v, slots, int(slots.shape[0]), self.k_cache, self.v_cache)
        torch.cuda.synchronize(self.device)

    def write_new(self):
        for k, v, slots in self.new_dev:
            mp.minipic_cache_write(self.cfg, k, v, slots, int(slots.shape[0]), self.k_cache, self.v_cache)

    # ---- a2-a11
    def attention(self):
        w = self.w
        if w.kind == "prefill":
            mp.minipic_prefill_attention(self.cfg, self.q, self.k_cache, self.v_cache, self.block_tables,
                                         int(self.block_tables.shape[1]), self.cu_q_lens, self.kv_lens, self.cu_kv_lens,
                                         self.kv_positions, self.q_seq_idx, self.q_vis_lo, w.num_reqs, w.num_q_tokens,
                                         w.max_kv_len, self.out, self.lse, self.workspace, self.ws_bytes)
        else:
            mp.minipic_decode_attention(self.cfg, self.q, self.k_cache, self.v_cache, self.block_tables,
                                        int(self.block_tables.shape[1]), self.kv_lens, self.cu_kv_lens,
                                        self.kv_positions, self.q_vis_lo, w.num_reqs, w.max_kv_len, self.out, self.lse,
                                        self.workspace, self.ws_bytes)

    def step(self):
        self.write_new()
        self.attention()

    def check_health(self):
        """Synchronise and raise if the prefill kernel recorded a hand-off timeout (minipic_prefill_status)."""
        if self.w.kind == "prefill":
            mp.minipic_prefill_status(self.workspace)

    # ---- results back on the host
    def out_f64(self) -> np.ndarray:
        o = self.out
        if self.w.dtype == "bf16":
            o = o.view(torch.bfloat16)
        return o.double().cpu().numpy()

    def lse_f64(self) -> np.ndarray:
        return self.lse.double().cpu().numpy()

    def cache_bits(self):
        k, v = self.k_cache.cpu().numpy(), self.v_cache.cpu().numpy()
        if self.w.dtype == "bf16":
            k, v = k.view(np.uint16), v.view(np.uint16)
        return k, v


class HostStep:
    """End-to-end step through the *_step_host entry points: pinned host inputs, device arena,
    host outputs.  The resident cache must already be on the device (a DeviceWorkload owns it)."""

    def __init__(self, dw: DeviceWorkload):
        self.dw = dw
        w = dw.w
        nb = w.new[0] if w.new else None
        self.n_new = int(nb.slots.shape[0]) if nb is not None else 0
        self.k_new = _pinned(nb.k) if nb is not None else None
        self.v_new = _pinned(nb.v) if nb is not None else None
        self.slots = _pinned(nb.slots) if nb is not None else None
        self.q = _pinned(w.q)
        self.bt = _pinned(w.block_tables)
        self.cu_q = _pinned(w.cu_q_lens)
        self.kv_lens = _pinned(w.kv_lens)
        self.cu_kv = _pinned(w.cu_kv_lens)
        self.pos = _pinned(w.kv_positions)
        self.idx = _pinned(w.q_seq_idx)
        self.lo = _pinned(w.q_vis_lo)
        self.out = torch.empty(self.q.shape, dtype=self.q.dtype).pin_memory()
        self.lse = torch.empty(self.q.shape[:2], dtype=torch.float32).pin_memory()
        total_kv = int(w.cu_kv_lens[-1])
        if w.kind == "prefill":
            self.arena_bytes = mp.minipic_prefill_host_arena_bytes(dw.cfg, w.num_reqs, w.num_q_tokens, self.n_new,
                                                                   int(w.block_tables.shape[1]), total_kv)
        else:
            self.arena_bytes = mp.minipic_decode_host_arena_bytes(dw.cfg, w.num_reqs, self.n_new,
                                                                  int(w.block_tables.shape[1]), total_kv, w.max_kv_len)
        self.arena = torch.empty(self.arena_bytes, dtype=torch.uint8, device=dw.device)
        self.h2d_bytes = sum(t.numel() * t.element_size() for t in
                             (self.k_new, self.v_new, self.slots, self.q, self.bt, self.kv_lens, self.cu_kv, self.pos)
                             if t is not None)
        if w.kind == "prefill":
            self.h2d_bytes += sum(t.numel() * t.element_size() for t in (self.cu_q, self.idx, self.lo))
        else:
            self.h2d_bytes += self.lo.numel() * 4
        self.d2h_bytes = self.out.numel() * self.out.element_size() + self.lse.numel() * 4

    def run(self):
        dw, w = self.dw, self.dw.w
        if w.kind == "prefill":
            mp.minipic_prefill_step_host(dw.cfg, self.k_new, self.v_new, self.slots, self.n_new, self.q, dw.k_cache,
                                         dw.v_cache, self.bt, int(w.block_tables.shape[1]), self.cu_q, self.kv_lens,
                                         self.cu_kv, self.pos, self.idx, self.lo, w.num_reqs, w.num_q_tokens,
                                         w.max_kv_len, self.out, self.lse, self.arena, self.arena_bytes)
        else:
            mp.minipic_decode_step_host(dw.cfg, self.k_new, self.v_new, self.slots, self.n_new, self.q, dw.k_cache,
                                        dw.v_cache, self.bt, int(w.block_tables.shape[1]), self.kv_lens, self.cu_kv,
                                        self.pos, self.lo, w.num_reqs, w.max_kv_len, self.out, self.lse, self.arena,
                                        self.arena_bytes)

    def out_f64(self):
        o = self.out
        if self.dw.w.dtype == "bf16":
            o = o.view(torch.bfloat16)
        return o.double().numpy()

    def lse_f64(self):
        return self.lse.double().numpy()
