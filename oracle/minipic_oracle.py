"""CPU ORACLE for the MiniPIC hot path.  TEST INFRASTRUCTURE - NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this file.  It shares no code with the CUDA path
(``paper_2606_13126_b200/csrc``) and imports nothing from the package.

What it computes is the plain definition the paper's method reaches exactly (up to
rounding order), written out in fp64 with numpy:

* cache write: scatter of unrotated K and V rows into paged blocks through a slot mapping
  (PAPER.md:47 paged blocks; :100 "stores unrotated key vectors k~_j and value vectors v_j");
* RoPE on read: k_j = R_{pi(j)} k~_j, q'_t = R_t q_t  (Eq. 2 :102);
* score(t, j) = q'_t . k_j / sqrt(d)                  (Eq. 2);
* mask: query row t sees sequence index j iff vis_lo[t] <= j <= idx[t]  - the block-level
  causal structure that the span primitives induce (
  DESIGN.md reading A6);
* softmax(scores) V and LSE = log sum exp(scores);
* split-KV merge identity used by decode (north star).

Readings of the paper that are baked in here (all listed in DESIGN.md "Readings"):
A1 rotate-half pairing (i, i+D/2); A2 f_i = theta^(-2i/D), full-head rotation, no frequency
scaling; A5 scale 1/sqrt(D), natural-log LSE; A10 slot = block*B + offset, negative = skip;
A11 cache layout [num_blocks, Hkv, B, D].

Parity pins (tests/test_oracle_pins.py, all ``-m "not gpu"``): brute-force dense attention in
pure Python on tiny inputs; RoPE closed forms (R(0)=I, norm preservation, relative-position
identity, shift invariance pi -> pi + c); D=2 closed form cos(j - t) golden fixture;
rotate-on-read == pre-rotated dense cache through torch's fp64 scaled_dot_product_attention;
closed-form softmax cases (one visible key, Q = 0, constant V); span rows == standalone span
request; shared / duplicated physical blocks; block-id
permutation invariance bit-for-bit; merge identity over random partitions.  No function here
is "parity unpinned".  The paper prints no worked numeric values for this path.
"""
from __future__ import annotations

import numpy as np

F64 = np.float64


# ----------------------------------------------------------------------------- storage formats
def bf16_bits_to_f64(bits: np.ndarray) -> np.ndarray:
    """Exact upcast of bfloat16 bit patterns (uint16) to float64."""
    u = np.asarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)
    return u.view(np.float32).astype(F64)


def to_f64(x: np.ndarray, dtype: str) -> np.ndarray:
    """Upcast an I/O-dtype array (bf16 carried as uint16 bits, or float32) to float64, exactly."""
    if dtype == "bf16":
        return bf16_bits_to_f64(x)
    if dtype == "f32":
        return np.asarray(x, dtype=np.float32).astype(F64)
    raise ValueError(dtype)


def round_to_dtype(x: np.ndarray, dtype: str) -> np.ndarray:
    """Round fp64 values once, round-to-nearest-even, to the I/O dtype; return them as fp64.

    Used only by comparison mode "Q" (what a conventional pre-rotated cache would store,
    PAPER.md:53 "storing already-rotated keys in the KV cache").
    """
    if dtype == "f32":
        return np.asarray(x, F64).astype(np.float32).astype(F64)
    if dtype == "bf16":
        # one rounding, fp64 -> 8 significant bits (1 implicit + 7 stored), ties to even:
        # x = m * 2^e with 0.5 <= |m| < 1, so m * 2^8 has its last bf16 bit at the units place and
        # np.rint (round-half-to-even) rounds there.  bf16 subnormals / overflow (|x| < 2^-126,
        # |x| >= 2^128) do not occur for the attention operands this is used on.
        m, e = np.frexp(np.asarray(x, F64))
        return np.ldexp(np.rint(m * 256.0) / 256.0, e)
    raise ValueError(dtype)


# ----------------------------------------------------------------------------- a1: cache write
def new_cache(num_blocks: int, num_kv_heads: int, block_size: int, head_dim: int, dtype: str, fill=0):
    """An empty paged cache in the layout of DESIGN.md reading A11: [num_blocks, Hkv, B, D]."""
    np_dtype = np.uint16 if dtype == "bf16" else np.float32
    return np.full((num_blocks, num_kv_heads, block_size, head_dim), fill, dtype=np_dtype)


def cache_write(k_cache: np.ndarray, v_cache: np.ndarray, k_new: np.ndarray, v_new: np.ndarray,
                slot_mapping: np.ndarray) -> None:
    """Scatter rows of new tokens into paged blocks, bit for bit, no rotation, no conversion.

    cache[slot // B, h, slot % B, :] = new[t, h, :]   for every t with slot >= 0
    (PAPER.md:47 fixed-size blocks; :100 K is stored UNROTATED; :113 "V vectors are unchanged").
    """
    block_size = k_cache.shape[2]
    for t in range(len(slot_mapping)):
        slot = int(slot_mapping[t])
        if slot < 0:
            continue
        blk, off = slot // block_size, slot % block_size
        k_cache[blk, :, off, :] = k_new[t, :, :]          # every KV head h: cache[blk, h, off, :] = new[t, h, :]
        v_cache[blk, :, off, :] = v_new[t, :, :]


# ----------------------------------------------------------------------------- a3/a5: RoPE
def rope_frequencies(head_dim: int, theta: float) -> np.ndarray:
    """f_i = theta^(-2i/D), i in [0, D/2)  (reading A2; RoFormer [22] as used by Llama-3)."""
    i = np.arange(head_dim // 2, dtype=F64)
    return F64(theta) ** (-2.0 * i / F64(head_dim))


def rope_rotate(x: np.ndarray, positions: np.ndarray, theta: float) -> np.ndarray:
    """R_p x with rotate-half pairing (reading A1): for i in [0, D/2), phi = p * f_i,

        y[i]       = x[i] cos(phi) - x[i + D/2] sin(phi)
        y[i + D/2] = x[i + D/2] cos(phi) + x[i] sin(phi)

    (Eq. 2, "two fused multiply-adds per K element").
    ``x``: [..., D] fp64; ``positions``: broadcastable to x.shape[:-1].
    """
    x = np.asarray(x, F64)
    d = x.shape[-1]
    half = d // 2
    phi = np.asarray(positions, F64)[..., None] * rope_frequencies(d, theta)
    c, s = np.cos(phi), np.sin(phi)
    lo, hi = x[..., :half], x[..., half:]
    return np.concatenate([lo * c - hi * s, hi * c + lo * s], axis=-1)


# ----------------------------------------------------------------------------- a4: gather
def gather_kv(k_cache: np.ndarray, v_cache: np.ndarray, block_table_row: np.ndarray, kv_len: int,
              kv_head: int, dtype: str):
    """k~_j, v_j for j in [0, kv_len) of one request and one KV head through its block table:
    blk = bt[j // B]; row = cache[blk, head, j % B]."""
    block_size = k_cache.shape[2]
    j = np.arange(kv_len)
    blk = np.asarray(block_table_row)[j // block_size]
    off = j % block_size
    return to_f64(k_cache[blk, kv_head, off, :], dtype), to_f64(v_cache[blk, kv_head, off, :], dtype)


# ----------------------------------------------------------------------------- a6-a9: attention
def _attend_rows(qr: np.ndarray, k: np.ndarray, v: np.ndarray, idx: np.ndarray, vis_lo: np.ndarray, scale: float,
                 key_ok: np.ndarray | None = None):
    """Masked softmax attention for a group of query rows of one (request, head).

    qr [n, D] rotated queries; k, v [kv_len, D] rotated keys / values; row i sees key j iff
    vis_lo[i] <= j <= idx[i] (and key_ok[j], when the key-masking variant is on: PAPER.md:294).
    Returns out [n, D], lse [n].  A row with no visible key returns out = 0, lse = -inf.
    """
    kv_len = k.shape[0]
    s = (qr @ k.T) * scale                                   # Eq. 2 scores for every (row, key)
    j = np.arange(kv_len)[None, :]
    visible = (j >= vis_lo[:, None]) & (j <= idx[:, None])
    if key_ok is not None:
        visible = visible & np.asarray(key_ok, bool)[None, :]
    s = np.where(visible, s, -np.inf)
    m = s.max(axis=1) if kv_len else np.full(qr.shape[0], -np.inf)
    empty = ~np.isfinite(m)
    m_safe = np.where(empty, 0.0, m)
    e = np.exp(s - m_safe[:, None])                          # exp(-inf) = 0 for masked keys
    l = e.sum(axis=1)
    with np.errstate(divide="ignore", invalid="ignore"):
        lse = np.where(empty, -np.inf, m_safe + np.log(l))
        out = np.where(empty[:, None], 0.0, (e @ v) / np.where(empty, 1.0, l)[:, None])
    return out, lse


def prefill_attention(*, q, k_cache, v_cache, block_tables, cu_q_lens, kv_lens, cu_kv_lens, kv_positions,
                      q_seq_idx, q_vis_lo, num_q_heads: int, dtype: str, rope_theta: float,
                      softmax_scale: float | None = None, mode: str = "F", q_prerotated: bool = False,
                      k_prerotated: bool = False, rows: np.ndarray | None = None,
                      heads: np.ndarray | None = None, row_chunk: int = 512, key_mask: bool = False):
    """Steps 2-6 of DESIGN.md "Oracle algorithm" for every query row (or for ``rows`` x ``heads``).

    Returns (out fp64 [Tq, Hq, D], lse fp64 [Tq, Hq]); entries outside ``rows`` x ``heads`` are NaN.
    mode "F": pure fp64.  mode "Q": q' and k_j are rounded once to the I/O dtype after rotation
    and before the scores (the conventional pre-rotated-cache arithmetic).
    Query rows are processed in chunks of ``row_chunk`` only to bound memory; rows are
    independent, so this changes no arithmetic.
    ``key_mask`` (the "key-vector zeroing" of marker / padding tokens that PAPER.md:294 defers, taken as a
    MASK variant): a key whose logical position is negative is invisible to every query row.
    """
    tq = q.shape[0]
    hq = num_q_heads
    hkv, d = k_cache.shape[1], k_cache.shape[3]
    group = hq // hkv
    scale = (1.0 / np.sqrt(F64(d))) if not softmax_scale else F64(softmax_scale)
    out = np.full((tq, hq, d), np.nan, F64)
    lse = np.full((tq, hq), np.nan, F64)
    head_list = list(range(hq)) if heads is None else [int(h) for h in heads]
    row_mask = None
    if rows is not None:
        row_mask = np.zeros(tq, bool); row_mask[np.asarray(rows)] = True
    for r in range(len(kv_lens)):
        t0, t1 = int(cu_q_lens[r]), int(cu_q_lens[r + 1])
        sel = np.arange(t0, t1)
        if row_mask is not None:
            sel = sel[row_mask[sel]]
        if sel.size == 0:
            continue
        kv_len = int(kv_lens[r])
        pos = np.asarray(kv_positions[int(cu_kv_lens[r]):int(cu_kv_lens[r]) + kv_len])
        idx = np.asarray(q_seq_idx)[sel].astype(np.int64)
        lo = np.asarray(q_vis_lo)[sel].astype(np.int64)
        q_pos = pos[idx]                                           # pi_r(idx_t)
        key_ok = (pos >= 0) if key_mask else None
        cache_kv = {}
        for h in head_list:
            g = h // group                                         # GQA: KV head of query head h
            if g not in cache_kv:
                kt, vv = gather_kv(k_cache, v_cache, block_tables[r], kv_len, g, dtype)     # step 2
                kk = kt if k_prerotated else rope_rotate(kt, pos, rope_theta)               # step 3
                if mode == "Q":
                    kk = round_to_dtype(kk, dtype)
                cache_kv[g] = (kk, vv)
            kk, vv = cache_kv[g]
            qh = to_f64(q[sel, h, :], dtype)
            qr = qh if q_prerotated else rope_rotate(qh, q_pos, rope_theta)                 # step 4
            if mode == "Q":
                qr = round_to_dtype(qr, dtype)
            for c0 in range(0, sel.size, row_chunk):
                c1 = min(c0 + row_chunk, sel.size)
                # keys outside [min vis_lo, max idx] of the chunk are invisible to every row of it
                klo, hi = max(int(lo[c0:c1].min()), 0), int(idx[c0:c1].max()) + 1
                o, l = _attend_rows(qr[c0:c1], kk[klo:hi], vv[klo:hi], idx[c0:c1] - klo, lo[c0:c1] - klo, scale,
                                    None if key_ok is None else key_ok[klo:hi])                                   # steps 5-6
                out[sel[c0:c1], h, :] = o
                lse[sel[c0:c1], h] = l
    return out, lse


def decode_attention(*, q, k_cache, v_cache, block_tables, kv_lens, cu_kv_lens, kv_positions, num_q_heads: int,
                     dtype: str, rope_theta: float, q_vis_lo=None, softmax_scale: float | None = None,
                     mode: str = "F", q_prerotated: bool = False, k_prerotated: bool = False,
                     seqs: np.ndarray | None = None, heads: np.ndarray | None = None, key_mask: bool = False):
    """Decode = the same definition with one query per sequence at idx = kv_len - 1 (step 7)."""
    n = len(kv_lens)
    idx = (np.asarray(kv_lens) - 1).astype(np.int32)
    lo = np.zeros(n, np.int32) if q_vis_lo is None else np.asarray(q_vis_lo, np.int32)
    return prefill_attention(q=q, k_cache=k_cache, v_cache=v_cache, block_tables=block_tables,
                             cu_q_lens=np.arange(n + 1), kv_lens=kv_lens, cu_kv_lens=cu_kv_lens,
                             kv_positions=kv_positions, q_seq_idx=idx, q_vis_lo=lo, num_q_heads=num_q_heads,
                             dtype=dtype, rope_theta=rope_theta, softmax_scale=softmax_scale, mode=mode,
                             q_prerotated=q_prerotated, k_prerotated=k_prerotated, rows=seqs, heads=heads,
                             key_mask=key_mask)


# ----------------------------------------------------------------------------- a11: LSE merge
def merge_partials(o_parts: np.ndarray, lse_parts: np.ndarray):
    """Merge identity for any partition of the key set (decode split-KV, step 7):

        lse = ln sum_s exp(lse_s);   o = sum_s exp(lse_s - lse) o_s

    o_parts [S, D] (each normalised over its own part), lse_parts [S]; parts with lse = -inf are empty.
    """
    lse_parts = np.asarray(lse_parts, F64)
    o_parts = np.asarray(o_parts, F64)
    m = lse_parts.max()
    if not np.isfinite(m):
        return np.zeros(o_parts.shape[1], F64), -np.inf
    w = np.exp(lse_parts - m)
    lse = m + np.log(w.sum())
    return (np.exp(lse_parts - lse)[:, None] * np.where(np.isfinite(lse_parts)[:, None], o_parts, 0.0)).sum(axis=0), lse


# ----------------------------------------------------------------------------- convenience for tests / bench
def build_cache(workload, fill=0):
    """Run the oracle's own scalar cache write over a workload's resident + new batches."""
    kc = new_cache(workload.num_blocks, workload.num_kv_heads, workload.block_size, workload.head_dim,
                   workload.dtype, fill)
    vc = new_cache(workload.num_blocks, workload.num_kv_heads, workload.block_size, workload.head_dim,
                   workload.dtype, fill)
    for b in list(workload.resident) + list(workload.new):
        cache_write(kc, vc, b.k, b.v, b.slots)
    return kc, vc


def run_workload(workload, kc, vc, mode="F", rows=None, heads=None, **kw):
    """Attention of a workload object (duck-typed: fields of workloads.Workload) on oracle caches."""
    common = dict(q=workload.q, k_cache=kc, v_cache=vc, block_tables=workload.block_tables,
                  kv_lens=workload.kv_lens, cu_kv_lens=workload.cu_kv_lens, kv_positions=workload.kv_positions,
                  num_q_heads=workload.num_q_heads, dtype=workload.dtype, rope_theta=workload.rope_theta,
                  mode=mode, heads=heads, **kw)
    if workload.kind == "decode":
        return decode_attention(q_vis_lo=workload.q_vis_lo, seqs=rows, **common)
    return prefill_attention(cu_q_lens=workload.cu_q_lens, q_seq_idx=workload.q_seq_idx,
                             q_vis_lo=workload.q_vis_lo, rows=rows, **common)
