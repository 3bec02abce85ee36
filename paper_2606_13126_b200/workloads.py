"""Seeded synthetic inputs for the MiniPIC hot path.

These stand in for the paper's RAG workload (system prompt + 10 retrieved documents +
task suffix; 1000-token synthetic documents): the dataset,
weights and serving engine are not available and are not needed.  What the engine's
block hasher / block pool / scheduler (Eq. 1 :83-88) would have produced
is emitted directly: slot mappings, block tables, the per-request logical-position table
 and the span/visibility descriptor induced by the Block-Attention
submission procedure.

This module holds NO arithmetic of the method (no RoPE, no scores, no softmax).  It only
draws random numbers, rounds them once to the I/O dtype (a storage-format conversion) and
lays out integer index tables.  Both the oracle (via tests / bench) and the CUDA path
consume its arrays; neither imports the other.

All arrays are numpy.  bf16 tensors are carried as ``uint16`` bit patterns.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import List, Optional, Sequence, Tuple

import numpy as np

BLOCK = 16  # PAPER.md:125 "pad to a block boundary (16 tokens)"


# --------------------------------------------------------------------------- storage format
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round float32 -> bfloat16 (round-to-nearest-even), returned as uint16 bits."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    rounding = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + rounding) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """uint16 bfloat16 bits -> float32 (exact)."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def _draw(rng: np.random.Generator, shape, sigma: float, dtype: str) -> np.ndarray:
    x = rng.standard_normal(shape, dtype=np.float32)
    if sigma != 1.0:
        x *= np.float32(sigma)
    return f32_to_bf16_bits(x) if dtype == "bf16" else x


# --------------------------------------------------------------------------- containers
@dataclass
class WriteBatch:
    """One ``minipic_cache_write`` call: rows ``k[t], v[t]`` go to slot ``slots[t]``."""
    k: np.ndarray            # [T, Hkv, D]  (uint16 bf16 bits | float32)
    v: np.ndarray            # [T, Hkv, D]
    slots: np.ndarray        # int64 [T]; slot = block_id * BLOCK + offset, <0 => skip
    tag: str = ""


@dataclass
class Workload:
    name: str
    kind: str                # "prefill" | "decode"
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    num_blocks: int
    dtype: str               # "bf16" | "f32"
    rope_theta: float
    resident: List[WriteBatch]   # cache contents that exist before the step (cached spans)
    new: List[WriteBatch]        # the step's own cache write (new tokens), 0 or 1 batch
    q: np.ndarray                # prefill [Tq,Hq,D]; decode [R,Hq,D]
    block_tables: np.ndarray     # int32 [R, max_blocks]
    cu_q_lens: np.ndarray        # int32 [R+1]
    kv_lens: np.ndarray          # int32 [R]
    cu_kv_lens: np.ndarray       # int32 [R+1]
    kv_positions: np.ndarray     # int32 [sum kv_lens]  logical position pi_r(j)
    q_seq_idx: np.ndarray        # int32 [Tq]
    q_vis_lo: np.ndarray         # int32 [Tq]
    block_size: int = BLOCK
    seed: int = 0
    notes: dict = field(default_factory=dict)

    @property
    def num_reqs(self) -> int:
        return int(self.kv_lens.shape[0])

    @property
    def num_q_tokens(self) -> int:
        return int(self.q.shape[0])

    @property
    def max_kv_len(self) -> int:
        return int(self.kv_lens.max()) if self.kv_lens.size else 0

    @property
    def itemsize(self) -> int:
        return 2 if self.dtype == "bf16" else 4

    # ---- algorithmic work: integer counting only
    def visible_pairs(self) -> int:
        """P = number of visible (query, key) pairs per query head."""
        return int((self.q_seq_idx.astype(np.int64) - self.q_vis_lo.astype(np.int64) + 1).clip(min=0).sum())

    def attention_flops(self) -> int:
        return 4 * self.head_dim * self.num_q_heads * self.visible_pairs()

    def logical_kv_bytes(self) -> int:
        return int(self.kv_lens.astype(np.int64).sum()) * self.num_kv_heads * self.head_dim * 2 * self.itemsize

    def written_tokens(self) -> int:
        return int(sum(int((b.slots >= 0).sum()) for b in self.new))


class _Composer:
    """Allocates physical blocks from a permuted pool and lays out requests."""

    def __init__(self, rng, num_blocks, hkv, d, dtype, sigma):
        self.rng, self.num_blocks, self.hkv, self.d = rng, num_blocks, hkv, d
        self.dtype, self.sigma = dtype, sigma
        self.perm = rng.permutation(num_blocks).astype(np.int64)  # nothing is contiguous
        self.next = 0
        self.resident: List[WriteBatch] = []
        self.new_k: list = []
        self.new_v: list = []
        self.new_slots: list = []

    def alloc(self, n_tokens: int) -> np.ndarray:
        nb = -(-n_tokens // BLOCK)
        if self.next + nb > self.num_blocks:
            raise ValueError("block pool exhausted")
        ids = self.perm[self.next:self.next + nb]
        self.next += nb
        return ids

    @staticmethod
    def slots_of(blocks: np.ndarray, n_tokens: int) -> np.ndarray:
        t = np.arange(n_tokens, dtype=np.int64)
        return blocks[t // BLOCK] * BLOCK + (t % BLOCK)

    def tokens(self, n_tokens: int, resident: bool, tag: str = "") -> np.ndarray:
        """Draw K/V for n_tokens, place them in freshly allocated blocks; return block ids."""
        blocks = self.alloc(n_tokens)
        k = _draw(self.rng, (n_tokens, self.hkv, self.d), self.sigma, self.dtype)
        v = _draw(self.rng, (n_tokens, self.hkv, self.d), self.sigma, self.dtype)
        slots = self.slots_of(blocks, n_tokens)
        if resident:
            self.resident.append(WriteBatch(k, v, slots, tag))
        else:
            self.new_k.append(k); self.new_v.append(v); self.new_slots.append(slots)
        return blocks

    def new_batch(self) -> List[WriteBatch]:
        if not self.new_k:
            return []
        return [WriteBatch(np.concatenate(self.new_k), np.concatenate(self.new_v),
                           np.concatenate(self.new_slots), "new")]


@dataclass
class _Seg:
    blocks: np.ndarray
    length: int
    local: bool      # True: span-local causal (vis_lo = span start); False: sees everything before it
    query: bool


def _layout(reqs: Sequence[Sequence[_Seg]], pos_offset: Sequence[int] | None = None):
    """Integer layout of composed requests -> block tables, positions, descriptor."""
    R = len(reqs)
    kv_lens = np.zeros(R, np.int32)
    tables, positions, q_idx, q_lo, q_counts = [], [], [], [], []
    for r, segs in enumerate(reqs):
        off = 0
        tb = []
        qi, ql = [], []
        for s_i, s in enumerate(segs):
            if off % BLOCK != 0:
                raise ValueError("segments must start block-aligned (PAPER.md:79 padding primitive)")
            tb.append(np.asarray(s.blocks, np.int64))
            if s.query:
                idx = np.arange(off, off + s.length, dtype=np.int32)
                qi.append(idx)
                ql.append(np.full(s.length, off if s.local else 0, np.int32))
            off += s.length
        kv_lens[r] = off
        tables.append(np.concatenate(tb) if tb else np.zeros(0, np.int64))
        base = 0 if pos_offset is None else int(pos_offset[r])
        positions.append(np.arange(off, dtype=np.int32) + np.int32(base))
        q_idx.append(np.concatenate(qi) if qi else np.zeros(0, np.int32))
        q_lo.append(np.concatenate(ql) if ql else np.zeros(0, np.int32))
        q_counts.append(q_idx[-1].shape[0])
    max_blocks = max((t.shape[0] for t in tables), default=1)
    bt = np.zeros((R, max(max_blocks, 1)), np.int32)
    for r, t in enumerate(tables):
        bt[r, :t.shape[0]] = t
    cu_q = np.zeros(R + 1, np.int32); cu_q[1:] = np.cumsum(q_counts)
    cu_kv = np.zeros(R + 1, np.int32); cu_kv[1:] = np.cumsum(kv_lens)
    return dict(block_tables=bt, cu_q_lens=cu_q, kv_lens=kv_lens, cu_kv_lens=cu_kv,
                kv_positions=np.concatenate(positions) if positions else np.zeros(0, np.int32),
                q_seq_idx=np.concatenate(q_idx) if q_idx else np.zeros(0, np.int32),
                q_vis_lo=np.concatenate(q_lo) if q_lo else np.zeros(0, np.int32))


def _round_up(n: int, m: int = BLOCK) -> int:
    return -(-n // m) * m


# --------------------------------------------------------------------------- config 1 / 2
def single_request_prefill(*, name: str, hq: int, hkv: int, d: int, theta: float, dtype: str,
                           sigma: float, span_lens: Sequence[int], suffix_len: int,
                           num_blocks: int, seed: int, pos_offset: int = 0) -> Workload:
    """BASELINE configs[0] / configs[1]: one request, every token is new and is a query.

    Spans attend causally within themselves; the suffix attends causally to everything
    (PAPER.md:123-128).  Draw order (fixed): block permutation, then per segment K, V, then Q.
    """
    rng = np.random.default_rng(seed)
    c = _Composer(rng, num_blocks, hkv, d, dtype, sigma)
    segs = []
    for L in span_lens:
        segs.append(_Seg(c.tokens(L, resident=False), L, local=True, query=True))
    if suffix_len:
        segs.append(_Seg(c.tokens(suffix_len, resident=False), suffix_len, local=False, query=True))
    lay = _layout([segs], [pos_offset])
    tq = int(lay["cu_q_lens"][-1])
    q = _draw(rng, (tq, hq, d), sigma, dtype)
    return Workload(name=name, kind="prefill", num_q_heads=hq, num_kv_heads=hkv, head_dim=d,
                    num_blocks=num_blocks, dtype=dtype, rope_theta=theta, resident=c.resident,
                    new=c.new_batch(), q=q, seed=seed, **lay)


def config1(seed: int = 0) -> Workload:
    """Tiny prefill (BASELINE.json configs[0])."""
    return single_request_prefill(name="c1_tiny_prefill", hq=4, hkv=1, d=64, theta=1e4, dtype="f32",
                                  sigma=1.0, span_lens=[32, 32, 32], suffix_len=16, num_blocks=32, seed=seed)


def config2(seed: int = 1) -> Workload:
    """Llama-3-8B shapes, single-request prefill (BASELINE.json configs[1])."""
    return single_request_prefill(name="c2_llama8b_single", hq=32, hkv=8, d=128, theta=5e5, dtype="bf16",
                                  sigma=2.0 ** -0.5, span_lens=[256] * 8, suffix_len=64,
                                  num_blocks=256, seed=seed)


# --------------------------------------------------------------------------- config 3
def rag_partial_prefill(*, name: str = "c3_rag_partial_prefill", seed: int = 2, hq: int = 32, hkv: int = 8,
                        d: int = 128, theta: float = 5e5, dtype: str = "bf16", sigma: float = 1.0,
                        pool_spans: int = 200, span_min: int = 128, span_max: int = 512,
                        num_reqs: int = 32, spans_per_req: int = 10, prefix_len: int = 32,
                        suffix_len: int = 64, uncached_per_req: int = 1) -> Workload:
    """BASELINE configs[2]: batched partial prefill with cache reuse.

    A pool of spans is resident in shared blocks; each request = shared system prefix +
    ``spans_per_req`` pool spans in draw order + question suffix.  ``uncached_per_req`` of the
    request's spans are *not* cached: fresh K/V of that span's padded length in private blocks.
    Queries = uncached span(s) (span-local causal) + suffix (sees everything).
    """
    rng = np.random.default_rng(seed)
    lens = [_round_up(int(x)) for x in rng.integers(span_min, span_max + 1, size=pool_spans)]
    new_tokens = num_reqs * (uncached_per_req * _round_up(span_max) + suffix_len)
    num_blocks = (sum(lens) + _round_up(prefix_len) + new_tokens) // BLOCK + 64
    c = _Composer(rng, num_blocks, hkv, d, dtype, sigma)
    prefix_blocks = c.tokens(prefix_len, resident=True, tag="prefix") if prefix_len else None
    pool = [c.tokens(L, resident=True, tag=f"span{i}") for i, L in enumerate(lens)]
    reqs = []
    for r in range(num_reqs):
        pick = rng.choice(pool_spans, size=spans_per_req, replace=False)
        unc = set(rng.choice(spans_per_req, size=uncached_per_req, replace=False).tolist())
        segs = []
        if prefix_len:
            segs.append(_Seg(prefix_blocks, prefix_len, local=False, query=False))
        for i, sp in enumerate(pick):
            L = lens[int(sp)]
            if i in unc:
                segs.append(_Seg(c.tokens(L, resident=False), L, local=True, query=True))
            else:
                segs.append(_Seg(pool[int(sp)], L, local=True, query=False))
        segs.append(_Seg(c.tokens(suffix_len, resident=False), suffix_len, local=False, query=True))
        reqs.append(segs)
    lay = _layout(reqs)
    q = _draw(rng, (int(lay["cu_q_lens"][-1]), hq, d), sigma, dtype)
    return Workload(name=name, kind="prefill", num_q_heads=hq, num_kv_heads=hkv, head_dim=d,
                    num_blocks=num_blocks, dtype=dtype, rope_theta=theta, resident=c.resident,
                    new=c.new_batch(), q=q, seed=seed, notes=dict(pool_span_lens=lens), **lay)


def config3(seed: int = 2) -> Workload:
    return rag_partial_prefill(seed=seed)


def question_over_context(ctx_spans: int = 64, span_len: int = 512, question: int = 64, seed: int = 8, **kw) -> Workload:
    """ONE request whose whole context (``ctx_spans`` spans of ``span_len`` tokens + the system prefix) is already cached:
    only the question's ``question`` tokens are computed (the partial prefill that sets TTFT once every chunk
    hits).  Few, long work items: the shape KV-range splits are for."""
    return rag_partial_prefill(name=f"question{question}_ctx{ctx_spans * span_len // 1024}k", seed=seed, num_reqs=1,
                               pool_spans=ctx_spans + 4, spans_per_req=ctx_spans, span_min=span_len, span_max=span_len,
                               uncached_per_req=0, suffix_len=question, **kw)


def epic_linked_prefill(*, name: str = "epic_linked_prefill", seed: int = 6, hq: int = 32, hkv: int = 8, d: int = 128,
                        theta: float = 5e5, dtype: str = "bf16", sigma: float = 1.0, pool_spans: int = 200,
                        span_min: int = 128, span_max: int = 512, num_reqs: int = 32, spans_per_req: int = 10,
                        prefix_len: int = 32, suffix_len: int = 64, link_tokens: int = 16) -> Workload:
    """EPIC / LegoLink through the same descriptor: every document is cached except its
    first ``link_tokens`` tokens (a block multiple: "with block-level granularity, k rounds to a block multiple"), which
    hash-depend on the preceding context and are RECOMPUTED inside the final prompt - they are queries that see everything
    before them (vis_lo = 0) and their fresh K/V go to private blocks; the rest of each document cache-hits from the shared
    pool.  Queries = the link tokens of every document + the question suffix."""
    if link_tokens % BLOCK:
        raise ValueError("link_tokens must be a block multiple")
    rng = np.random.default_rng(seed)
    lens = [max(_round_up(int(x)), link_tokens + BLOCK) for x in rng.integers(span_min, span_max + 1, size=pool_spans)]
    new_tokens = num_reqs * (spans_per_req * link_tokens + suffix_len)
    num_blocks = (sum(lens) + _round_up(prefix_len) + new_tokens) // BLOCK + 64
    c = _Composer(rng, num_blocks, hkv, d, dtype, sigma)
    prefix_blocks = c.tokens(prefix_len, resident=True, tag="prefix") if prefix_len else None
    pool = [c.tokens(L, resident=True, tag=f"span{i}") for i, L in enumerate(lens)]
    reqs = []
    for r in range(num_reqs):
        pick = rng.choice(pool_spans, size=spans_per_req, replace=False)
        segs = []
        if prefix_len:
            segs.append(_Seg(prefix_blocks, prefix_len, local=False, query=False))
        for sp in pick:
            L = lens[int(sp)]
            segs.append(_Seg(c.tokens(link_tokens, resident=False), link_tokens, local=False, query=True))
            segs.append(_Seg(pool[int(sp)][link_tokens // BLOCK:], L - link_tokens, local=True, query=False))
        segs.append(_Seg(c.tokens(suffix_len, resident=False), suffix_len, local=False, query=True))
        reqs.append(segs)
    lay = _layout(reqs)
    q = _draw(rng, (int(lay["cu_q_lens"][-1]), hq, d), sigma, dtype)
    return Workload(name=name, kind="prefill", num_q_heads=hq, num_kv_heads=hkv, head_dim=d,
                    num_blocks=num_blocks, dtype=dtype, rope_theta=theta, resident=c.resident,
                    new=c.new_batch(), q=q, seed=seed, notes=dict(pool_span_lens=lens, link_tokens=link_tokens), **lay)


def with_masked_keys(w: Workload, seed: int = 0, frac: float = 0.06) -> Workload:
    """Key-masking variant (minipic.h MINIPIC_KEY_MASK): a copy of ``w`` in which a random ``frac`` of the
    keys that are NOT query tokens - plus, per request, one whole 16-token block and sequence index 0 when they are not
    queries - carry logical position -1 (marker / padding tokens).  Run it with flags = MINIPIC_KEY_MASK."""
    rng = np.random.default_rng(seed)
    pos = w.kv_positions.copy()
    for r in range(w.num_reqs):
        n, o = int(w.kv_lens[r]), int(w.cu_kv_lens[r])
        is_q = np.zeros(n, bool)
        if w.kind == "prefill":
            is_q[w.q_seq_idx[int(w.cu_q_lens[r]):int(w.cu_q_lens[r + 1])]] = True
        else:
            is_q[n - 1] = True
        dead = (rng.random(n) < frac)
        b = int(rng.integers(0, max(n // BLOCK, 1))) * BLOCK
        dead[b:b + BLOCK] = True
        dead[0] = True
        dead &= ~is_q
        pos[o:o + n][dead] = -1
    return replace(w, name=w.name + "_keymask", kv_positions=pos, notes=dict(w.notes, key_mask=True))


# --------------------------------------------------------------------------- config 4
def shared_pool_decode(*, name: str = "c4_decode_shared_pool", seed: int = 3, hq: int = 32, hkv: int = 8,
                       d: int = 128, theta: float = 5e5, dtype: str = "bf16", sigma: float = 1.0,
                       num_seqs: int = 256, ctx_min: int = 4096, ctx_max: int = 8192,
                       span_len: int = 512, pool_spans: int = 64, private_pool: bool = False) -> Workload:
    """BASELINE configs[3]: decode over shared position-free blocks.

    Each context = n_full = (ctx-1)//span_len pool spans (drawn without replacement, placed
    consecutively from position 0) + a private tail of ctx - span_len*n_full tokens whose last
    token is the query; that token's K/V is the step's cache write.
    ``private_pool=True`` is control 4': identical shapes and values, every sequence's spans
    copied into private blocks (the write batches alias the pool arrays: no extra host memory).
    """
    rng = np.random.default_rng(seed)
    ctx = rng.integers(ctx_min, ctx_max + 1, size=num_seqs)
    n_full = (ctx - 1) // span_len
    tails = ctx - span_len * n_full
    shared_blocks = pool_spans * span_len // BLOCK
    private_blocks = int(sum(_round_up(int(t)) for t in tails)) // BLOCK
    copies = int(n_full.sum()) * span_len // BLOCK if private_pool else 0
    num_blocks = shared_blocks + private_blocks + copies + 64
    c = _Composer(rng, num_blocks, hkv, d, dtype, sigma)
    pool = [c.tokens(span_len, resident=True, tag=f"span{i}") for i in range(pool_spans)]
    pool_batches = list(c.resident)
    reqs = []
    for r in range(num_seqs):
        pick = rng.choice(pool_spans, size=int(n_full[r]), replace=False)
        segs = []
        for sp in pick:
            if private_pool:
                blocks = c.alloc(span_len)
                src = pool_batches[int(sp)]
                c.resident.append(WriteBatch(src.k, src.v, c.slots_of(blocks, span_len), f"copy{sp}"))
            else:
                blocks = pool[int(sp)]
            segs.append(_Seg(blocks, span_len, local=True, query=False))
        t = int(tails[r])
        blocks = c.alloc(t)
        k = _draw(rng, (t, hkv, d), sigma, dtype); v = _draw(rng, (t, hkv, d), sigma, dtype)
        slots = c.slots_of(blocks, t)
        if t > 1:
            c.resident.append(WriteBatch(k[:-1], v[:-1], slots[:-1], "tail"))
        c.new_k.append(k[-1:]); c.new_v.append(v[-1:]); c.new_slots.append(slots[-1:])
        segs.append(_Seg(blocks, t, local=False, query=False))
        reqs.append(segs)
    lay = _layout(reqs)
    kv_lens = lay["kv_lens"]
    lay["q_seq_idx"] = (kv_lens - 1).astype(np.int32)
    lay["q_vis_lo"] = np.zeros(num_seqs, np.int32)
    lay["cu_q_lens"] = np.arange(num_seqs + 1, dtype=np.int32)
    q = _draw(rng, (num_seqs, hq, d), sigma, dtype)
    return Workload(name=name + ("_private" if private_pool else ""), kind="decode", num_q_heads=hq,
                    num_kv_heads=hkv, head_dim=d, num_blocks=num_blocks, dtype=dtype, rope_theta=theta,
                    resident=c.resident, new=c.new_batch(), q=q, seed=seed, **lay)


def config4(seed: int = 3, private_pool: bool = False) -> Workload:
    return shared_pool_decode(seed=seed, private_pool=private_pool)


# --------------------------------------------------------------------------- config 5
def long_context_prefill(*, name: str = "c5_long_context_prefill", seed: int = 4, hq: int = 64, hkv: int = 8,
                         d: int = 128, theta: float = 5e5, dtype: str = "bf16", sigma: float = 1.0,
                         num_reqs: int = 4, slots_per_req: int = 64, span_len: int = 512,
                         suffix_len: int = 256, pool_spans: int = 64, cached_per_req: Optional[int] = None) -> Workload:
    """BASELINE configs[4]: long-context prefill, Llama-3-70B per-layer shapes.

    Each request holds ``slots_per_req`` span slots + suffix.  A random half of the slots hold
    cached spans drawn without replacement from a shared pool (so blocks recur across requests at
    different offsets); the other half are new (private blocks, part of the step's cache write).
    """
    rng = np.random.default_rng(seed)
    if cached_per_req is None:
        cached_per_req = slots_per_req // 2
    new_per_req = slots_per_req - cached_per_req
    num_blocks = (pool_spans * span_len + num_reqs * (new_per_req * span_len + _round_up(suffix_len))) // BLOCK + 64
    c = _Composer(rng, num_blocks, hkv, d, dtype, sigma)
    pool = [c.tokens(span_len, resident=True, tag=f"span{i}") for i in range(pool_spans)]
    reqs = []
    for r in range(num_reqs):
        cached_slots = set(rng.choice(slots_per_req, size=cached_per_req, replace=False).tolist())
        pick = iter(rng.choice(pool_spans, size=cached_per_req, replace=False).tolist())
        segs = []
        for s in range(slots_per_req):
            if s in cached_slots:
                segs.append(_Seg(pool[next(pick)], span_len, local=True, query=False))
            else:
                segs.append(_Seg(c.tokens(span_len, resident=False), span_len, local=True, query=True))
        segs.append(_Seg(c.tokens(suffix_len, resident=False), suffix_len, local=False, query=True))
        reqs.append(segs)
    lay = _layout(reqs)
    q = _draw(rng, (int(lay["cu_q_lens"][-1]), hq, d), sigma, dtype)
    return Workload(name=name, kind="prefill", num_q_heads=hq, num_kv_heads=hkv, head_dim=d,
                    num_blocks=num_blocks, dtype=dtype, rope_theta=theta, resident=c.resident,
                    new=c.new_batch(), q=q, seed=seed, **lay)


def config5(seed: int = 4) -> Workload:
    return long_context_prefill(seed=seed)


# --------------------------------------------------------------------------- reduced cases for CPU-speed parity
def small_variants(seed: int = 11) -> List[Workload]:
    """Reduced-size relatives of configs 2-5 that the oracle finishes in seconds while still
    spanning several 128-key tiles, ragged tails and shared blocks."""
    out = [
        single_request_prefill(name="s2_single", hq=8, hkv=2, d=128, theta=5e5, dtype="bf16", sigma=2.0 ** -0.5,
                               span_lens=[256, 144, 272], suffix_len=48, num_blocks=96, seed=seed),
        rag_partial_prefill(name="s3_rag", seed=seed + 1, hq=8, hkv=2, pool_spans=12, span_min=96, span_max=400,
                            num_reqs=5, spans_per_req=4, prefix_len=32, suffix_len=64),
        shared_pool_decode(name="s4_decode", seed=seed + 2, hq=8, hkv=2, num_seqs=9, ctx_min=300, ctx_max=1500,
                           span_len=128, pool_spans=12),
        long_context_prefill(name="s5_long", seed=seed + 3, hq=16, hkv=2, num_reqs=2, slots_per_req=6, span_len=256,
                             suffix_len=96, pool_spans=5),
    ]
    return out


def decode_from_prefill(w: Workload, seed: int = 0) -> Workload:
    """Re-use a prefill workload's cache + tables as a decode problem: one query per request at
    the last sequence index (used to test decode on fp32 / D=64 shapes)."""
    rng = np.random.default_rng(seed + 977)
    R = w.num_reqs
    q = _draw(rng, (R, w.num_q_heads, w.head_dim), 1.0, w.dtype)
    return Workload(name=w.name + "_as_decode", kind="decode", num_q_heads=w.num_q_heads,
                    num_kv_heads=w.num_kv_heads, head_dim=w.head_dim, num_blocks=w.num_blocks, dtype=w.dtype,
                    rope_theta=w.rope_theta, resident=w.resident, new=w.new, q=q,
                    block_tables=w.block_tables, cu_q_lens=np.arange(R + 1, dtype=np.int32), kv_lens=w.kv_lens,
                    cu_kv_lens=w.cu_kv_lens, kv_positions=w.kv_positions,
                    q_seq_idx=(w.kv_lens - 1).astype(np.int32), q_vis_lo=np.zeros(R, np.int32), seed=seed)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}
