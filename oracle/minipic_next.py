"""CPU ORACLE for the steps adjacent to the MiniPIC hot path.  TEST INFRASTRUCTURE - NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s CPU legs may import this file; it shares no code
with ``paper_2606_13126_b200/csrc`` and imports nothing from the package.  Plain numpy / hashlib, fp64.

* ``preattn_fused``   (f1) the step right before attention: the QKV-projection output of the new tokens is split, K and V
                      go UNROTATED into the paged cache through the slot mapping, Q is rotated once at the tokens' logical
                      positions and rounded to the I/O dtype ("rotated once by the model's RotaryEmbedding
                      layer ... stores unrotated key vectors"; Table 2 row rotary_embedding/base.py).
* ``block_rerotate``  (f4) what a POSITION-DEPENDENT cache has to do to reuse a span at a new offset: copy the block and
                      re-rotate its (already rotated, already rounded) keys by the position delta ("block-by-
                      block copy and repositioning"; App. A :284-286).  MiniPIC does none of this - it is the control.
* ``block_hashes`` / ``Pool`` (f3) Eq. 1: chained block hashes with SSEP (detach) and PDEP (depend on the
                      whole prompt) handled when the marker is the FIRST token of a block; a block pool keyed by hash
                      that turns token streams into block tables, slot mappings and the visibility descriptor.

Pins: tests/test_oracle_next_pins.py (``-m "not gpu"``).
"""
from __future__ import annotations

import hashlib

import numpy as np

from . import minipic_oracle as O

F64 = np.float64


# ----------------------------------------------------------------------------- f1
def preattn_fused(qkv: np.ndarray, slot_mapping: np.ndarray, positions: np.ndarray, k_cache: np.ndarray,
                  v_cache: np.ndarray, *, num_q_heads: int, num_kv_heads: int, dtype: str, rope_theta: float,
                  rotate_q: bool = True) -> np.ndarray:
    """qkv [T, Hq + 2 Hkv, D] in the I/O dtype: heads [0, Hq) are Q, [Hq, Hq + Hkv) are K, the rest V.

    1. K and V rows go into the paged cache bit for bit through ``slot_mapping`` (negative slot = skip): exactly
       ``cache_write`` - no rotation, no conversion.
    2. q'_t = R_{positions[t]} q_t in fp64, rounded ONCE to the I/O dtype (what the model's rotary layer hands to
       attention, consumed there with MINIPIC_Q_PREROTATED).  ``rotate_q=False`` returns Q unchanged.
    Returns q' as fp64 [T, Hq, D] (values exactly representable in the I/O dtype).
    """
    hq, hkv = num_q_heads, num_kv_heads
    O.cache_write(k_cache, v_cache, qkv[:, hq:hq + hkv, :], qkv[:, hq + hkv:hq + 2 * hkv, :], slot_mapping)
    q = O.to_f64(qkv[:, :hq, :], dtype)
    if not rotate_q:
        return q
    return O.round_to_dtype(O.rope_rotate(q, np.asarray(positions)[:, None], rope_theta), dtype)


# ----------------------------------------------------------------------------- f4
def block_rerotate(k_cache: np.ndarray, v_cache: np.ndarray, src_blocks: np.ndarray, dst_blocks: np.ndarray,
                   delta: np.ndarray, *, dtype: str, rope_theta: float) -> None:
    """For every i: K[dst_i] = round(R_{delta_i} K[src_i]) (all heads, all 16 tokens), V[dst_i] = V[src_i] bit for bit.

    The source keys are what a position-dependent cache holds: already rotated and already rounded to the I/O dtype;
    R composes additively in the position (R_a R_b = R_{a+b}), so rotating by the position DELTA repositions them.
    """
    for s, d, dl in zip(np.asarray(src_blocks), np.asarray(dst_blocks), np.asarray(delta)):
        k = O.to_f64(k_cache[int(s)], dtype)                                   # [Hkv, B, D]
        kr = O.round_to_dtype(O.rope_rotate(k, F64(dl), rope_theta), dtype)
        if dtype == "bf16":
            k_cache[int(d)] = (kr.astype(np.float32).view(np.uint32) >> np.uint32(16)).astype(np.uint16)
        else:
            k_cache[int(d)] = kr.astype(np.float32)
        v_cache[int(d)] = v_cache[int(s)]


# ----------------------------------------------------------------------------- f3
def _h(parent: bytes, tokens: np.ndarray) -> bytes:
    """H(parent, x) = SHA-256(parent || tokens as little-endian int32)."""
    return hashlib.sha256(parent + np.asarray(tokens, dtype="<i4").tobytes()).digest()


def seed_hash(seed: int) -> bytes:
    """h_0: the global seed constant of Eq. 1 = SHA-256 of the 8-byte little-endian seed."""
    return hashlib.sha256(int(seed).to_bytes(8, "little")).digest()


def block_hashes(tokens: np.ndarray, block_size: int, ssep: int, pdep: int, seed: int = 0) -> list:
    """Eq. 1 over the FULL blocks of a token stream (a trailing partial block has no hash):

        h_i = H(h_0, x_i)        if block i starts with SSEP      (detached from the chain)
              H(h_0, x_{<=i})    if block i starts with PDEP      (depends on the whole prompt so far)
              H(h_{i-1}, x_i)    otherwise                        (h_{-1} = h_0)
    """
    tokens = np.asarray(tokens)
    h0 = seed_hash(seed)
    out, prev = [], h0
    for i in range(len(tokens) // block_size):
        x = tokens[i * block_size:(i + 1) * block_size]
        if int(x[0]) == ssep:
            h = _h(h0, x)
        elif int(x[0]) == pdep:
            h = _h(h0, tokens[:(i + 1) * block_size])
        else:
            h = _h(prev, x)
        out.append(h)
        prev = h
    return out


def visibility(tokens: np.ndarray, block_size: int, ssep: int, pdep: int) -> np.ndarray:
    """vis_lo per token of a composed prompt (reading A6): a block that starts with SSEP opens a span whose
    tokens see [span start, self]; a block that starts with PDEP (and everything after it up to the next SSEP) sees
    [0, self]; tokens before the first marker see [0, self]."""
    tokens = np.asarray(tokens)
    lo = np.zeros(len(tokens), np.int32)
    cur = 0
    for i in range(0, len(tokens), block_size):
        t = int(tokens[i])
        if t == ssep:
            cur = i
        elif t == pdep:
            cur = 0
        lo[i:i + block_size] = cur
    return lo


class Pool:
    """Block pool keyed by the Eq. 1 hash: ``admit`` turns a token stream into (block table, hit flags, slot mapping of
    the tokens that must be written, vis_lo).  Blocks are handed out in increasing id order, never evicted (the tests
    size the pool to the stream); a trailing partial block always gets a fresh block."""

    def __init__(self, num_blocks: int, block_size: int, ssep: int, pdep: int, seed: int = 0):
        self.n, self.b, self.ssep, self.pdep, self.seed = num_blocks, block_size, ssep, pdep, seed
        self.by_hash = {}
        self.next = 0
        self.hits = self.misses = 0

    def _fresh(self) -> int:
        if self.next >= self.n:
            raise MemoryError("pool exhausted")
        self.next += 1
        return self.next - 1

    def admit(self, tokens: np.ndarray):
        tokens = np.asarray(tokens)
        hs = block_hashes(tokens, self.b, self.ssep, self.pdep, self.seed)
        nblk = (len(tokens) + self.b - 1) // self.b
        table = np.zeros(nblk, np.int32)
        hit = np.zeros(nblk, np.int8)
        slots = np.full(len(tokens), -1, np.int64)
        for i in range(nblk):
            lo, hi = i * self.b, min((i + 1) * self.b, len(tokens))
            if i < len(hs) and hs[i] in self.by_hash:
                table[i] = self.by_hash[hs[i]]; hit[i] = 1; self.hits += 1
                continue
            blk = self._fresh()
            if i < len(hs):
                self.by_hash[hs[i]] = blk
            table[i] = blk; self.misses += 1
            slots[lo:hi] = blk * self.b + np.arange(hi - lo)
        return table, hit, slots, visibility(tokens, self.b, self.ssep, self.pdep)
