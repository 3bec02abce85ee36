"""Pins of the oracle functions for the steps adjacent to the hot path: key masking, the fused
pre-attention step, the copy-and-re-rotate control and the Eq. 1 block hasher / pool.  CPU only.

Every pin is something other than the oracle's own formula retyped: pure-Python brute force with ``math``, torch's
bf16 cast, algebraic identities (R_a R_b = R_{a+b}, R_0 = I), "masking a key == deleting it", and hashlib digests
computed here from the definition of Eq. 1.
"""
import hashlib
import math

import numpy as np
import torch

from oracle import minipic_next as N
from oracle import minipic_oracle as O


def _bf16_bits(x32: np.ndarray) -> np.ndarray:
    return torch.from_numpy(np.ascontiguousarray(x32, np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)


def _bf16_round(x64: np.ndarray) -> np.ndarray:
    """fp64 -> nearest bf16 (ties to even) -> fp64, through torch's cast (fp64 -> bf16 is a single rounding there)."""
    return torch.from_numpy(np.ascontiguousarray(x64, np.float64)).to(torch.bfloat16).double().numpy()


# ----------------------------------------------------------------------------------------------- key masking (f2)
def _tiny_request(rng, kv_len, hq, hkv, d, nblk_pool=16):
    nb = (kv_len + 15) // 16
    bt = rng.permutation(nblk_pool)[:nb].astype(np.int32)[None, :]
    kc = O.new_cache(nblk_pool, hkv, 16, d, "f32"); vc = O.new_cache(nblk_pool, hkv, 16, d, "f32")
    k = rng.standard_normal((kv_len, hkv, d)).astype(np.float32); v = rng.standard_normal((kv_len, hkv, d)).astype(np.float32)
    slots = (bt[0][np.arange(kv_len) // 16].astype(np.int64) * 16 + np.arange(kv_len) % 16)
    O.cache_write(kc, vc, k, v, slots)
    q = rng.standard_normal((kv_len, hq, d)).astype(np.float32)
    return bt, kc, vc, k, v, q


def test_key_mask_equals_deleting_the_keys():
    """PAPER.md:294 (key zeroing, taken as a mask variant): a key with a negative logical position is invisible to every
    row.  Deleting those keys from the sequence (re-packed cache, remapped indices) must give the same rows."""
    rng = np.random.default_rng(5)
    kv_len, hq, hkv, d, theta = 75, 4, 2, 16, 1e4
    bt, kc, vc, k, v, q = _tiny_request(rng, kv_len, hq, hkv, d)
    pos = np.arange(kv_len, dtype=np.int32) + 7
    dead = np.zeros(kv_len, bool); dead[[0, 3, 16, 17, 40, 63, 74]] = True
    pos_m = np.where(dead, -1, pos).astype(np.int32)
    lo = np.where(np.arange(kv_len) < 32, 0, 32).astype(np.int32)          # two spans: [0, 32) and [32, 75)
    idx = np.arange(kv_len, dtype=np.int32)
    om, lm = O.prefill_attention(q=q, k_cache=kc, v_cache=vc, block_tables=bt, cu_q_lens=np.array([0, kv_len]),
                                 kv_lens=np.array([kv_len]), cu_kv_lens=np.array([0, kv_len]), kv_positions=pos_m,
                                 q_seq_idx=idx, q_vis_lo=lo, num_q_heads=hq, dtype="f32", rope_theta=theta, key_mask=True)
    # the same request with the dead keys physically removed
    keep = np.flatnonzero(~dead)
    new_of = -np.ones(kv_len, np.int64); new_of[keep] = np.arange(len(keep))
    n2 = len(keep)
    kc2 = O.new_cache(16, hkv, 16, d, "f32"); vc2 = O.new_cache(16, hkv, 16, d, "f32")
    bt2 = np.arange((n2 + 15) // 16, dtype=np.int32)[None, :]
    O.cache_write(kc2, vc2, k[keep], v[keep], np.arange(n2, dtype=np.int64))
    for t in range(kv_len):                                     # every query row, including rows whose own key is dead
        vis = [j for j in range(int(lo[t]), t + 1) if not dead[j]]
        if not vis:
            assert np.all(om[t] == 0) and np.all(np.isneginf(lm[t]))
            continue
        # query t rotated at ITS position attends to the kept keys new_of[vis]; in the packed request that is the index
        # range [new_of[vis[0]], new_of[vis[-1]]] (kept keys are contiguous there), with the query's own position passed
        # through a one-off "prerotated" q
        qr = O.rope_rotate(q[t].astype(np.float64), np.float64(pos_m[t]), theta)[None]     # a dead token queries at the position it was given
        o2, l2 = O.prefill_attention(q=qr.astype(np.float64), k_cache=kc2, v_cache=vc2, block_tables=bt2,
                                     cu_q_lens=np.array([0, 1]), kv_lens=np.array([n2]), cu_kv_lens=np.array([0, n2]),
                                     kv_positions=pos[keep], q_seq_idx=np.array([new_of[vis[-1]]], np.int32),
                                     q_vis_lo=np.array([new_of[vis[0]]], np.int32), num_q_heads=hq, dtype="f32",
                                     rope_theta=theta, q_prerotated=True)
        # (q passed as float64 through to_f64's float32 cast: compare with fp32-level tolerance)
        assert np.allclose(om[t], o2[0], atol=2e-6) and np.allclose(lm[t], l2[0], atol=2e-6), t


def test_key_mask_brute_force_and_off_switch():
    rng = np.random.default_rng(6)
    kv_len, hq, hkv, d, theta = 21, 2, 1, 8, 1e4
    bt, kc, vc, k, v, q = _tiny_request(rng, kv_len, hq, hkv, d)
    pos = np.arange(kv_len, dtype=np.int32)
    pos_m = pos.copy(); pos_m[[2, 9, 20]] = -5
    args = dict(q=q, k_cache=kc, v_cache=vc, block_tables=bt, cu_q_lens=np.array([0, kv_len]), kv_lens=np.array([kv_len]),
                cu_kv_lens=np.array([0, kv_len]), q_seq_idx=pos, q_vis_lo=np.zeros(kv_len, np.int32), num_q_heads=hq,
                dtype="f32", rope_theta=theta)
    om, lm = O.prefill_attention(kv_positions=pos_m, key_mask=True, **args)
    f = [theta ** (-2.0 * i / d) for i in range(d // 2)]

    def rot(x, p):
        y = [0.0] * d
        for i in range(d // 2):
            c, s = math.cos(p * f[i]), math.sin(p * f[i])
            y[i] = x[i] * c - x[i + d // 2] * s
            y[i + d // 2] = x[i + d // 2] * c + x[i] * s
        return y
    for t in (1, 5, 9, 20):
        for h in range(hq):
            qq = rot([float(z) for z in q[t, h]], int(pos_m[t]))          # a dead token still queries at its own position
            sc, vs = [], []
            for j in range(t + 1):
                if pos_m[j] < 0:
                    continue
                kk = rot([float(z) for z in k[j, 0]], int(pos_m[j]))
                sc.append(sum(a * b for a, b in zip(qq, kk)) / math.sqrt(d)); vs.append(v[j, 0])
            m = max(sc); w = [math.exp(x - m) for x in sc]; l = sum(w)
            o = sum(wi * vi.astype(np.float64) for wi, vi in zip(w, vs)) / l
            assert np.allclose(om[t, h], o, atol=1e-12) and abs(lm[t, h] - (m + math.log(l))) < 1e-12
    # switched off, negative positions are ordinary positions (the flag, not the sign, turns the mask on)
    o0, l0 = O.prefill_attention(kv_positions=pos_m, key_mask=False, **args)
    assert not np.allclose(o0[20], om[20])


# ----------------------------------------------------------------------------------------------- fused pre-attention (f1)
def test_preattn_fused_brute_force_bf16():
    """Q rotated once at the token's logical position, K / V stored UNROTATED, bit for bit."""
    rng = np.random.default_rng(8)
    T, hq, hkv, d, theta = 9, 4, 2, 8, 5e5
    x = rng.standard_normal((T, hq + 2 * hkv, d)).astype(np.float32)
    bits = _bf16_bits(x)
    xb = O.bf16_bits_to_f64(bits)
    pos = np.array([0, 1, 2, 100, 101, 33000, 7, 7, 65535], np.int32)
    slots = np.array([16 * 3 + 0, 16 * 3 + 1, -1, 5, 16 * 7 + 15, 0, 16 * 2 + 4, 16 * 2 + 5, 16 * 8 + 2], np.int64)
    kc = O.new_cache(9, hkv, 16, d, "bf16", fill=0xABCD); vc = O.new_cache(9, hkv, 16, d, "bf16", fill=0xABCD)
    qr = N.preattn_fused(bits, slots, pos, kc, vc, num_q_heads=hq, num_kv_heads=hkv, dtype="bf16", rope_theta=theta)
    # cache: written slots hold the K / V bit patterns, every other slot keeps the sentinel
    touched = np.zeros((9, 16), bool)
    for t in range(T):
        if slots[t] < 0:
            continue
        b, o = divmod(int(slots[t]), 16)
        touched[b, o] = True
        assert np.array_equal(kc[b, :, o, :], bits[t, hq:hq + hkv]) and np.array_equal(vc[b, :, o, :], bits[t, hq + hkv:])
    untouched = np.transpose(kc, (0, 2, 1, 3))[~touched], np.transpose(vc, (0, 2, 1, 3))[~touched]
    assert np.all(untouched[0] == 0xABCD) and np.all(untouched[1] == 0xABCD)
    # Q: brute force in Python floats, rounded by torch's bf16 cast
    want = np.zeros((T, hq, d))
    for t in range(T):
        for h in range(hq):
            for i in range(d // 2):
                phi = float(pos[t]) * theta ** (-2.0 * i / d)
                a, b = float(xb[t, h, i]), float(xb[t, h, i + d // 2])
                want[t, h, i] = a * math.cos(phi) - b * math.sin(phi)
                want[t, h, i + d // 2] = b * math.cos(phi) + a * math.sin(phi)
    assert np.array_equal(qr, _bf16_round(want))
    assert np.array_equal(qr[0], xb[0, :hq])                      # R_0 = I: position 0 returns Q bit for bit
    q0 = N.preattn_fused(bits, -np.ones(T, np.int64), pos, kc, vc, num_q_heads=hq, num_kv_heads=hkv, dtype="bf16",
                         rope_theta=theta, rotate_q=False)
    assert np.array_equal(q0, xb[:, :hq])


def test_preattn_fused_then_attention_equals_plain_path():
    """Attention on (q' from the fused step, Q_PREROTATED) == attention on raw q with in-attention Q rotation, up to the one
    bf16 rounding of q' (mode Q rounds q' too, so the two agree exactly there once K is rounded the same way)."""
    rng = np.random.default_rng(9)
    T, hq, hkv, d, theta = 48, 4, 2, 16, 1e4
    bits = _bf16_bits(rng.standard_normal((T, hq + 2 * hkv, d)).astype(np.float32))
    pos = (np.arange(T) + 11).astype(np.int32)
    bt = np.array([[2, 0, 1]], np.int32)
    slots = bt[0][np.arange(T) // 16].astype(np.int64) * 16 + np.arange(T) % 16
    kc = O.new_cache(3, hkv, 16, d, "bf16"); vc = O.new_cache(3, hkv, 16, d, "bf16")
    qr = N.preattn_fused(bits, slots, pos, kc, vc, num_q_heads=hq, num_kv_heads=hkv, dtype="bf16", rope_theta=theta)
    qr_bits = (qr.astype(np.float32).view(np.uint32) >> 16).astype(np.uint16)
    common = dict(k_cache=kc, v_cache=vc, block_tables=bt, cu_q_lens=np.array([0, T]), kv_lens=np.array([T]),
                  cu_kv_lens=np.array([0, T]), kv_positions=pos, q_seq_idx=np.arange(T, dtype=np.int32),
                  q_vis_lo=np.zeros(T, np.int32), num_q_heads=hq, dtype="bf16", rope_theta=theta, mode="Q")
    o1, l1 = O.prefill_attention(q=qr_bits, q_prerotated=True, **common)
    o2, l2 = O.prefill_attention(q=bits[:, :hq], **common)
    assert np.allclose(o1, o2, atol=1e-12) and np.allclose(l1, l2, atol=1e-12)


# ----------------------------------------------------------------------------------------------- copy-and-re-rotate (f4)
def test_block_rerotate_composition_and_brute_force():
    """repositioning a cached span = copy + rotation by the position delta; R_a R_b = R_{a+b}."""
    rng = np.random.default_rng(10)
    hkv, d, theta = 2, 16, 5e5
    k = rng.standard_normal((16, hkv, d))                       # one block of unrotated keys, fp64
    p0 = 4096 + np.arange(16)
    # fp32 cache: composition identity to fp32 rounding (two roundings vs one)
    kc = O.new_cache(4, hkv, 16, d, "f32"); vc = O.new_cache(4, hkv, 16, d, "f32")
    kc[1] = np.transpose(O.rope_rotate(k, p0[:, None], theta), (1, 0, 2)).astype(np.float32)
    vc[1] = rng.standard_normal((hkv, 16, d)).astype(np.float32)
    N.block_rerotate(kc, vc, np.array([1, 1]), np.array([3, 0]), np.array([777, 0]), dtype="f32", rope_theta=theta)
    want = np.transpose(O.rope_rotate(k, (p0 + 777)[:, None], theta), (1, 0, 2))
    assert np.allclose(kc[3], want, atol=5e-6) and np.array_equal(vc[3], vc[1])
    assert np.array_equal(kc[0], kc[1]) and np.array_equal(vc[0], vc[1])      # delta 0: a plain copy, bit for bit
    # bf16: brute force on the stored (rounded) values, rounded by torch
    kb = _bf16_bits(np.transpose(O.rope_rotate(k, p0[:, None], theta), (1, 0, 2)).astype(np.float32))
    kc2 = O.new_cache(2, hkv, 16, d, "bf16"); vc2 = O.new_cache(2, hkv, 16, d, "bf16")
    kc2[0] = kb; vc2[0] = _bf16_bits(rng.standard_normal((hkv, 16, d)).astype(np.float32))
    N.block_rerotate(kc2, vc2, np.array([0]), np.array([1]), np.array([-1234]), dtype="bf16", rope_theta=theta)
    src = O.bf16_bits_to_f64(kb)
    want = np.zeros_like(src)
    for h in range(hkv):
        for t in range(16):
            for i in range(d // 2):
                phi = -1234.0 * theta ** (-2.0 * i / d)
                a, b = src[h, t, i], src[h, t, i + d // 2]
                want[h, t, i] = a * math.cos(phi) - b * math.sin(phi)
                want[h, t, i + d // 2] = b * math.cos(phi) + a * math.sin(phi)
    assert np.array_equal(O.bf16_bits_to_f64(kc2[1]), _bf16_round(want)) and np.array_equal(vc2[1], vc2[0])


# ----------------------------------------------------------------------------------------------- Eq. 1 hasher / pool (f3)
SSEP, PDEP, PAD = 9001, 9002, 9000


def _sha(parent: bytes, toks) -> bytes:
    return hashlib.sha256(parent + b"".join(int(t).to_bytes(4, "little", signed=True) for t in toks)).digest()


def test_block_hashes_follow_eq1():
    rng = np.random.default_rng(12)
    B = 16
    sys_p = rng.integers(0, 5000, 2 * B)
    doc = lambda n: np.concatenate([[SSEP], rng.integers(0, 5000, n * B - 1)])
    d1, d2 = doc(3), doc(2)
    task = np.concatenate([[PDEP], rng.integers(0, 5000, B + 4)])          # trailing partial block: no hash
    prompt = np.concatenate([sys_p, d1, d2, task])
    hs = N.block_hashes(prompt, B, SSEP, PDEP, seed=42)
    assert len(hs) == len(prompt) // B == 8
    h0 = hashlib.sha256((42).to_bytes(8, "little")).digest()
    blk = lambda i: prompt[i * B:(i + 1) * B]
    assert hs[0] == _sha(h0, blk(0)) and hs[1] == _sha(hs[0], blk(1))        # ordinary chain from the seed
    assert hs[2] == _sha(h0, blk(2))                                          # SSEP: detached
    assert hs[3] == _sha(hs[2], blk(3)) and hs[4] == _sha(hs[3], blk(4))      # ... chain continues inside the span
    assert hs[5] == _sha(h0, blk(5)) and hs[6] == _sha(hs[5], blk(6))
    assert hs[7] == _sha(h0, prompt[:8 * B])                                  # PDEP: the whole prompt so far
    # a span hashes the same wherever it appears and whatever precedes it (the point of SSEP) ...
    alone = N.block_hashes(d1, B, SSEP, PDEP, seed=42)
    assert alone == hs[2:5]
    swapped = N.block_hashes(np.concatenate([sys_p, d2, d1, task]), B, SSEP, PDEP, seed=42)
    assert swapped[4:7] == hs[2:5] and swapped[2:4] == hs[5:7]
    # ... the PDEP block does not (false-hit protection), and neither do ordinary blocks after a changed prefix
    assert swapped[7] != hs[7]
    p2 = prompt.copy(); p2[1] += 1
    h2 = N.block_hashes(p2, B, SSEP, PDEP, seed=42)
    assert h2[0] != hs[0] and h2[1] != hs[1] and h2[2:7] == hs[2:7] and h2[7] != hs[7]
    assert N.block_hashes(prompt, B, SSEP, PDEP, seed=43)[2] != hs[2]         # the seed is part of every hash
    # a marker that is NOT the first token of its block has no effect on the rule
    p3 = prompt.copy(); p3[B + 3] = SSEP
    h3 = N.block_hashes(p3, B, SSEP, PDEP, seed=42)
    assert h3[1] == _sha(h3[0], p3[B:2 * B])


def test_pool_derives_tables_slots_and_mask():
    rng = np.random.default_rng(13)
    B = 16
    pool = N.Pool(64, B, SSEP, PDEP, seed=1)
    sys_p = rng.integers(0, 5000, B)
    docs = [np.concatenate([[SSEP], rng.integers(0, 5000, n * B - 1)]) for n in (2, 3, 1)]
    # step 3 of PAPER.md:123-128: every padded document (and the system prompt) is prefilled as its own request
    t_sys, hit, slots, lo = pool.admit(sys_p)
    assert hit.tolist() == [0] and np.array_equal(slots, t_sys[0] * B + np.arange(B)) and np.all(lo == 0)
    tables = []
    for dd in docs:
        t, hit, slots, lo = pool.admit(dd)
        assert not hit.any() and np.all(lo == 0) and np.all(slots >= 0)      # a span alone: local causal from its start
        tables.append(t)
    # step 4: the final prompt - system + docs in another order + PDEP task; only the task is a miss
    task = np.concatenate([[PDEP], rng.integers(0, 5000, 20)])
    order = [2, 0, 1]
    prompt = np.concatenate([sys_p] + [docs[i] for i in order] + [task])
    t, hit, slots, lo = pool.admit(prompt)
    want_tab = np.concatenate([t_sys] + [tables[i] for i in order])
    assert np.array_equal(t[:len(want_tab)], want_tab) and hit[:len(want_tab)].all() and not hit[len(want_tab):].any()
    n_hit = len(want_tab) * B
    assert np.all(slots[:n_hit] == -1) and np.all(slots[n_hit:] >= 0)
    assert len(set(t[len(want_tab):].tolist()) & set(want_tab.tolist())) == 0
    # visibility: system prefix sees from 0, each document from its own start, the PDEP task from 0
    starts = np.cumsum([B] + [len(docs[i]) for i in order])
    assert np.all(lo[:B] == 0)
    for s0, i in zip(starts[:-1], order):
        assert np.all(lo[s0:s0 + len(docs[i])] == s0)
    assert np.all(lo[starts[-1]:] == 0)
    # the same final prompt again: the PDEP block hits too now (same whole-prompt hash), the partial tail never does
    t2, hit2, slots2, _ = pool.admit(prompt)
    assert hit2[:-1].all() and hit2[-1] == 0 and np.array_equal(t2[:-1], t[:-1]) and t2[-1] != t[-1]
    assert pool.hits > 0 and pool.misses > 0
