"""Pins for the CPU oracle (oracle/minipic_oracle.py): everything here is `-m "not gpu"`.

Each test checks the oracle against something that is NOT the oracle: a closed form, a pure-Python
brute force written separately, an invariant of the mathematics, or a library routine
(torch fp64 scaled_dot_product_attention).  Citations are PAPER.md:<line>.
"""
import cmath
import math
import os

import numpy as np
import pytest
import torch

from oracle import minipic_oracle as O
from paper_2606_13126_b200 import workloads as W

B = 16


# --------------------------------------------------------------------------- helpers (independent restatements)
def brute_force(q, k, v, pos, idx, lo, theta, hq, hkv):
    """Pure-Python loops: explicit 2x2 rotations per frequency pair, dense mask, textbook softmax.
    q [Tq][hq][D], k/v [T][hkv][D] (already gathered in sequence order), pos [T]."""
    tq, d = len(q), len(q[0][0])
    half = d // 2
    g = hq // hkv

    def rot(x, p):
        y = [0.0] * d
        for i in range(half):
            f = theta ** (-2.0 * i / d)
            c, s = math.cos(p * f), math.sin(p * f)
            y[i] = x[i] * c - x[i + half] * s
            y[i + half] = x[i] * s + x[i + half] * c
        return y

    out = [[[0.0] * d for _ in range(hq)] for _ in range(tq)]
    lse = [[-math.inf] * hq for _ in range(tq)]
    for t in range(tq):
        for h in range(hq):
            qr = rot(q[t][h], pos[idx[t]])
            scores = []
            for j in range(len(k)):
                if lo[t] <= j <= idx[t]:
                    kr = rot(k[j][h // g], pos[j])
                    scores.append((j, sum(a * b for a, b in zip(qr, kr)) / math.sqrt(d)))
            if not scores:
                continue
            m = max(s for _, s in scores)
            z = sum(math.exp(s - m) for _, s in scores)
            lse[t][h] = m + math.log(z)
            for j, s in scores:
                p = math.exp(s - m) / z
                for e in range(d):
                    out[t][h][e] += p * v[j][h // g][e]
    return np.array(out), np.array(lse)


def complex_rope(x, p, theta):
    """RoFormer's complex form: z_i = x_i + i x_{i+D/2}; z_i <- z_i * exp(i p f_i)."""
    d = x.shape[-1]
    half = d // 2
    y = np.empty_like(x, dtype=np.float64)
    for i in range(half):
        w = cmath.exp(1j * p * theta ** (-2.0 * i / d))
        z = complex(x[i], x[i + half]) * w
        y[i], y[i + half] = z.real, z.imag
    return y


def dense_request(rng, T, hq, hkv, d, dtype="f32"):
    k = rng.standard_normal((T, hkv, d)).astype(np.float32)
    v = rng.standard_normal((T, hkv, d)).astype(np.float32)
    q = rng.standard_normal((T, hq, d)).astype(np.float32)
    if dtype == "bf16":
        k, v, q = (W.f32_to_bf16_bits(a) for a in (k, v, q))
    return q, k, v


def paged(k, v, blocks, num_blocks, dtype="f32"):
    """Place dense [T,hkv,d] K/V into a paged oracle cache via the oracle's cache_write."""
    T, hkv, d = k.shape
    kc = O.new_cache(num_blocks, hkv, B, d, dtype)
    vc = O.new_cache(num_blocks, hkv, B, d, dtype)
    t = np.arange(T)
    slots = np.asarray(blocks, np.int64)[t // B] * B + t % B
    O.cache_write(kc, vc, k, v, slots)
    return kc, vc


def one_request(q, kc, vc, blocks, pos, idx, lo, hq, theta, dtype="f32", **kw):
    T = len(pos)
    return O.prefill_attention(q=q, k_cache=kc, v_cache=vc, block_tables=np.asarray([blocks], np.int32),
                               cu_q_lens=np.array([0, q.shape[0]]), kv_lens=np.array([T]),
                               cu_kv_lens=np.array([0, T]), kv_positions=np.asarray(pos, np.int32),
                               q_seq_idx=np.asarray(idx, np.int32), q_vis_lo=np.asarray(lo, np.int32),
                               num_q_heads=hq, dtype=dtype, rope_theta=theta, **kw)


# --------------------------------------------------------------------------- cache write / indexing
def test_cache_write_bit_exact_and_untouched_slots():
    """raw scatter; K is NOT rotated on write; untouched slots keep a sentinel."""
    rng = np.random.default_rng(5)
    hkv, d, nb = 2, 8, 6
    for dtype, sentinel in (("bf16", 0xBEEF), ("f32", -7.25)):
        kc = O.new_cache(nb, hkv, B, d, dtype, sentinel)
        vc = O.new_cache(nb, hkv, B, d, dtype, sentinel)
        T = 40
        if dtype == "bf16":
            k = rng.integers(0, 65536, (T, hkv, d)).astype(np.uint16)   # every bit pattern incl. NaNs
            v = rng.integers(0, 65536, (T, hkv, d)).astype(np.uint16)
        else:
            k = rng.standard_normal((T, hkv, d)).astype(np.float32)
            v = rng.standard_normal((T, hkv, d)).astype(np.float32)
        slots = rng.permutation(nb * B)[:T].astype(np.int64)
        slots[3] = -1
        slots[17] = -5
        O.cache_write(kc, vc, k, v, slots)
        written = np.zeros((nb, B), bool)
        for t, s in enumerate(slots):
            if s < 0:
                continue
            written[s // B, s % B] = True
            for h in range(hkv):
                assert kc[s // B, h, s % B].tobytes() == k[t, h].tobytes()
                assert vc[s // B, h, s % B].tobytes() == v[t, h].tobytes()
        sent = np.asarray(sentinel, kc.dtype)
        for blk in range(nb):
            for off in range(B):
                if not written[blk, off]:
                    assert (kc[blk, :, off] == sent).all() and (vc[blk, :, off] == sent).all()
        assert written.sum() == T - 2


def test_gather_reads_through_block_table():
    """blk = bt[j // B], row = j % B: gathering returns the dense rows in order."""
    rng = np.random.default_rng(6)
    q, k, v = dense_request(rng, 50, 2, 2, 8)
    blocks = [9, 2, 7, 4]
    kc, vc = paged(k, v, blocks, 12)
    for h in range(2):
        kk, vv = O.gather_kv(kc, vc, np.asarray(blocks), 50, h, "f32")
        assert np.array_equal(kk, k[:, h].astype(np.float64)) and np.array_equal(vv, v[:, h].astype(np.float64))


def test_block_permutation_invariance_bit_for_bit():
    """Physical block ids are arbitrary names: permuting them (and the table
    consistently) leaves the oracle's output unchanged bit for bit."""
    rng = np.random.default_rng(7)
    T, hq, hkv, d = 70, 4, 2, 16
    q, k, v = dense_request(rng, T, hq, hkv, d)
    pos, idx, lo = np.arange(T), np.arange(T), np.zeros(T, int)
    ref = None
    for trial in range(3):
        blocks = rng.permutation(20)[:5]
        kc, vc = paged(k, v, blocks, 20)
        out = one_request(q, kc, vc, blocks, pos, idx, lo, hq, 1e4)
        if ref is None:
            ref = out
        else:
            assert out[0].tobytes() == ref[0].tobytes() and out[1].tobytes() == ref[1].tobytes()


# --------------------------------------------------------------------------- RoPE closed forms
def test_rope_identity_norm_and_relative_property():
    rng = np.random.default_rng(8)
    for d, theta in ((64, 1e4), (128, 5e5), (2, 10.0)):
        x = rng.standard_normal((5, d))
        y = rng.standard_normal((5, d))
        assert np.array_equal(O.rope_rotate(x, np.zeros(5), theta), x)                       # R(0) = I
        for p in (1, 17, 4096, 33023):
            rx = O.rope_rotate(x, np.full(5, p), theta)
            assert np.allclose(np.linalg.norm(rx, axis=-1), np.linalg.norm(x, axis=-1), rtol=1e-13)
            for a in (0, 3, 2048):                                                            # (R(a)x).(R(a+p)y) = x.(R(p)y)
                lhs = (O.rope_rotate(x, np.full(5, a), theta) * O.rope_rotate(y, np.full(5, a + p), theta)).sum(-1)
                rhs = (x * O.rope_rotate(y, np.full(5, p), theta)).sum(-1)
                assert np.allclose(lhs, rhs, rtol=0, atol=1e-9)
        # composition R(a)R(b) = R(a+b)
        assert np.allclose(O.rope_rotate(O.rope_rotate(x, np.full(5, 5), theta), np.full(5, 11), theta),
                           O.rope_rotate(x, np.full(5, 16), theta), atol=1e-12)


def test_rope_matches_complex_form_and_pairing():
    """Rotate-half pairing (i, i+D/2) with f_i = theta^(-2i/D) (readings A1, A2), against RoFormer's
    complex multiplication written separately; a transposed pairing or wrong sign fails."""
    rng = np.random.default_rng(9)
    for d, theta in ((8, 1e4), (128, 5e5)):
        x = rng.standard_normal(d)
        for p in (1, 5, 1000, 33023):
            assert np.allclose(O.rope_rotate(x, np.asarray(p), theta), complex_rope(x, p, theta), atol=1e-10)
    # explicit small case: D=4, p=1, theta=100 -> f = [1, 0.1]
    x = np.array([1.0, 2.0, 3.0, 4.0])
    y = O.rope_rotate(x, np.asarray(1), 100.0)
    exp = np.array([1 * math.cos(1) - 3 * math.sin(1), 2 * math.cos(.1) - 4 * math.sin(.1),
                    3 * math.cos(1) + 1 * math.sin(1), 4 * math.cos(.1) + 2 * math.sin(.1)])
    assert np.allclose(y, exp, atol=1e-14)
    assert np.allclose(O.rope_frequencies(4, 100.0), [1.0, 0.1], rtol=1e-15)


def test_golden_d2_closed_form_scores():
    """Eq. 2 at D=2 (single frequency 1): score = |q||k| cos(p_j - p_t + arg k - arg q)/sqrt(2).
    The score is read back from the oracle through a two-key softmax: key 0 = k at p_j with v=1,
    key 1 = the query's own token with k=0 (score 0) and v=0, so out = sigmoid(score), lse = ln(1+e^s)."""
    path = os.path.join(os.path.dirname(__file__), "golden", "rope_d2_closed_form.txt")
    rows = [l.split() for l in open(path) if not l.startswith("#")]
    assert len(rows) >= 5
    for r in rows:
        pt, pj = int(r[0]), int(r[1])
        qv, kv, s = (float(r[2]), float(r[3])), (float(r[4]), float(r[5])), float(r[6])
        k = np.zeros((2, 1, 2), np.float32); k[0, 0] = kv
        v = np.zeros((2, 1, 2), np.float32); v[0, 0] = (1.0, 1.0)
        kc, vc = paged(k, v, [3], 5)
        q = np.asarray([[qv]], np.float32)
        out, lse = one_request(q, kc, vc, [3], [pj, pt], [1], [0], 1, 777.0)
        assert abs(math.log(math.expm1(lse[0, 0])) - s) < 1e-9
        assert abs(out[0, 0, 0] - 1.0 / (1.0 + math.exp(-s))) < 1e-10


def test_shift_invariance_of_logical_positions():
    """a span prefilled at offset 0 is reusable at offset 2048 - adding a constant
    to all logical positions of a request leaves every score unchanged (to fp64 precision)."""
    rng = np.random.default_rng(10)
    T, hq, hkv, d = 96, 4, 2, 64
    q, k, v = dense_request(rng, T, hq, hkv, d)
    blocks = rng.permutation(10)[:6]
    kc, vc = paged(k, v, blocks, 10)
    idx = np.arange(T); lo = np.where(idx < 48, 0, 48)
    base = one_request(q, kc, vc, blocks, np.arange(T), idx, lo, hq, 5e5)
    for c in (1, 2048, 4096, 10 ** 6):
        sh = one_request(q, kc, vc, blocks, np.arange(T) + c, idx, lo, hq, 5e5)
        assert np.abs(sh[1] - base[1]).max() < 1e-9 and np.abs(sh[0] - base[0]).max() < 1e-9
    # and a non-constant change of positions DOES change the result (the test can fail)
    pos2 = np.arange(T).copy(); pos2[10] += 3
    ch = one_request(q, kc, vc, blocks, pos2, idx, lo, hq, 5e5)
    assert np.abs(ch[1] - base[1]).max() > 1e-4


# --------------------------------------------------------------------------- attention vs brute force / library
@pytest.mark.parametrize("seed,T,hq,hkv,d,theta", [(0, 37, 2, 1, 8, 1e4), (1, 50, 4, 2, 4, 5e5), (2, 20, 3, 3, 16, 1e4)])
def test_attention_matches_pure_python_brute_force(seed, T, hq, hkv, d, theta):
    rng = np.random.default_rng(seed)
    q, k, v = dense_request(rng, T, hq, hkv, d)
    blocks = rng.permutation(9)[:-(-T // B)]
    kc, vc = paged(k, v, blocks, 9)
    pos = np.arange(T) + int(rng.integers(0, 100))
    # span structure: two local spans then a suffix that sees all
    idx = np.arange(T)
    s1, s2 = T // 3, 2 * T // 3
    lo = np.where(idx < s1, 0, np.where(idx < s2, s1, 0))
    qsel = np.array([0, 1, s1 - 1, s1, s1 + 2, s2 - 1, s2, T - 1])
    out, lse = one_request(q[qsel], kc, vc, blocks, pos, idx[qsel], lo[qsel], hq, theta)
    bo, bl = brute_force(q[qsel].tolist(), k.tolist(), v.tolist(), pos.tolist(), idx[qsel].tolist(),
                         lo[qsel].tolist(), theta, hq, hkv)
    assert np.abs(out - bo).max() < 1e-11 and np.abs(lse - bl).max() < 1e-11


def test_rotate_on_read_equals_prerotated_cache_via_library_sdpa():
    """in-kernel rotation is algebraically equivalent to a pre-rotated cache.  The
    pre-rotated side is dense K rotated with the complex form (written separately) and fed, with an
    explicit boolean mask, to torch's fp64 scaled_dot_product_attention (a library routine)."""
    rng = np.random.default_rng(11)
    T, hq, hkv, d, theta = 80, 4, 2, 32, 5e5
    q, k, v = dense_request(rng, T, hq, hkv, d)
    blocks = rng.permutation(8)[:5]
    kc, vc = paged(k, v, blocks, 8)
    pos = np.arange(T) + 300
    idx = np.arange(T); lo = np.where(idx < 32, 0, np.where(idx < 64, 32, 0))
    out, lse = one_request(q, kc, vc, blocks, pos, idx, lo, hq, theta)
    kr = np.array([[complex_rope(k[j, h].astype(np.float64), int(pos[j]), theta) for h in range(hkv)] for j in range(T)])
    qr = np.array([[complex_rope(q[t, h].astype(np.float64), int(pos[t]), theta) for h in range(hq)] for t in range(T)])
    mask = torch.from_numpy((np.arange(T)[None, :] >= lo[:, None]) & (np.arange(T)[None, :] <= idx[:, None]))
    g = hq // hkv
    Q = torch.from_numpy(qr).permute(1, 0, 2)[None]                                  # [1,hq,T,d]
    K = torch.from_numpy(kr).permute(1, 0, 2).repeat_interleave(g, 0)[None]
    V = torch.from_numpy(v.astype(np.float64)).permute(1, 0, 2).repeat_interleave(g, 0)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(Q, K, V, attn_mask=mask)[0].permute(1, 0, 2).numpy()
    assert np.abs(out - ref).max() < 1e-12
    # LSE against torch.logsumexp of the masked scaled scores
    s = (Q[0] @ K[0].transpose(1, 2)) / math.sqrt(d)
    s = s.masked_fill(~mask[None], -math.inf)
    assert np.abs(lse - torch.logsumexp(s, -1).T.numpy()).max() < 1e-12
    # the oracle's own "k_prerotated" path on a cache that stores the rotated keys agrees too
    kc2, vc2 = paged(kr.astype(np.float32), v, blocks, 8)
    out2, lse2 = one_request(q, kc2, vc2, blocks, pos, idx, lo, hq, theta, k_prerotated=True)
    assert np.abs(out2 - out).max() < 1e-5 and np.abs(lse2 - lse).max() < 1e-5      # fp32 storage of rotated K


def test_softmax_closed_forms():
    rng = np.random.default_rng(12)
    T, hq, hkv, d = 40, 2, 1, 16
    q, k, v = dense_request(rng, T, hq, hkv, d)
    blocks = [1, 0, 2]
    pos = np.arange(T)
    # one visible key (vis_lo = idx): out = v_idx, lse = q'.k'/sqrt(d) = q.k/sqrt(d) (same position => R cancels)
    kc, vc = paged(k, v, blocks, 3)
    idx = np.arange(T)
    out, lse = one_request(q, kc, vc, blocks, pos, idx, idx, hq, 1e4)
    for h in range(hq):
        assert np.abs(out[:, h] - v[:, 0].astype(np.float64)).max() < 1e-12
        s = (q[:, h].astype(np.float64) * k[:, 0].astype(np.float64)).sum(-1) / math.sqrt(d)
        assert np.abs(lse[:, h] - s).max() < 1e-12
    # Q = 0: out = mean of visible V, lse = ln(count)
    out, lse = one_request(np.zeros_like(q), kc, vc, blocks, pos, idx, np.zeros(T, int), hq, 1e4)
    cum = np.cumsum(v[:, 0].astype(np.float64), 0) / (idx + 1)[:, None]
    assert np.abs(out[:, 0] - cum).max() < 1e-12 and np.abs(lse[:, 1] - np.log(idx + 1)).max() < 1e-12
    # constant V: out = that constant
    vconst = np.broadcast_to(np.linspace(-1, 1, d, dtype=np.float32), (T, hkv, d)).copy()
    kc, vc = paged(k, vconst, blocks, 3)
    out, _ = one_request(q, kc, vc, blocks, pos, idx, np.zeros(T, int), hq, 1e4)
    assert np.abs(out - vconst[0, 0].astype(np.float64)).max() < 1e-12
    # no visible key (vis_lo > idx): out = 0, lse = -inf
    out, lse = one_request(q[:1], kc, vc, blocks, pos, [3], [4], hq, 1e4)
    assert (out == 0).all() and np.isneginf(lse).all()


def test_gqa_head_mapping():
    """Query head h reads KV head h // G."""
    rng = np.random.default_rng(13)
    T, hq, hkv, d = 24, 6, 3, 8
    q, k, v = dense_request(rng, T, hq, hkv, d)
    kc, vc = paged(k, v, [0, 1], 2)
    pos = idx = np.arange(T); lo = np.zeros(T, int)
    out, lse = one_request(q, kc, vc, [0, 1], pos, idx, lo, hq, 1e4)
    for h in range(hq):
        g = h // 2
        kc1, vc1 = paged(k[:, g:g + 1], v[:, g:g + 1], [0, 1], 2)
        o1, l1 = one_request(q[:, h:h + 1], kc1, vc1, [0, 1], pos, idx, lo, 1, 1e4)
        assert np.array_equal(o1[:, 0], out[:, h]) and np.array_equal(l1[:, 0], lse[:, h])


# --------------------------------------------------------------------------- span structure / sharing
def test_span_rows_equal_standalone_span_request_and_suffix_is_full_causal():
    """each document is prefilled as a separate request (positions 0..L-1); in the
    composed prompt its rows must be the same.  Suffix rows equal plain full-causal attention."""
    w = W.single_request_prefill(name="t", hq=4, hkv=2, d=32, theta=1e4, dtype="f32", sigma=1.0,
                                 span_lens=[48, 32, 64], suffix_len=24, num_blocks=20, seed=21)
    kc, vc = O.build_cache(w)
    out, lse = O.run_workload(w, kc, vc)
    off = 0
    for L in (48, 32, 64):
        rows = np.arange(off, off + L)
        blocks = w.block_tables[0, off // B:(off + L) // B]
        o, l = one_request(w.q[rows], kc, vc, blocks, np.arange(L), np.arange(L), np.zeros(L, int), 4, 1e4)
        assert np.abs(o - out[rows]).max() < 1e-12 and np.abs(l - lse[rows]).max() < 1e-12
        off += L
    T = 168
    rows = np.arange(off, T)
    o, l = one_request(w.q[rows], kc, vc, w.block_tables[0], np.arange(T), rows, np.zeros(len(rows), int), 4, 1e4)
    assert np.array_equal(o, out[rows]) and np.array_equal(l, lse[rows])
    # the mask is not vacuous: a span row differs from full-causal attention
    o_full, _ = one_request(w.q[100:101], kc, vc, w.block_tables[0], np.arange(T), [100], [0], 4, 1e4)
    assert np.abs(o_full - out[100:101]).max() > 1e-3


def test_shared_and_duplicated_blocks_equal_isolated_runs():
    """PAPER.md:145 (same physical blocks serve concurrent requests at different offsets) and :232
    (same block twice in one prompt): a batch equals per-request isolated runs exactly."""
    rng = np.random.default_rng(14)
    hq, hkv, d, nb, theta = 4, 2, 16, 12, 5e5
    kc = O.new_cache(nb, hkv, B, d, "f32"); vc = O.new_cache(nb, hkv, B, d, "f32")
    kc[:] = rng.standard_normal(kc.shape).astype(np.float32)
    vc[:] = rng.standard_normal(vc.shape).astype(np.float32)
    tables = [[5, 2, 7, 3], [2, 5, 9, 0], [7, 7, 5, 7]]          # block 5 at offsets 0 / 16 / 32; 7 three times
    kv_lens = np.array([64, 60, 57])
    R = 3
    bt = np.asarray(tables, np.int32)
    q_counts = [10, 7, 12]
    idx = np.concatenate([np.arange(64 - 10, 64), np.arange(60 - 7, 60), np.arange(57 - 12, 57)]).astype(np.int32)
    lo = np.zeros_like(idx); lo[3:6] = 32
    q = rng.standard_normal((idx.size, hq, d)).astype(np.float32)
    cu_q = np.concatenate([[0], np.cumsum(q_counts)])
    cu_kv = np.concatenate([[0], np.cumsum(kv_lens)])
    pos = np.concatenate([np.arange(n) + 100 * r for r, n in enumerate(kv_lens)]).astype(np.int32)
    out, lse = O.prefill_attention(q=q, k_cache=kc, v_cache=vc, block_tables=bt, cu_q_lens=cu_q, kv_lens=kv_lens,
                                   cu_kv_lens=cu_kv, kv_positions=pos, q_seq_idx=idx, q_vis_lo=lo, num_q_heads=hq,
                                   dtype="f32", rope_theta=theta)
    for r in range(R):
        sl = slice(cu_q[r], cu_q[r + 1])
        # isolated: private copy of the request's blocks in a fresh pool, renumbered 0..n-1
        kc1 = kc[bt[r]].copy(); vc1 = vc[bt[r]].copy()
        o, l = one_request(q[sl], kc1, vc1, np.arange(4), pos[cu_kv[r]:cu_kv[r + 1]], idx[sl], lo[sl], hq, theta)
        assert np.array_equal(o, out[sl]) and np.array_equal(l, lse[sl])
    # duplicated block really is read twice: request 2 keys 0..15 == keys 16..31 before rotation
    k0, _ = O.gather_kv(kc, vc, bt[2], 57, 0, "f32")
    assert np.array_equal(k0[:16], k0[16:32]) and np.array_equal(k0[:9], k0[48:57]) and not np.array_equal(k0[:16], k0[32:48])


def test_merge_identity_random_partitions():
    """Split-KV: for any partition of the visible keys, merging (o_s, lse_s) reproduces the whole."""
    rng = np.random.default_rng(15)
    T, hq, hkv, d, theta = 150, 2, 1, 16, 1e4
    q, k, v = dense_request(rng, T, hq, hkv, d)
    blocks = rng.permutation(12)[:10]
    kc, vc = paged(k, v, blocks, 12)
    pos = np.arange(T) + 7
    full_o, full_l = one_request(q[-1:], kc, vc, blocks, pos, [T - 1], [0], hq, theta)
    for trial in range(4):
        cuts = np.sort(rng.choice(np.arange(1, T), size=int(rng.integers(1, 6)), replace=False))
        bounds = [0, *cuts.tolist(), T]
        parts_o, parts_l = [], []
        for a, b in zip(bounds[:-1], bounds[1:]):
            # keys [a, b): the query sits at seq index T-1 (its position), visibility window restricted
            kk, vv = O.gather_kv(kc, vc, blocks, T, 0, "f32")
            kr = O.rope_rotate(kk[a:b], pos[a:b], theta)
            for h in range(hq):
                qr = O.rope_rotate(q[-1, h].astype(np.float64), np.asarray(pos[T - 1]), theta)
                s = kr @ qr / math.sqrt(d)
                m = s.max(); e = np.exp(s - m)
                parts_o.append((e @ vv[a:b]) / e.sum()); parts_l.append(m + math.log(e.sum()))
        po = np.array(parts_o).reshape(len(bounds) - 1, hq, d); pl = np.array(parts_l).reshape(len(bounds) - 1, hq)
        for h in range(hq):
            o, l = O.merge_partials(po[:, h], pl[:, h])
            assert np.abs(o - full_o[0, h]).max() < 1e-12 and abs(l - full_l[0, h]) < 1e-12
    # empty parts (lse = -inf) are ignored
    o, l = O.merge_partials(np.array([[1.0, 2.0], [9.0, 9.0]]), np.array([0.5, -np.inf]))
    assert np.allclose(o, [1.0, 2.0]) and abs(l - 0.5) < 1e-15
    o, l = O.merge_partials(np.array([[1.0, 0.0], [0.0, 1.0]]), np.array([math.log(3.0), math.log(1.0)]))
    assert np.allclose(o, [0.75, 0.25]) and abs(l - math.log(4.0)) < 1e-15


def test_decode_equals_last_row_of_prefill():
    w = W.small_variants()[2]
    kc, vc = O.build_cache(w)
    out, lse = O.run_workload(w, kc, vc, rows=np.array([0, 4]), heads=np.array([0, 5]))
    for r in (0, 4):
        T = int(w.kv_lens[r])
        pos = w.kv_positions[w.cu_kv_lens[r]:w.cu_kv_lens[r + 1]]
        o, l = one_request(w.q[r:r + 1], kc, vc, w.block_tables[r], pos, [T - 1], [0], w.num_q_heads, w.rope_theta,
                           dtype="bf16")
        for h in (0, 5):
            assert np.array_equal(o[0, h], out[r, h]) and l[0, h] == lse[r, h]
    assert np.isnan(out[1]).all()          # rows outside the sample are not computed


# --------------------------------------------------------------------------- rounding mode Q / formats
def test_bf16_rounding_is_rne_and_mode_q_rounds_operands_only():
    x = np.array([1.0, 1.00390625, 1.005859375, 1.01171875, -3.1415926, 1e-3, 123456.0])
    got = O.round_to_dtype(x, "bf16")
    exp = torch.tensor(x, dtype=torch.float64).to(torch.bfloat16).double().numpy()
    assert np.array_equal(got, exp)
    # ties to even: 1 + 2^-8 is a tie between 1 and 1 + 2^-7 -> 1; 1 + 3*2^-8 -> 1 + 2^-6
    assert O.round_to_dtype(np.array([1 + 2 ** -8]), "bf16")[0] == 1.0
    assert O.round_to_dtype(np.array([1 + 3 * 2 ** -8]), "bf16")[0] == 1 + 2 ** -6
    bits = np.arange(0x3F00, 0x4100, dtype=np.uint16)
    assert np.array_equal(O.bf16_bits_to_f64(bits), torch.from_numpy(bits.view(np.int16)).view(torch.bfloat16).double().numpy())
    w = W.small_variants()[0]
    kc, vc = O.build_cache(w)
    rows = np.arange(0, w.num_q_tokens, 37)
    of, lf = O.run_workload(w, kc, vc, mode="F", rows=rows, heads=np.array([1]))
    oq, lq = O.run_workload(w, kc, vc, mode="Q", rows=rows, heads=np.array([1]))
    d = np.abs(lf[rows, 1] - lq[rows, 1])
    assert 1e-7 < d.max() < 2e-2                       # differs (operands were rounded) but only by bf16 rounding


def _bf16(x: float) -> float:
    """One round-to-nearest-even of a Python float to bfloat16 through torch's cast (not the oracle's rounding code)."""
    return float(torch.tensor(x, dtype=torch.float64).to(torch.bfloat16).double())


def brute_force_mode_q(q, k, v, pos, idx, lo, theta, hq, hkv, round_scores=False, round_p=False, round_before_rotation=False):
    """Pure-Python restatement of comparison mode Q ("storing already-rotated keys"): rotate in fp64,
    round every element of q' and k_j ONCE to bf16 with torch's cast, then everything else (dot product, scale, softmax,
    P.V) in fp64 with nothing else rounded.  The three keyword switches are the plausible mistakes the pin must reject."""
    tq, d = len(q), len(q[0][0])
    half = d // 2
    g = hq // hkv

    def rot_round(x, p):
        if round_before_rotation:
            x = [_bf16(e) for e in x]
        y = [0.0] * d
        for i in range(half):
            f = theta ** (-2.0 * i / d)
            c, s = math.cos(p * f), math.sin(p * f)
            y[i] = x[i] * c - x[i + half] * s
            y[i + half] = x[i] * s + x[i + half] * c
        return y if round_before_rotation else [_bf16(e) for e in y]

    out = np.zeros((tq, hq, d))
    lse = np.full((tq, hq), -math.inf)
    for h in range(hq):
        kr = [rot_round(k[j][h // g], pos[j]) for j in range(len(k))]
        for t in range(tq):
            qr = rot_round(q[t][h], pos[idx[t]])
            vis = [j for j in range(len(k)) if lo[t] <= j <= idx[t]]
            if not vis:
                continue
            sc = [sum(a * b for a, b in zip(qr, kr[j])) / math.sqrt(d) for j in vis]
            if round_scores:
                sc = [_bf16(s) for s in sc]
            m = max(sc)
            z = sum(math.exp(s - m) for s in sc)
            lse[t, h] = m + math.log(z)
            for j, s in zip(vis, sc):
                p = math.exp(s - m) / z
                if round_p:
                    p = _bf16(p)
                for e in range(d):
                    out[t, h, e] += p * v[j][h // g][e]
    return out, lse


def test_mode_q_pinned_by_brute_force_with_torch_bf16_rounding():
    """Mode Q is the comparison the tensor-core LSE gate rests on (R1), so it gets its own pin: a brute-force
    restatement that rounds exactly q' and k_j (after rotation, before the dot product) must agree to 1e-12, and the
    variants that round something else - the scores, the probabilities, or the operands BEFORE the rotation - must not."""
    rng = np.random.default_rng(21)
    T, hq, hkv, d, theta = 37, 4, 2, 16, 1e4
    q, k, v = dense_request(rng, T, hq, hkv, d, dtype="bf16")
    blocks = [5, 1, 7]
    kc, vc = paged(k, v, blocks, 9, dtype="bf16")
    pos = (np.arange(T) * 3 + 11).astype(np.int64)               # positions are not the index
    idx = np.arange(T)
    lo = np.where(idx < 16, 0, np.where(idx < 32, 16, 0))        # one span-local stretch, suffix sees all
    oq, lq = one_request(q, kc, vc, blocks, pos, idx, lo, hq, theta, dtype="bf16", mode="Q")
    qf, kf, vf = (O.bf16_bits_to_f64(a) for a in (q, k, v))
    bo, bl = brute_force_mode_q(qf.tolist(), kf.tolist(), vf.tolist(), pos.tolist(), idx.tolist(), lo.tolist(), theta, hq, hkv)
    assert np.abs(oq - bo).max() < 1e-12 and np.abs(lq - bl).max() < 1e-12
    # the pin discriminates: each plausible mis-reading of "mode Q" is far outside 1e-12
    for wrong in (dict(round_scores=True), dict(round_p=True), dict(round_before_rotation=True)):
        wo, wl = brute_force_mode_q(qf.tolist(), kf.tolist(), vf.tolist(), pos.tolist(), idx.tolist(), lo.tolist(), theta,
                                    hq, hkv, **wrong)
        assert max(np.abs(oq - wo).max(), np.abs(lq - wl).max()) > 1e-6, wrong
    # V is never rounded by mode Q: with identical scores (Q = 0 -> every score is 0 in both modes) outputs agree exactly
    q0 = np.zeros_like(q)
    of0, lf0 = one_request(q0, kc, vc, blocks, pos, idx, lo, hq, theta, dtype="bf16", mode="F")
    oq0, lq0 = one_request(q0, kc, vc, blocks, pos, idx, lo, hq, theta, dtype="bf16", mode="Q")
    assert np.array_equal(of0, oq0) and np.array_equal(lf0, lq0)
    # f32 I/O: mode Q rounds the rotated operands to float32
    q32, k32, v32 = dense_request(rng, 20, 2, 1, 8)
    kc32, vc32 = paged(k32, v32, [3, 0], 4)
    p32 = np.arange(20)
    o32, l32 = one_request(q32, kc32, vc32, [3, 0], p32, p32, np.zeros(20, int), 2, 1e4, dtype="f32", mode="Q")
    kr = O.rope_rotate(k32[:, 0].astype(np.float64), p32, 1e4).astype(np.float32).astype(np.float64)
    for t in (0, 7, 19):
        qr = O.rope_rotate(q32[t, 1].astype(np.float64), np.asarray(t), 1e4).astype(np.float32).astype(np.float64)
        s = kr[:t + 1] @ qr / math.sqrt(8)
        assert abs(l32[t, 1] - (s.max() + math.log(np.exp(s - s.max()).sum()))) < 1e-12


# --------------------------------------------------------------------------- generator sanity (integer structure)
def test_workload_structure_matches_baseline_configs():
    w1 = W.config1()
    assert (w1.num_q_heads, w1.num_kv_heads, w1.head_dim, w1.dtype, w1.num_blocks) == (4, 1, 64, "f32", 32)
    assert w1.num_q_tokens == 112 and w1.visible_pairs() == 3256
    assert len(set(w1.block_tables[0, :7].tolist())) == 7
    assert (w1.q_vis_lo == np.repeat([0, 32, 64, 0], [32, 32, 32, 16])).all()
    assert (w1.kv_positions == np.arange(112)).all()
    w2 = W.config2()
    assert w2.num_q_tokens == 2112 and w2.visible_pairs() == 396320 and w2.attention_flops() == 4 * 128 * 32 * 396320
    s3 = W.small_variants()[1]
    # shared blocks recur across requests at different logical offsets
    seen = {}
    multi = 0
    for r in range(s3.num_reqs):
        nb = -(-int(s3.kv_lens[r]) // B)
        for i, b in enumerate(s3.block_tables[r, :nb].tolist()):
            if b in seen and seen[b] != i:
                multi += 1
            seen.setdefault(b, i)
    assert multi > 0
    for w in W.small_variants():
        assert (w.q_vis_lo <= w.q_seq_idx).all() and (w.q_vis_lo % B == 0).all()
        for b in w.resident + w.new:
            assert b.slots.max() < w.num_blocks * B
        allslots = np.concatenate([b.slots for b in w.resident + w.new])
        assert np.unique(allslots).size == allslots.size       # no duplicate slot writes
