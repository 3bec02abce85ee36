"""f3: the host-side C++ block hasher / pool (csrc/hasher.cu, Eq. 1) against the oracle (hashlib).  CPU only:
the library loads without a GPU and these entry points never touch one."""
import hashlib

import numpy as np
import pytest

from oracle import minipic_next as N
from paper_2606_13126_b200 import binding as mp

SSEP, PDEP, B = 128001, 128002, 16


def _rag_stream(rng, n_docs=6):
    sys_p = rng.integers(0, 100000, 2 * B)
    docs = [np.concatenate([[SSEP], rng.integers(0, 100000, int(rng.integers(2, 9)) * B - 1)]) for _ in range(n_docs)]
    task = np.concatenate([[PDEP], rng.integers(0, 100000, int(rng.integers(20, 90)))])
    return sys_p, docs, task


def test_sha256_known_answer_through_the_chain():
    # an ordinary first block: h = SHA-256(h0 || tokens), h0 = SHA-256(seed bytes): both written out with hashlib here
    toks = np.arange(16, dtype=np.int32)
    got = mp.minipic_block_hashes(toks, 16, SSEP, PDEP, seed=7)
    h0 = hashlib.sha256((7).to_bytes(8, "little")).digest()
    assert got.shape == (1, 32) and got[0].tobytes() == hashlib.sha256(h0 + toks.astype("<i4").tobytes()).digest()
    assert mp.minipic_block_hashes(toks[:15], 16, SSEP, PDEP).shape == (0, 32)      # no full block, no hash


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_block_hashes_match_oracle(seed):
    rng = np.random.default_rng(seed)
    sys_p, docs, task = _rag_stream(rng)
    prompt = np.concatenate([sys_p] + docs + [task])
    prompt[3 * B + 5] = SSEP                                  # a marker in the middle of a block does nothing
    got = mp.minipic_block_hashes(prompt, B, SSEP, PDEP, seed=seed)
    want = N.block_hashes(prompt, B, SSEP, PDEP, seed=seed)
    assert len(want) == got.shape[0] and all(got[i].tobytes() == want[i] for i in range(len(want)))
    # negative token ids (two's complement little endian) and a long prompt that crosses many SHA blocks
    odd = rng.integers(-2 ** 31, 2 ** 31 - 1, 40 * B).astype(np.int64); odd[7 * B] = PDEP; odd[20 * B] = SSEP
    got = mp.minipic_block_hashes(odd.astype(np.int32), B, SSEP, PDEP, seed=seed)
    want = N.block_hashes(odd.astype(np.int32), B, SSEP, PDEP, seed=seed)
    assert all(got[i].tobytes() == want[i] for i in range(len(want)))


def test_pool_matches_oracle_on_the_block_attention_procedure():
    """documents prefilled as separate requests, then final prompts composed in other orders."""
    rng = np.random.default_rng(5)
    sys_p, docs, _ = _rag_stream(rng, n_docs=8)
    pool, ref = mp.Pool(512, B, SSEP, PDEP, seed=3), N.Pool(512, B, SSEP, PDEP, seed=3)
    streams = [sys_p] + docs
    for r in range(6):
        pick = rng.permutation(len(docs))[:4]
        task = np.concatenate([[PDEP], rng.integers(0, 100000, int(rng.integers(20, 90)))])
        streams.append(np.concatenate([sys_p] + [docs[i] for i in pick] + [task]))
    streams.append(streams[-1].copy())                        # the same final prompt again: the PDEP block hits now
    for s in streams:
        t, hit, slots, lo, n_new = pool.admit(s)
        t2, hit2, slots2, lo2 = ref.admit(s)
        assert np.array_equal(t, t2) and np.array_equal(hit, hit2) and np.array_equal(slots, slots2) and np.array_equal(lo, lo2)
        assert n_new == int((slots >= 0).sum())
    st = pool.stats()
    assert st["hits"] == ref.hits and st["misses"] == ref.misses and st["evictions"] == 0


def test_pool_release_and_lru_eviction():
    rng = np.random.default_rng(9)
    pool = mp.Pool(8, B, SSEP, PDEP)
    a = np.concatenate([[SSEP], rng.integers(0, 1000, 4 * B - 1)])
    b = np.concatenate([[SSEP], rng.integers(0, 1000, 4 * B - 1)])
    c = np.concatenate([[SSEP], rng.integers(0, 1000, 4 * B - 1)])
    ta = pool.admit(a)[0]; tb = pool.admit(b)[0]
    assert sorted(ta.tolist() + tb.tolist()) == list(range(8))
    with pytest.raises(mp.MinipicError):
        pool.admit(c)                                         # every block is referenced: nothing to evict
    assert pool.admit(a)[1].all()                             # a failed admit leaves the pool usable; a still hits
    pool.release(ta); pool.release(ta)                        # both references of a
    assert pool.admit(a)[1].all()                             # unreferenced but still cached: hits
    pool.release(ta); pool.release(tb)
    tc, hit_c = pool.admit(c)[:2]                             # evicts the least recently released blocks: a's
    assert not hit_c.any() and sorted(tc.tolist()) == sorted(ta.tolist()) and pool.stats()["evictions"] == 4
    assert pool.admit(b)[1].all()                             # b was released too but not evicted: still hits
    pool.release(tc)
    ta2, hit_a2 = pool.admit(a)[:2]                           # a's digests were forgotten at eviction: misses, evicts c's
    assert not hit_a2.any() and sorted(ta2.tolist()) == sorted(tc.tolist()) and pool.stats()["evictions"] == 8
    pool.close()


def test_isps_replay_block_attention_vs_prefix_caching():
    """with SSEP / PDEP only the system prompt, each distinct document ONCE and the task suffixes are
    prefilled; without the markers (ordinary chained hashing) only the shared system prefix ever hits."""
    from paper_2606_13126_b200 import isps
    rng = np.random.default_rng(11)
    PAD = 128000
    system = rng.integers(0, 100000, 40)
    corpus = [rng.integers(0, 100000, int(rng.integers(100, 400))) for _ in range(12)]
    batches = [[(system, [corpus[i] for i in rng.permutation(12)[:5]], rng.integers(0, 100000, 30)) for _ in range(4)]
               for _ in range(3)]
    ordered = isps.isps_order(batches, B, SSEP, PDEP, PAD)
    assert [k for k, _ in ordered[:3]] == ["span"] * 3 and sum(k == "final" for k, _ in ordered) == 12
    # spans come before the final prompts of their own mini-batch, and no span is prefilled twice
    spans = [t.tobytes() for k, t in ordered if k == "span"]
    assert len(spans) == len(set(spans))
    pool = mp.Pool(4096, B, SSEP, PDEP)
    st = isps.replay(pool, ordered)
    span_tokens = sum(len(t) for k, t in ordered if k == "span")
    task_tokens = 12 * 31                                    # PDEP + 30 task tokens per final prompt: always recomputed
    assert st["prefilled_tokens"] == span_tokens + task_tokens and st["final_prompt_prefilled"] == task_tokens
    assert st["evictions"] == 0
    # control: the same final prompts with the markers replaced by ordinary tokens -> only the system prefix hits
    plain = [("final", np.where((t == SSEP) | (t == PDEP), PAD, t).astype(np.int32)) for k, t in ordered if k == "final"]
    st0 = isps.replay(mp.Pool(4096, B, SSEP, PDEP), plain)
    expect = 0                                               # chained hashing = longest common block prefix with an earlier prompt
    for i, (_, t) in enumerate(plain):
        common = 0
        for _, u in plain[:i]:
            m = min(len(t), len(u)) // B * B
            eq = (t[:m].reshape(-1, B) == u[:m].reshape(-1, B)).all(axis=1)
            common = max(common, int(np.argmin(np.append(eq, False))) * B)
        expect += len(t) - common
    assert st0["prefilled_tokens"] == expect and expect > 5 * st["final_prompt_prefilled"]
    # EPIC / LegoLink: the link tokens of every document are recomputed as well
    ordered_e = isps.isps_order(batches, B, SSEP, PDEP, PAD, link_tokens=16)
    st_e = isps.replay(mp.Pool(4096, B, SSEP, PDEP), ordered_e)
    # (a link block right after the system prompt chains on the same context in every prompt that starts with that document,
    # so it can legitimately hit; every later one depends on a different preceding context)
    assert task_tokens + 12 * 4 * 16 <= st_e["final_prompt_prefilled"] <= task_tokens + 12 * 5 * 16
