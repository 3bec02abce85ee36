"""minipic_decode_attention_static: decode attention with the split-KV partials in the library's file-scope static device
array (include/minipic.h) - for callers that may not allocate.  Collected LAST on purpose (the suite runs with pytest -x).

The new entry point runs the same kernels as minipic_decode_attention, so its output is compared with the existing path's
within the tolerance of tests/test_gpu_parity.py (and is in fact expected to be identical), on two calls in a row: the array
keeps the first call's contents when the second one runs."""
import numpy as np
import pytest
import torch

from paper_2606_13126_b200 import binding as mp
from paper_2606_13126_b200 import workloads as W
from paper_2606_13126_b200.runner import DeviceWorkload

pytestmark = pytest.mark.gpu

OUT_MAX, OUT_MEAN, LSE_TOL = 2e-2, 2e-3, 1e-3      # as in tests/test_gpu_parity.py


def _call_static(dw, out, lse, num_seqs=None, max_kv_len=None):
    w = dw.w
    mp.minipic_decode_attention_static(dw.cfg, dw.q, dw.k_cache, dw.v_cache, dw.block_tables, int(dw.block_tables.shape[1]),
                                       dw.kv_lens, dw.cu_kv_lens, dw.kv_positions, dw.q_vis_lo,
                                       w.num_reqs if num_seqs is None else num_seqs,
                                       w.max_kv_len if max_kv_len is None else max_kv_len, out, lse)


def _f64(t, dtype):
    return (t.view(torch.bfloat16) if dtype == "bf16" else t).double().cpu().numpy()


def test_static_scratch_decode_matches_workspace_path_twice_in_a_row():
    assert mp.minipic_static_scratch_bytes() == 16 << 20
    # two different problems back to back: the second call finds the first one's partials in the array
    first = W.small_variants()[2]                                                       # s4_decode: 9 sequences, 300-1500 keys
    second = W.shared_pool_decode(name="noalloc2", seed=31, hq=16, hkv=4, num_seqs=5, ctx_min=700, ctx_max=2600,
                                  span_len=128, pool_spans=24)
    for rep, w in enumerate((first, second, first)):
        dw = DeviceWorkload(w)
        dw.step(); torch.cuda.synchronize()                                             # existing path (caller workspace)
        want_o, want_l = _f64(dw.out, w.dtype), dw.lse.double().cpu().numpy()
        assert mp.minipic_decode_workspace_bytes(dw.cfg, w.num_reqs, w.max_kv_len) <= mp.minipic_static_scratch_bytes()
        out, lse = torch.full_like(dw.out, 0x7FC1 if w.dtype == "bf16" else float("nan")), torch.full_like(dw.lse, float("nan"))
        launches = mp.minipic_launch_count()
        for call in range(2):                                                           # two calls in a row, same array
            out.fill_(0x7FC1 if w.dtype == "bf16" else float("nan")); lse.fill_(float("nan"))
            _call_static(dw, out, lse)
            torch.cuda.synchronize()
            got_o, got_l = _f64(out, w.dtype), lse.double().cpu().numpy()
            assert np.isfinite(got_o).all() and np.isfinite(got_l).all(), (rep, call)
            do, dl = np.abs(got_o - want_o), np.abs(got_l - want_l)
            assert do.max() <= OUT_MAX and do.mean() <= OUT_MEAN and dl.max() <= LSE_TOL, (rep, call, float(do.max()), float(dl.max()))
            assert np.array_equal(got_o, want_o) and np.array_equal(got_l, want_l)      # same kernels, same split plan
        assert mp.minipic_launch_count() - launches >= 4                               # the library's own kernels ran
        assert mp.minipic_last_variant() == "decode_mma"


def test_static_scratch_rejects_problems_beyond_its_size():
    w = W.small_variants()[2]
    dw = DeviceWorkload(w)
    dw.step(); torch.cuda.synchronize()
    before = dw.out.clone()
    # 2048 sequences x 8 K keys with these 8 heads need ~ 34 MB of partials: rejected before anything is launched
    assert mp.minipic_decode_workspace_bytes(dw.cfg, 2048, 8192) > mp.minipic_static_scratch_bytes()
    launches = mp.minipic_launch_count()
    with pytest.raises(mp.MinipicError) as ei:
        _call_static(dw, dw.out, dw.lse, num_seqs=2048, max_kv_len=8192)
    assert ei.value.status == mp.MINIPIC_ERR_WORKSPACE_TOO_SMALL
    assert b"static scratch" in mp.lib().minipic_last_cuda_error()
    torch.cuda.synchronize()
    assert mp.minipic_launch_count() == launches and torch.equal(before, dw.out)
    # and the entry point still works afterwards
    _call_static(dw, dw.out, dw.lse); torch.cuda.synchronize()
    assert torch.equal(before, dw.out)
