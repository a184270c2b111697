"""The allocation-free entry point ``elpa2_trans_ev_band_to_full_noalloc_d`` (include/elpa2_bt.h): Eq. 6e with its
scratch in a static device array inside the library, for callers that cannot call cudaMalloc.  Its output is
compared with the existing path's (``elpa2_trans_ev_band_to_full_d``, scratch from the stream-ordered pool) on
two calls in a row -- different shapes, so the array's stale contents from the first call are in the way of
the second -- and with the oracle.  Both paths run the same kernels, so the results are bit-identical; the
comparison is written with the tolerance of tests/test_gpu_b2f.py.  Collected last on purpose (file name):
the suite runs with ``pytest -x``.
"""
import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import synth_inputs as si

pytestmark = pytest.mark.gpu

TOL = 1e-11


def _problem(N, nbw, nev, seed):
    hv, tau = si.synthetic_full_reflectors(N, nbw, seed, False, "cuda")
    q = si.gaussian_block(N, nev, seed + 1, False, "cuda")
    return hv, tau, q


def test_noalloc_matches_the_pool_path_on_two_calls_in_a_row():
    import torch

    from paper_2002_10991_b200 import binding

    assert binding.noalloc_scratch_bytes() == 16 << 20
    results = []
    for N, nbw, nev, seed in ((1500, 64, 300, 71), (777, 32, 1201, 72), (1500, 64, 300, 71)):
        hv, tau, q = _problem(N, nbw, nev, seed)
        ref = q.clone()
        binding.trans_ev_band_to_full(N, nbw, hv, tau, ref)
        got = q.clone()
        binding.trans_ev_band_to_full_noalloc(N, nbw, hv, tau, got)
        torch.cuda.synchronize()
        assert binding.last_launch_count() == 2
        xmax = float(q.abs().max())
        assert float((got - ref).abs().max()) <= TOL * xmax
        assert torch.equal(got, ref)                     # same kernels, same scratch contents: same bits
        # and against the oracle on a few columns
        cols = torch.tensor([0, nev // 2, nev - 1], device="cuda")
        want = np.asfortranarray(q[:, cols].cpu().numpy())
        orc.band_to_full_back(N, nbw, np.asfortranarray(hv.cpu().numpy()), tau.cpu().numpy(), want)
        assert np.abs(got[:, cols].cpu().numpy() - want).max() <= TOL * xmax
        results.append(got)
    assert torch.equal(results[0], results[2])           # the first problem again, after another one used the array


def test_noalloc_rejects_problems_beyond_the_static_scratch_and_handles_no_work():
    import torch

    from paper_2002_10991_b200 import binding

    # 32 KB per block of 64 reflectors, 16 MiB: N - nbw - 1 <= 32768.  The size check comes before any pointer
    # is touched, so tiny stand-in tensors are enough (nothing is launched).
    L = binding.lib()
    x = torch.zeros(4, dtype=torch.float64, device="cuda")
    N = 32768 + 64 + 1 + 1
    rc = L.elpa2_trans_ev_band_to_full_noalloc_d(N, 64, 8, x.data_ptr(), N, x.data_ptr(), x.data_ptr(), N, 0)
    assert rc == -20
    with pytest.raises(binding.Elpa2BtError, match="static no-alloc array"):
        raise binding.Elpa2BtError(rc)
    N = 32768 + 64 + 1                                    # the largest problem that fits passes the size check
    rc = L.elpa2_trans_ev_band_to_full_noalloc_d(N, 64, 8, 0, N, x.data_ptr(), x.data_ptr(), N, 0)
    assert rc == -4                                       # ... and fails on the NULL hv instead
    # no work: success, nothing launched
    assert L.elpa2_trans_ev_band_to_full_noalloc_d(40, 64, 8, 0, 40, 0, 0, 40, 0) == 0
    assert binding.last_launch_count() == 0
