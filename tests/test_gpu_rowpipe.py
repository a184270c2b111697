"""SURVEY.md 8(f) NEXT-3 on the GPU: the row-block call ``elpa2_trans_ev_tridi_to_band_rows_{d,z}`` and the
row pipeline built on it (paper_2002_10991_b200/rowpipe.py), with R ranks emulated on ONE device in a
dependency-respecting order (device-to-device copies in place of the NCCL sends: kernels of different
ranks never wait on one another, B200_PROFILING.md).  The sub-range launches run the same kernels over a
part of their block sequence, so the assembled result must equal the single call's BIT FOR BIT (same plan:
P = 1) -- and that one is checked against the oracle."""
import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import rowpipe, synth_inputs as si

pytestmark = pytest.mark.gpu


def _setup(N, nbw, nev, cplx):
    import torch

    from paper_2002_10991_b200 import binding

    lengths = binding.hh_lengths(N, nbw)
    hh_v, hh_tau = si.synthetic_reflectors(lengths, nbw, 91, cplx, "cuda")
    x = si.gaussian_block(N, nev, 92, cplx, "cuda")
    return hh_v, hh_tau, x


def _single_call(N, nbw, hh_v, hh_tau, x):
    from paper_2002_10991_b200 import binding

    q = x.clone()
    old = binding.set_chain_parallel(1)
    try:
        binding.trans_ev_tridi_to_band(N, nbw, hh_v, hh_tau, q)
    finally:
        binding.set_chain_parallel(old)
    return q


def _pipeline(N, nbw, hh_v, hh_tau, x, R):
    import torch

    bounds = rowpipe.partition_rows(N, R, nbw)
    bufs = []
    for r in range(R):
        n = rowpipe.local_rows(N, nbw, bounds, r)
        back = torch.full((x.shape[1], n + 2), float("nan"), dtype=x.dtype, device="cuda")   # ldq = n + 2; halo = NaN
        buf = back.t()[:n, :]
        buf[: bounds[r + 1] - bounds[r]] = x[bounds[r]:bounds[r + 1]]
        bufs.append(buf)
    rowpipe.run_emulated(N, nbw, bounds, bufs, rowpipe.device_apply(N, nbw, hh_v, hh_tau))
    torch.cuda.synchronize()
    return torch.cat([bufs[r][: bounds[r + 1] - bounds[r]] for r in range(R)], dim=0), bounds


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw,nev,R", [(300, 32, 40, 2), (517, 64, 100, 3), (1000, 32, 333, 4), (1029, 128, 24, 2),
                                         (96, 32, 9, 3), (2000, 64, 2500, 4), (777, 96, 50, 2)])
def test_emulated_row_pipeline_is_bit_identical_to_the_single_call(N, nbw, nev, R, cplx):
    import torch

    hh_v, hh_tau, x = _setup(N, nbw, nev, cplx)
    ref = _single_call(N, nbw, hh_v, hh_tau, x)
    got, bounds = _pipeline(N, nbw, hh_v, hh_tau, x, R)
    assert torch.equal(got, ref), (bounds, float((got - ref).abs().max()))
    # and the single call is the oracle's result (sampled columns)
    cols = np.unique(np.array([0, nev // 2, nev - 1]))
    xs = np.asfortranarray(x[:, torch.from_numpy(cols).cuda()].cpu().numpy())
    want = np.array(xs, order="F", copy=True)
    orc.back_transform(N, nbw, hh_v.cpu().numpy(), hh_tau.cpu().numpy(), want)
    assert np.abs(ref[:, torch.from_numpy(cols).cuda()].cpu().numpy() - want).max() <= 1e-11 * np.abs(xs).max()


@pytest.mark.parametrize("cplx", [False, True])
def test_rows_call_over_the_whole_matrix_and_chain_ranges(cplx):
    """One 'rank' that owns everything: all chains in one call, and the same split into chain ranges."""
    import torch

    from paper_2002_10991_b200 import binding

    N, nbw, nev = 700, 64, 77
    hh_v, hh_tau, x = _setup(N, nbw, nev, cplx)
    ref = _single_call(N, nbw, hh_v, hh_tau, x)
    K0 = (N - 2 + nbw) // nbw
    q = x.clone()
    binding.trans_ev_tridi_to_band_rows(N, nbw, hh_v, hh_tau, q, 0, N, 0, K0)
    assert torch.equal(q, ref)
    assert binding.last_launch_count() == 2
    q = x.clone()
    for kb, ke in ((0, 1), (1, 4), (4, 4), (4, K0 + 5)):
        binding.trans_ev_tridi_to_band_rows(N, nbw, hh_v, hh_tau, q, 0, N, kb, ke)
    assert torch.equal(q, ref)


def test_rows_call_argument_validation():
    import torch

    from paper_2002_10991_b200 import binding

    N, nbw = 300, 32
    hh_v, hh_tau, x = _setup(N, nbw, 8, False)
    K0 = (N - 2 + nbw) // nbw
    for row0, nown, nloc, kb, ke, code in ((4, 64, 96, 0, 1, -8), (0, 60, 92, 0, 1, -9), (0, 64, 80, 0, 1, -10),
                                           (0, 64, 96, 2, 1, -11), (296, 8, 4, 0, 1, -9)):
        buf = x[row0:row0 + nloc] if row0 + nloc <= N else x[row0:]
        with pytest.raises(binding.Elpa2BtError) as ei:
            # the binding derives nloc from the tensor; pass a view with that many rows
            binding.trans_ev_tridi_to_band_rows(N, nbw, hh_v, hh_tau, buf, row0, nown, kb, ke)
        assert ei.value.rc == code, (row0, nown, nloc, code, ei.value.rc)
