"""Out-of-bounds writes (compute-sanitizer is not available on the GPU pool): every output buffer sits between
sentinel-filled guard bands inside one allocation; after the call the guards must be intact and the read-only
inputs bit-identical."""
import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import synth_inputs as si
from gpu_util import oracle_apply

pytestmark = pytest.mark.gpu
GUARD = 4096          # elements on each side
SENT = -7.5e300


def _banded(t):
    """Copy tensor t into the middle of a guard-banded allocation; returns (whole, view)."""
    import torch

    whole = torch.full((t.numel() + 2 * GUARD,), SENT, dtype=t.dtype, device="cuda")
    view = whole[GUARD:GUARD + t.numel()].view(t.shape)
    view.copy_(t)
    return whole, view


def _guards_ok(whole, n):
    import torch

    s = torch.full((1,), SENT, dtype=whole.dtype, device="cuda")
    return bool((whole[:GUARD] == s).all().item()) and bool((whole[GUARD + n:] == s).all().item())


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw,nev,variant", [(3 * 32 + 5, 32, 33, 0), (9 * 64 + 3, 64, 5, 0), (17 * 32 + 1, 32, 9, 0),
                                              (140, 128, 9, 0), (2 * 64 + 9, 64, 1500, 0), (8 * 64, 64, 2500, 3),
                                              (200, 64, 50, 2)])
def test_back_transform_stays_inside_its_buffers(N, nbw, nev, variant, cplx):
    import torch

    from paper_2002_10991_b200 import binding

    ab = si.band_matrix(N, nbw, 3, cplx)
    hv, ht, _, _ = orc.bulge_chase(ab, nbw)
    rng = np.random.default_rng(1)
    x = rng.standard_normal((N, nev)) + (1j * rng.standard_normal((N, nev)) if cplx else 0)
    x = np.asfortranarray(x)
    want = oracle_apply(N, nbw, hv, ht, x)
    wq, q_cm = _banded(torch.from_numpy(np.ascontiguousarray(x.T)).cuda())      # (nev, N): column-major q
    wv, dv = _banded(torch.from_numpy(hv).cuda())
    wt, dt = _banded(torch.from_numpy(ht).cuda())
    old = binding.set_variant(variant)
    try:
        binding.trans_ev_tridi_to_band(N, nbw, dv, dt, q_cm.t())
        torch.cuda.synchronize()
    finally:
        binding.set_variant(old)
    assert np.abs(q_cm.t().cpu().numpy() - want).max() <= 1e-11 * np.abs(x).max()
    assert _guards_ok(wq, N * nev) and _guards_ok(wv, hv.size) and _guards_ok(wt, ht.size)
    assert np.array_equal(dv.cpu().numpy(), hv) and np.array_equal(dt.cpu().numpy(), ht)   # inputs untouched


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw", [(2, 32), (70, 32), (300, 64), (257, 128)])
def test_bulge_chase_stays_inside_its_buffers(N, nbw, cplx):
    import ctypes

    import torch

    from paper_2002_10991_b200 import binding

    ab = si.band_matrix(N, nbw, 9, cplx)
    ab_o = ab.copy(order="F")
    hv_o, ht_o, d_o, e_o = orc.bulge_chase(ab_o, nbw)
    dt_ = torch.complex128 if cplx else torch.float64
    G = orc.hh_count(N, nbw)
    wab, dab = _banded(torch.from_numpy(np.ascontiguousarray(ab.T)).cuda())
    wv, dv = _banded(torch.zeros((G, nbw), dtype=dt_, device="cuda"))
    wt, dtau = _banded(torch.zeros((G,), dtype=dt_, device="cuda"))
    wd, dd = _banded(torch.zeros((N,), dtype=torch.float64, device="cuda"))
    we, de = _banded(torch.zeros((max(N - 1, 1),), dtype=torch.float64, device="cuda"))
    fn = binding.lib().elpa2_bulge_chase_z if cplx else binding.lib().elpa2_bulge_chase_d
    rc = fn(N, nbw, dab.data_ptr(), dv.data_ptr(), dtau.data_ptr(), dd.data_ptr(), de.data_ptr(),
            torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert rc == 0
    assert np.array_equal(dv.cpu().numpy(), hv_o) and np.array_equal(dtau.cpu().numpy(), ht_o)
    assert np.array_equal(dd.cpu().numpy(), d_o) and np.array_equal(de.cpu().numpy()[:N - 1], e_o)
    assert _guards_ok(wab, N * (2 * nbw + 1)) and _guards_ok(wv, G * nbw) and _guards_ok(wt, G)
    assert _guards_ok(wd, N) and _guards_ok(we, max(N - 1, 1))


def test_real_q_that_is_only_8_byte_aligned():
    """q starting one double past a 16-byte boundary: the kernel must take its 8-byte access path."""
    import torch

    from paper_2002_10991_b200 import binding

    N, nbw, nev = 2 * 64 + 10, 64, 77
    ab = si.band_matrix(N, nbw, 4, False)
    hv, ht, _, _ = orc.bulge_chase(ab, nbw)
    x = np.asfortranarray(np.random.default_rng(2).standard_normal((N, nev)))
    want = oracle_apply(N, nbw, hv, ht, x)
    whole = torch.full((N * nev + 2 * GUARD + 1,), SENT, dtype=torch.float64, device="cuda")
    q_cm = whole[GUARD + 1:GUARD + 1 + N * nev].view(nev, N)
    assert q_cm.data_ptr() % 16 == 8
    q_cm.copy_(torch.from_numpy(np.ascontiguousarray(x.T)).cuda())
    binding.trans_ev_tridi_to_band(N, nbw, torch.from_numpy(hv).cuda(), torch.from_numpy(ht).cuda(), q_cm.t())
    torch.cuda.synchronize()
    assert np.abs(q_cm.t().cpu().numpy() - want).max() <= 1e-11 * np.abs(x).max()
    s_ = torch.full((1,), SENT, dtype=torch.float64, device="cuda")
    assert bool((whole[:GUARD + 1] == s_).all().item()) and bool((whole[GUARD + 1 + N * nev:] == s_).all().item())
