"""FP32 real / complex back-transformation (``elpa2_trans_ev_tridi_to_band_{s,c}``)
against the FP32 oracle (``orc_back_transform_{s,c}``: Eq. 8 with every product and sum in float, reading
R16), element by element on the same rounded inputs.

Tolerance: both sides apply the same unitary operators in float and differ
in the summation order of each dot product (oracle: left to right; kernel: four partial sums, FMA), so
each is within about u sqrt(N) ||X||_max of the exact result, u = 2^-24; the bar is 8 u sqrt(N) ||X||_max,
the same bound that pins the FP32 oracle to the FP64 one.  The FP64 oracle on the same inputs is checked
too: the kernel must not be further from it than that bound either.
"""
import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import synth_inputs as si

pytestmark = pytest.mark.gpu

WIDTHS = [(False, 32), (False, 64), (False, 96), (False, 128), (True, 32), (True, 64)]


def tol32(N):
    return 8.0 * 2.0 ** -24 * np.sqrt(max(N, 1))


def _inputs(N, nbw, nev, cplx, seed=0):
    f32 = np.complex64 if cplx else np.float32
    ab = si.band_matrix(N, nbw, 8000 + N + nbw + seed, cplx)
    hh_v, hh_tau, _, _ = orc.bulge_chase(ab, nbw)
    rng = np.random.default_rng(31 + N + seed)
    x = rng.standard_normal((N, nev)) + (1j * rng.standard_normal((N, nev)) if cplx else 0)
    return hh_v.astype(f32), hh_tau.astype(f32), np.asfortranarray(x.astype(f32))


def _run(N, nbw, v32, t32, x32, ldq=None, offset=0):
    import torch

    from paper_2002_10991_b200 import binding

    nev = x32.shape[1]
    ldq = ldq or max(N, 1)
    dt = torch.complex64 if np.iscomplexobj(x32) else torch.float32
    flat = torch.full((nev * ldq + offset,), 7.25, dtype=dt, device="cuda")
    back = flat[offset:].view(nev, ldq)
    q = back.t()[:N, :]
    if N and nev:
        q.copy_(torch.from_numpy(np.ascontiguousarray(x32)).cuda())
    dv = torch.from_numpy(np.ascontiguousarray(v32)).cuda()
    dtau = torch.from_numpy(np.ascontiguousarray(t32)).cuda()
    if dv.numel() == 0:
        dv = torch.zeros((1, nbw), dtype=dt, device="cuda")
        dtau = torch.zeros((1,), dtype=dt, device="cuda")
    binding.trans_ev_tridi_to_band(N, nbw, dv, dtau, q)
    torch.cuda.synchronize()
    assert binding.last_launch_count() == (1 if N > 1 and nev > 0 else 0)
    return q.cpu().numpy(), back.t()[N:, :].cpu().numpy()


def _check(N, nbw, nev, cplx, ldq=None, offset=0):
    v32, t32, x32 = _inputs(N, nbw, nev, cplx)
    want = np.array(x32, order="F", copy=True)
    if N >= 2 and nev > 0:
        orc.back_transform(N, nbw, v32, t32, want)
    got, pad = _run(N, nbw, v32, t32, x32, ldq=ldq, offset=offset)
    assert got.dtype == x32.dtype
    xmax = max(float(np.abs(x32).max(initial=0.0)), 1e-30)
    assert np.abs(got - want).max(initial=0.0) <= tol32(N) * xmax, (N, nbw, nev, cplx)
    if N >= 2 and nev > 0:
        f64 = np.complex128 if cplx else np.float64
        w64 = np.asfortranarray(x32.astype(f64))
        orc.back_transform(N, nbw, v32.astype(f64), t32.astype(f64), w64)
        assert np.abs(got - w64).max() <= tol32(N) * xmax, (N, nbw, nev, cplx)
    assert np.all(pad == 7.25)


@pytest.mark.parametrize("cplx,nbw", WIDTHS)
def test_edge_rows(cplx, nbw):
    for N in (2, 3, 17, nbw - 1, nbw, nbw + 1, nbw + 2, 2 * nbw - 1, 2 * nbw + 1, 3 * nbw + 5):
        _check(N, nbw, 7, cplx)


@pytest.mark.parametrize("cplx,nbw", WIDTHS)
@pytest.mark.parametrize("nev", [1, 31, 32, 33, 100])
def test_edge_columns(cplx, nbw, nev):
    _check(3 * nbw + 5, nbw, nev, cplx)


@pytest.mark.parametrize("cplx,nbw", WIDTHS)
def test_leading_dimension_and_alignment(cplx, nbw):
    N = 2 * nbw + 9
    _check(N, nbw, 19, cplx, ldq=N + 7)             # 16-byte vector path (N + 7 a multiple of 4 when N = 2 nbw + 9)
    _check(N, nbw, 19, cplx, ldq=N + 2)             # scalar path (real) / vector path only if even (complex)
    _check(N, nbw, 19, cplx, ldq=N + 7, offset=1)   # q not 16-byte aligned
    _check(N + 3, nbw, 40, cplx)


@pytest.mark.parametrize("cplx,nbw", WIDTHS)
def test_many_strips_and_ctas(cplx, nbw):
    _check(5 * nbw + 3, nbw, 148 * 32 + 32 * 9 + 5, cplx)       # more strips than SMs: 1-2 warps per CTA, ragged strip
    if nbw == 32:
        _check(70, nbw, 148 * 8 * 32 + 32 * 40 + 3, cplx)       # more than one wave of 8-strip CTAs


@pytest.mark.parametrize("cplx", [False, True])
def test_larger_problem(cplx):
    _check(1500, 64, 64, cplx)


def test_degenerate_and_identity():
    import torch

    from paper_2002_10991_b200 import binding

    for N, nev in ((0, 5), (1, 5), (40, 0)):
        x = np.zeros((N, nev), order="F", dtype=np.float32)
        got, _ = _run(N, 32, np.zeros((0, 32), np.float32), np.zeros(0, np.float32), x)
        assert got.shape == (N, nev)
    N, nbw, nev = 200, 64, 50
    G = orc.hh_count(N, nbw)
    v = np.zeros((G, nbw), np.float32)
    v[:, 0] = 1.0
    x = np.asfortranarray(np.random.default_rng(3).standard_normal((N, nev)).astype(np.float32))
    got, _ = _run(N, nbw, v, np.zeros(G, np.float32), x)
    assert np.array_equal(got, x)
    # widths the FP32 path does not instantiate
    for dt, nbw in ((torch.float32, 160), (torch.complex64, 128), (torch.float32, 48)):
        G = binding.hh_count(300, nbw)
        with pytest.raises(binding.Elpa2BtError) as ei:
            binding.trans_ev_tridi_to_band(300, nbw, torch.zeros((G, nbw), dtype=dt, device="cuda"),
                                           torch.zeros((G,), dtype=dt, device="cuda"),
                                           torch.zeros((4, 300), dtype=dt, device="cuda").t())
        assert ei.value.rc == -2


@pytest.mark.parametrize("cplx", [False, True])
def test_host_entry_point(cplx):
    from paper_2002_10991_b200 import binding

    N, nbw, nev = 260, 64, 45
    v32, t32, x32 = _inputs(N, nbw, nev, cplx, seed=5)
    want = np.array(x32, order="F", copy=True)
    orc.back_transform(N, nbw, v32, t32, want)
    y = np.array(x32, order="F", copy=True)
    binding.trans_ev_tridi_to_band_host(N, nbw, v32, t32, y)
    assert np.abs(y - want).max() <= tol32(N) * np.abs(x32).max()
    assert binding.last_launch_count() == 1
