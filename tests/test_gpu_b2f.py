"""GPU parity of the band -> full back-transformation (Eq. 6e PAPER.md:93,
``elpa2_trans_ev_band_to_full_*``) against the oracle's plain sequential application
(``orc_band_to_full_back_*``), element by element.

Reflectors: the oracle's own full -> band reduction (Eq. 6a) of a seeded dense matrix at sizes where its
O(N^3) loop finishes in seconds; the seeded synthetic unitary set (``synthetic_full_reflectors``, same
layout) at the larger sizes, including the shape ``bench.py --step 6e`` times, on sampled columns.
Tolerance: the back-transformation's: 1e-11 ||X||_max, and the tighter
diagnostic 1.6e-13 sqrt(N/64) that would expose a skipped reflector.
"""
import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import synth_inputs as si
from helpers import band_from_dense, fortran

pytestmark = pytest.mark.gpu

TOL = 1e-11


def _tight(N):
    return 1.6e-13 * max(1.0, N / 64.0) ** 0.5


def _x(N, nev, seed, cplx):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((N, nev))
    if cplx:
        x = x + 1j * rng.standard_normal((N, nev))
    return np.asfortranarray(x)


def _run_gpu(N, nbw, hv, tau, x, ldq=None, ldv=None, q_offset=0):
    """hv (N, Nv) / tau numpy -> device with the requested leading dimensions; returns (result, padding rows)."""
    import torch

    from paper_2002_10991_b200 import binding

    nev = x.shape[1]
    Nv = hv.shape[1]
    ldq = ldq or max(N, 1)
    ldv = ldv or (N + (N & 1))
    dt = torch.complex128 if np.iscomplexobj(x) else torch.float64
    flat = torch.full((nev * ldq + q_offset,), 7.25, dtype=dt, device="cuda")
    back = flat[q_offset:].view(nev, ldq)
    q = back.t()[:N, :]
    if N and nev:
        q.copy_(torch.from_numpy(np.ascontiguousarray(x)).cuda())
    vback = torch.zeros((max(Nv, 1), ldv), dtype=dt, device="cuda")
    if Nv:
        vback[:Nv, :N] = torch.from_numpy(np.ascontiguousarray(hv.T)).cuda()
    dv = vback[:Nv].t()[:N, :]
    dtau = torch.from_numpy(np.ascontiguousarray(tau)).cuda()
    binding.trans_ev_band_to_full(N, nbw, dv, dtau, q)
    torch.cuda.synchronize()
    return q.cpu().numpy(), back.t()[N:, :].cpu().numpy()


def _oracle(N, nbw, hv, tau, x):
    y = np.array(x, order="F", copy=True)
    orc.band_to_full_back(N, nbw, np.asfortranarray(hv), tau, y)
    return y


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw,nev", [(34, 32, 5), (35, 32, 8), (50, 32, 3), (97, 32, 17), (100, 64, 33), (129, 64, 64),
                                       (200, 32, 40), (257, 128, 9), (300, 16, 31), (333, 48, 20), (500, 64, 130)])
def test_b2f_matches_oracle_on_reduction_output(N, nbw, nev, cplx):
    """Reflectors from the oracle's Eq. 6a reduction of a dense seeded matrix (ragged N, nev, short last block)."""
    H = si.dense_hermitian(N, 700 + N, cplx)
    hv, tau = orc.full_to_band(fortran(H), nbw)
    x = _x(N, nev, N + nev, cplx)
    want = _oracle(N, nbw, hv, tau, x)
    got, pad = _run_gpu(N, nbw, hv, tau, x)
    err = np.abs(got - want).max() / np.abs(x).max()
    assert err <= TOL and err <= _tight(N), (N, nbw, nev, err)


@pytest.mark.parametrize("cplx", [False, True])
def test_b2f_leading_dimensions_alignment_and_padding(cplx):
    N, nbw, nev = 203, 32, 21
    H = si.dense_hermitian(N, 5, cplx)
    hv, tau = orc.full_to_band(fortran(H), nbw)
    x = _x(N, nev, 9, cplx)
    want = _oracle(N, nbw, hv, tau, x)
    for ldq, ldv, off in ((N, N + 1, 0), (N + 5, N + 7, 0), (N + 4, N + 1, 1), (N + 2, N + 3, 0)):
        got, pad = _run_gpu(N, nbw, hv, tau, x, ldq=ldq, ldv=ldv, q_offset=off)
        assert np.abs(got - want).max() / np.abs(x).max() <= _tight(N), (ldq, ldv, off)
        assert np.all(pad == 7.25), (ldq, ldv, off)          # rows >= N of every column untouched


@pytest.mark.parametrize("cplx", [False, True])
def test_b2f_no_work_and_identity_reflectors(cplx):
    import torch

    from paper_2002_10991_b200 import binding

    dt = np.complex128 if cplx else np.float64
    # Nv = 0 (band as wide as the matrix), nev = 0
    for N, nbw, nev in ((10, 16, 4), (33, 32, 4), (100, 32, 0), (0, 32, 3)):
        x = _x(N, nev, 1, cplx)
        hv = np.zeros((N, max(N - nbw - 1, 0)), dtype=dt)
        got, _ = _run_gpu(N, nbw, hv, np.zeros(hv.shape[1], dtype=dt), x)
        assert np.array_equal(got, x)
        assert binding.last_launch_count() == 0
    # tau = 0 everywhere: q comes back bit for bit
    N, nbw, nev = 150, 32, 24
    Nv = N - nbw - 1
    hv = np.zeros((N, Nv), dtype=dt)
    hv[np.arange(Nv) + nbw, np.arange(Nv)] = 1.0
    x = _x(N, nev, 2, cplx)
    got, _ = _run_gpu(N, nbw, hv, np.zeros(Nv, dtype=dt), x)
    assert np.array_equal(got, x)
    assert binding.last_launch_count() == 2


@pytest.mark.parametrize("cplx", [False, True])
def test_b2f_end_to_end_on_device(cplx):
    """6a (oracle) -> 6b, 6d, 6e on the GPU: eigenvectors of the ORIGINAL full matrix."""
    import torch
    from scipy.linalg import eigh_tridiagonal

    from paper_2002_10991_b200 import binding

    N, nbw = 260, 32
    H = si.dense_hermitian(N, 44, cplx)
    A = fortran(H)
    hv, tau = orc.full_to_band(A, nbw)
    ab = band_from_dense(A, nbw)
    dab = torch.from_numpy(np.ascontiguousarray(ab.T)).cuda()
    hh_v, hh_tau, d, e = binding.bulge_chase(N, nbw, dab)                       # 6b on the device
    lam, X = eigh_tridiagonal(d.cpu().numpy(), e.cpu().numpy())                 # 6c (LAPACK, test side)
    q = torch.from_numpy(np.ascontiguousarray(X.astype(H.dtype).T)).cuda().t()
    binding.trans_ev_tridi_to_band(N, nbw, hh_v, hh_tau, q)                     # 6d
    vback = torch.zeros((hv.shape[1], N + (N & 1)), dtype=q.dtype, device="cuda")
    vback[:, :N] = torch.from_numpy(np.ascontiguousarray(hv.T)).cuda()
    binding.trans_ev_band_to_full(N, nbw, vback.t()[:N, :], torch.from_numpy(tau).cuda(), q)   # 6e
    torch.cuda.synchronize()
    C = q.cpu().numpy()
    nH = np.linalg.norm(H, 2)
    assert np.abs(H @ C - C * lam[None, :]).max() / nH <= 1e-12 * N
    assert np.abs(C.conj().T @ C - np.eye(N)).max() <= 1e-12 * N


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw,nev,nsamp", [(1500, 64, 2500, 64), (4096, 64, 20000, 64)])
def test_b2f_many_slabs_synthetic(N, nbw, nev, nsamp, cplx):
    """More than one round of 16 (complex: 8) slabs per CTA (nev = 20000: 2500 slabs on 148 CTAs), several waves of
    T-factor CTAs; synthetic unitary reflectors; sampled columns + the norm of every column."""
    import torch

    from paper_2002_10991_b200 import binding

    dv, dtau = si.synthetic_full_reflectors(N, nbw, 31, cplx, "cuda")
    q = si.gaussian_block(N, nev, 32, cplx, "cuda")
    cols = si.sample_columns(nev, nsamp, 33)
    # always include the first and last slab and a round boundary
    cols = np.unique(np.concatenate([cols, [0, 7, nev - 1, min(nev - 1, 148 * 16 * 8 - 1), min(nev - 1, 148 * 16 * 8)]]))
    ct = torch.from_numpy(cols).cuda()
    xs = np.asfortranarray(q[:, ct].cpu().numpy())
    nrm0 = torch.linalg.vector_norm(q, dim=0)
    binding.trans_ev_band_to_full(N, nbw, dv, dtau, q)
    torch.cuda.synchronize()
    got = q[:, ct].cpu().numpy()
    nrm1 = torch.linalg.vector_norm(q, dim=0)
    want = _oracle(N, nbw, dv.cpu().numpy(), dtau.cpu().numpy(), xs)
    err = np.abs(got - want).max() / np.abs(xs).max()
    assert err <= TOL and err <= _tight(N), err
    assert float((nrm1 / nrm0 - 1.0).abs().max().item()) <= 1e-12
