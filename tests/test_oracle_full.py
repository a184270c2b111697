"""Pins for orc_full_to_band_{d,z} (Eq. 6a) and orc_band_to_full_back_{d,z} (Eq. 6e
PAPER.md:93), reading R15 of DESIGN.md: P* = H_0 H_1 .. H_{Nv-1}, reflector j clears column j below the
band (rows j+nbw .. N-1).

The oracle is the plain unblocked definition; it is pinned against (a) the dense product Qf of
textbook reflectors built here in numpy: Qf^H H Qf = B, banded, Qf unitary; (b) numpy's dense
eigenvalues; (c) the special case nbw = 1, which is LAPACK's one-stage tridiagonalization
(scipy.linalg.hessenberg, same Householder convention); (d) nbw >= N-1: nothing to do; (e) the
back-transformation equals Qf Y, Y = I returns Qf, column norms are preserved, a wrong order / a
conjugated tau / an unconjugated v give O(1) errors; (f) the whole chain 6a -> 6b -> 6c -> 6d -> 6e
reproduces eigenpairs of the ORIGINAL full matrix.
"""
import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import synth_inputs as si
from helpers import band_from_dense, dense_reflector, fortran


def _qf(N, nbw, hv, tau):
    Q = np.eye(N, dtype=hv.dtype)
    for j in range(hv.shape[1]):
        Q = Q @ dense_reflector(N, j + nbw, hv[j + nbw:, j], tau[j])
    return Q


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw", [(3, 1), (6, 2), (17, 4), (40, 7), (64, 32), (50, 32), (70, 3), (33, 31), (96, 16)])
def test_full_to_band_against_dense_reflectors(N, nbw, cplx):
    H = si.dense_hermitian(N, 100 + N, cplx)
    A = fortran(H)
    hv, tau = orc.full_to_band(A, nbw)
    Nv = max(N - nbw - 1, 0)
    assert hv.shape == (N, Nv) and tau.shape == (Nv,)
    # layout: unit head stored, zeros above it
    for j in range(Nv):
        assert hv[j + nbw, j] == 1.0
        assert np.all(hv[: j + nbw, j] == 0.0)
    Qf = _qf(N, nbw, hv, tau)
    nH = np.linalg.norm(H, 2)
    assert np.abs(Qf.conj().T @ Qf - np.eye(N)).max() <= 1e-13 * N
    B = Qf.conj().T @ H @ Qf
    assert np.abs(B - A).max() <= 1e-13 * N * nH
    # banded, Hermitian, real diagonal
    i, j = np.indices((N, N))
    assert np.all(A[np.abs(i - j) > nbw] == 0.0)
    assert np.abs(A - A.conj().T).max() <= 1e-13 * N * nH
    assert np.all(np.diagonal(A).imag == 0.0) if cplx else True
    # same spectrum as the full matrix
    assert np.abs(np.linalg.eigvalsh(A) - np.linalg.eigvalsh(H)).max() <= 1e-12 * N * nH
    # every head element below the band is real (beta of larfg), so the band edge is real
    assert np.abs(np.diagonal(A, -nbw)[:Nv].imag).max(initial=0.0) == 0.0


@pytest.mark.parametrize("N", [5, 30, 61])
def test_nbw_one_is_lapack_tridiagonalization(N):
    """nbw = 1: one reflector per column on rows j+1.. -- dsytrd / dgehrd's algorithm with the same
    larfg convention, so d and e agree with LAPACK to rounding (signs included)."""
    from scipy.linalg import hessenberg

    H = si.dense_hermitian(N, 7, False)
    A = fortran(H)
    orc.full_to_band(A, 1)
    T = hessenberg(H)
    scale = np.abs(H).max() * N
    assert np.abs(np.diagonal(A) - np.diagonal(T)).max() <= 1e-13 * scale
    assert np.abs(np.diagonal(A, -1) - np.diagonal(T, -1)).max() <= 1e-13 * scale


@pytest.mark.parametrize("cplx", [False, True])
def test_wide_band_needs_no_reflector(cplx):
    N = 12
    H = si.dense_hermitian(N, 3, cplx)
    for nbw in (N - 1, N, 40):
        A = fortran(H)
        hv, tau = orc.full_to_band(A, nbw)
        assert hv.shape[1] == 0 and tau.size == 0 and np.array_equal(A, H)
        Y = fortran(H[:, :3])
        orc.band_to_full_back(N, nbw, hv, tau, Y)
        assert np.array_equal(Y, H[:, :3])


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw,ncols", [(6, 2, 4), (17, 4, 12), (40, 7, 9), (64, 32, 64), (70, 3, 5)])
def test_back_transform_equals_dense_qf(N, nbw, ncols, cplx):
    H = si.dense_hermitian(N, 200 + N, cplx)
    hv, tau = orc.full_to_band(fortran(H), nbw)
    Qf = _qf(N, nbw, hv, tau)
    rng = np.random.default_rng(N)
    X = rng.standard_normal((N, ncols)) + (1j * rng.standard_normal((N, ncols)) if cplx else 0)
    Y = fortran(X)
    orc.band_to_full_back(N, nbw, hv, tau, Y)
    assert np.abs(Y - Qf @ X).max() <= 1e-13 * N
    E = fortran(np.eye(N, dtype=hv.dtype))
    orc.band_to_full_back(N, nbw, hv, tau, E)
    assert np.abs(E - Qf).max() <= 1e-13 * N
    assert np.abs(np.linalg.norm(Y, axis=0) - np.linalg.norm(X, axis=0)).max() <= 1e-13 * N
    # ldq > N and a single column: padding untouched, columns independent bit for bit
    big = np.full((N + 3, ncols), 7.0, dtype=X.dtype, order="F")
    big[:N] = X
    orc.band_to_full_back(N, nbw, hv, tau, big[:N])
    assert np.all(big[N:] == 7.0) and np.array_equal(big[:N], Y)
    one = fortran(X[:, 1:2])
    orc.band_to_full_back(N, nbw, hv, tau, one)
    assert np.array_equal(one[:, 0], Y[:, 1])


@pytest.mark.parametrize("cplx", [False, True])
def test_order_and_conjugation_matter(cplx):
    N, nbw = 30, 4
    H = si.dense_hermitian(N, 11, cplx)
    hv, tau = orc.full_to_band(fortran(H), nbw)
    Qf = _qf(N, nbw, hv, tau)
    X = np.eye(N, dtype=hv.dtype)
    good = fortran(X)
    orc.band_to_full_back(N, nbw, hv, tau, good)
    assert np.abs(good - Qf).max() <= 1e-13 * N
    # generation order instead of reverse order: H_{Nv-1} .. H_0 X = Qf^H-like product, O(1) off
    wrong = X.copy()
    for j in range(hv.shape[1]):
        wrong = dense_reflector(N, j + nbw, hv[j + nbw:, j], tau[j]) @ wrong
    assert np.abs(wrong - Qf).max() > 1e-2
    if cplx:
        conj_tau = np.eye(N, dtype=hv.dtype)
        for j in range(hv.shape[1]):
            conj_tau = conj_tau @ dense_reflector(N, j + nbw, hv[j + nbw:, j], np.conj(tau[j]))
        assert np.abs(conj_tau - Qf).max() > 1e-3


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw", [(48, 4), (120, 8), (256, 32)])
def test_end_to_end_eigenpairs_of_the_full_matrix(N, nbw, cplx):
    """Eq. 6a -> 6b -> 6c -> 6d -> 6e, all in the oracle: C = P* Q* X are eigenvectors of H."""
    H = si.dense_hermitian(N, 300 + N, cplx)
    A = fortran(H)
    hv, tau = orc.full_to_band(A, nbw)                           # 6a
    ab = band_from_dense(A, nbw)
    hh_v, hh_tau, d, e = orc.bulge_chase(ab, nbw)                # 6b
    lam, X = orc.tridiag_ql(d, e)                                # 6c
    Y = fortran(X.astype(H.dtype))
    orc.back_transform(N, nbw, hh_v, hh_tau, Y)                  # 6d
    orc.band_to_full_back(N, nbw, hv, tau, Y)                    # 6e
    nH = np.linalg.norm(H, 2)
    assert np.abs(H @ Y - Y * lam[None, :]).max() / nH <= 1e-12 * N
    assert np.abs(Y.conj().T @ Y - np.eye(N)).max() <= 1e-12 * N
    assert np.abs(lam - np.linalg.eigvalsh(H)).max() <= 1e-12 * N * nH
