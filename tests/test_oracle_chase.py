"""Pins for the oracle's Householder generator, bulge chase and tridiagonal QL.

None of these compare the oracle with itself: they use the dense definition H = I - tau v v^H
(Eq. 7) formed by numpy, numpy.linalg.eigvalsh as the brute-force eigensolver, and
algebraic invariants (SURVEY.md 8(c) "What pins each part").
"""
import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import synth_inputs as si
from helpers import dense_from_band, dense_reflector, tridiag_dense, fortran

TOL = 1e-13


# ----------------------------------------------------------------------------- larfg (O2)
@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("L", [1, 2, 3, 8, 64])
def test_larfg_invariants(L, cplx):
    rng = np.random.default_rng(100 + L + 1000 * cplx)
    for trial in range(6):
        x = rng.uniform(-1, 1, L) + (1j * rng.uniform(-1, 1, L) if cplx else 0)
        if trial == 1:
            x[0] = -x[0]
        if trial == 2 and L > 1:
            x[0] = 0.0                       # sign(0) = +1 branch
        v, tau, beta = orc.larfg(x)
        assert v[0] == 1.0
        H = dense_reflector(L, 0, v, tau)
        y = H.conj().T @ x
        nrm = np.linalg.norm(x)
        assert abs(y[0] - beta) <= TOL * max(nrm, 1)
        assert np.abs(y[1:]).max(initial=0.0) <= TOL * max(nrm, 1)
        assert abs(abs(beta) - nrm) <= TOL * max(nrm, 1)          # |beta| = ||x||
        assert np.abs(H.conj().T @ H - np.eye(L)).max() <= TOL    # unitary
        if L > 1 or (cplx and x[0].imag != 0):
            # beta = -sign(Re alpha) ||x||
            assert np.sign(beta) == (-1.0 if x[0].real >= 0 else 1.0)
        if not cplx and L > 1:
            assert 1.0 <= tau <= 2.0


def test_larfg_identity_cases():
    v, tau, beta = orc.larfg(np.array([0.75, 0.0, 0.0]))
    assert tau == 0 and beta == 0.75 and list(v) == [1.0, 0.0, 0.0]
    v, tau, beta = orc.larfg(np.array([-0.5]))
    assert tau == 0 and beta == -0.5
    # complex length-1 with an imaginary part is a phase rotation that makes beta real (R4)
    v, tau, beta = orc.larfg(np.array([0.3 + 0.4j]))
    assert abs(beta + 0.5) < 1e-15 and abs((1 - np.conj(tau)) * (0.3 + 0.4j) - beta) < 1e-15


# ----------------------------------------------------------------------------- chase (O3/O4)
def _q2_dense(N, nbw, hh_v, hh_tau):
    """Q2 = H_1 H_2 ... H_G (generation order), each H formed from the dense definition."""
    Q = np.eye(N, dtype=hh_v.dtype)
    g = 0
    for s in range(N - 1):
        for k in range(orc.hh_blocks(N, nbw, s)):
            r0, r1, L = orc.hh_rows(N, nbw, s, k)
            Q = Q @ dense_reflector(N, r0, hh_v[g, :L], hh_tau[g])
            g += 1
    return Q


CASES = [(5, 2), (9, 3), (17, 4), (23, 7), (40, 4), (64, 32), (45, 32), (33, 2), (12, 3)]


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw", CASES)
def test_chase_reduces_to_tridiagonal(N, nbw, cplx):
    ab = si.band_matrix(N, nbw, 500 + N + nbw, cplx)
    B = dense_from_band(ab, nbw)
    work = fortran(ab)
    hh_v, hh_tau, d, e = orc.bulge_chase(work, nbw)
    T = tridiag_dense(d, e)
    Q2 = _q2_dense(N, nbw, hh_v, hh_tau)
    scale = np.abs(B).max() * N
    assert np.abs(Q2.conj().T @ Q2 - np.eye(N)).max() <= TOL
    R = Q2.conj().T @ B @ Q2
    assert np.abs(R - T).max() <= TOL * scale               # includes everything off the tridiagonal
    assert np.abs(R.imag).max() <= TOL * scale if cplx else True
    # brute-force dense eigenvalues of B equal those of T
    assert np.abs(np.linalg.eigvalsh(B) - np.linalg.eigvalsh(T)).max() <= TOL * scale
    assert abs(np.trace(B).real - d.sum()) <= TOL * scale
    assert abs(np.linalg.norm(B) - np.linalg.norm(T)) <= TOL * scale
    # what is left in the work array is T and nothing else
    left = np.array(work)
    assert np.abs(left[2:, :]).max(initial=0.0) == 0.0 or np.abs(left[2:, :]).max() <= TOL * scale
    # stored vectors: v[0] = 1, zero padded beyond L (R8); identity slots have tau = 0
    g = 0
    nonid = 0
    for s in range(N - 1):
        for k in range(orc.hh_blocks(N, nbw, s)):
            _, _, L = orc.hh_rows(N, nbw, s, k)
            assert hh_v[g, 0] == 1.0
            assert not np.any(hh_v[g, L:])
            nonid += hh_tau[g] != 0
            g += 1
    want = sum(-(-(N - 2 - s) // nbw) for s in range(N - 2))   # R3: ceil((N-2-s)/nbw), s <= N-3
    assert nonid == want + (1 if cplx and N >= 2 else 0)      # R4: complex phase slot (N-2, 0)


@pytest.mark.parametrize("cplx", [False, True])
def test_chase_fill_bound(cplx):
    """The fill never exceeds distance 2*nbw-1 (O1): give the chase extra room and look."""
    N, nbw = 40, 4
    ab = si.band_matrix(N, nbw, 77, cplx)
    B = dense_from_band(ab, nbw)
    # replay the reflectors densely and record the widest intermediate band
    hh_v, hh_tau, d, e = orc.bulge_chase(fortran(ab), nbw)
    A = B.copy()
    g = 0
    widest = 0
    for s in range(N - 1):
        for k in range(orc.hh_blocks(N, nbw, s)):
            r0, r1, L = orc.hh_rows(N, nbw, s, k)
            H = dense_reflector(N, r0, hh_v[g, :L], hh_tau[g])
            A = H.conj().T @ A @ H
            ii, jj = np.nonzero(np.abs(A) > 1e-12)
            widest = max(widest, int(np.abs(ii - jj).max()))
            g += 1
    assert widest <= 2 * nbw - 1
    assert np.abs(A - tridiag_dense(d, e)).max() <= 1e-12


@pytest.mark.parametrize("cplx", [False, True])
def test_chase_wide_band_is_one_stage_householder(cplx):
    """nbw >= N-1: one reflector per column = textbook Householder tridiagonalization; each
    reflector must annihilate its column of the current matrix below the sub-diagonal."""
    N, nbw = 12, 32
    rng = np.random.default_rng(5)
    A = rng.uniform(-1, 1, (N, N)) + (1j * rng.uniform(-1, 1, (N, N)) if cplx else 0)
    A = (A + A.conj().T) / 2
    ab = np.zeros((2 * nbw + 1, N), dtype=A.dtype, order="F")
    for j in range(N):
        for dd in range(N - j):
            ab[dd, j] = A[j + dd, j]
    hh_v, hh_tau, d, e = orc.bulge_chase(ab, nbw)
    assert orc.hh_count(N, nbw) == N - 1
    M = A.copy()
    for s in range(N - 1):
        L = N - 1 - s
        H = dense_reflector(N, s + 1, hh_v[s, :L], hh_tau[s])
        M = H.conj().T @ M @ H
        assert np.abs(M[s + 2:, s]).max(initial=0.0) <= 1e-13
    assert np.abs(M - tridiag_dense(d, e)).max() <= 1e-13


# ----------------------------------------------------------------------------- QL (O5)
@pytest.mark.parametrize("N", [1, 2, 3, 10, 64, 200])
def test_tridiag_ql(N):
    rng = np.random.default_rng(N)
    d = rng.uniform(-1, 1, N)
    e = rng.uniform(-1, 1, max(N - 1, 0))
    if N == 10:
        e[4] = 0.0        # a split
    lam, X = orc.tridiag_ql(d, e)
    T = tridiag_dense(d, e) if N > 1 else np.array([[d[0]]])
    assert np.all(np.diff(lam) >= 0)
    assert np.abs(lam - np.linalg.eigvalsh(T)).max() <= 1e-13 * N
    assert np.abs(T @ X - X * lam).max() <= 1e-13 * N
    assert np.abs(X.T @ X - np.eye(N)).max() <= 1e-13 * N
    # Sturm count: number of eigenvalues below a shift = negative pivots of T - shift
    for shift in (-0.5, 0.0, 0.3):
        cnt, p = 0, 1.0
        for i in range(N):
            p = d[i] - shift - (e[i - 1] ** 2 / p if i > 0 else 0.0)
            if p == 0.0:
                p = 1e-300
            cnt += p < 0
        assert cnt == int(np.sum(lam < shift))
