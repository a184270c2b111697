"""Pins for orc_back_transform_{d,z} (Eq. 6d, Eq. 8).

The oracle is the plain definition; it is pinned against (a) the closed form Q2 X with Q2 built by
numpy from dense reflectors, (b) X = I returning Q2, (c) unitarity (column norms), (d) the
end-to-end eigen-residual with the ORIGINAL band matrix, (e) the paper's order statement
("reverse of the order in which they are generated"): applying in generation order
instead must NOT reproduce the result, and (f) conjugation conventions (R2).
"""
import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import synth_inputs as si
from helpers import dense_from_band, dense_reflector, fortran


def _reflector_list(N, nbw):
    out = []
    g = 0
    for s in range(N - 1):
        for k in range(orc.hh_blocks(N, nbw, s)):
            r0, r1, L = orc.hh_rows(N, nbw, s, k)
            out.append((g, s, k, r0, L))
            g += 1
    return out


def _q2(N, nbw, hh_v, hh_tau):
    Q = np.eye(N, dtype=hh_v.dtype)
    for g, s, k, r0, L in _reflector_list(N, nbw):
        Q = Q @ dense_reflector(N, r0, hh_v[g, :L], hh_tau[g])
    return Q


def _chase(N, nbw, seed, cplx):
    ab = si.band_matrix(N, nbw, seed, cplx)
    B = dense_from_band(ab, nbw)
    hh_v, hh_tau, d, e = orc.bulge_chase(fortran(ab), nbw)
    return B, hh_v, hh_tau, d, e


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw,ncols", [(2, 2, 3), (3, 2, 1), (17, 4, 12), (40, 7, 9), (64, 32, 64),
                                         (50, 32, 5), (33, 32, 7)])
def test_back_transform_equals_dense_q2(N, nbw, ncols, cplx):
    B, hh_v, hh_tau, d, e = _chase(N, nbw, 900 + N, cplx)
    Q2 = _q2(N, nbw, hh_v, hh_tau)
    rng = np.random.default_rng(N)
    X = rng.standard_normal((N, ncols)) + (1j * rng.standard_normal((N, ncols)) if cplx else 0)
    Y = fortran(X)
    orc.back_transform(N, nbw, hh_v, hh_tau, Y)
    assert np.abs(Y - Q2 @ X).max() <= 1e-13 * N
    # X = I returns Q2 itself
    E = fortran(np.eye(N, dtype=hh_v.dtype))
    orc.back_transform(N, nbw, hh_v, hh_tau, E)
    assert np.abs(E - Q2).max() <= 1e-13 * N
    # unitary: column norms preserved
    assert np.abs(np.linalg.norm(Y, axis=0) - np.linalg.norm(X, axis=0)).max() <= 1e-13 * N


@pytest.mark.parametrize("cplx", [False, True])
def test_back_transform_ldq_and_column_independence(cplx):
    N, nbw = 45, 4
    B, hh_v, hh_tau, d, e = _chase(N, nbw, 31, cplx)
    rng = np.random.default_rng(1)
    dt = np.complex128 if cplx else np.float64
    big = np.full((N + 5, 11), 7.0, dtype=dt, order="F")
    X = (rng.standard_normal((N, 11)) + (1j * rng.standard_normal((N, 11)) if cplx else 0)).astype(dt)
    big[:N, :] = X
    view = big[:N, :]                      # ldq = N + 5
    orc.back_transform(N, nbw, hh_v, hh_tau, view)
    assert np.all(big[N:, :] == 7.0)       # padding rows untouched
    one = fortran(X[:, 3:4])
    orc.back_transform(N, nbw, hh_v, hh_tau, one)
    assert np.array_equal(one[:, 0], big[:N, 3])   # PAPER.md:134 columns are independent, bit for bit


@pytest.mark.parametrize("cplx", [False, True])
def test_order_and_conjugation_matter(cplx):
    """A wrong order, a conjugated tau, or an unconjugated v in the dot gives an O(1) error:
    the definition pinned above is sensitive to each of these slips."""
    N, nbw = 30, 4
    B, hh_v, hh_tau, d, e = _chase(N, nbw, 3, cplx)
    Q2 = _q2(N, nbw, hh_v, hh_tau)
    rng = np.random.default_rng(2)
    X = rng.standard_normal((N, 4)) + (1j * rng.standard_normal((N, 4)) if cplx else 0)
    Y = fortran(X)
    orc.back_transform(N, nbw, hh_v, hh_tau, Y)
    # generation order applied to X = Q2^H-like product, differs at O(1)
    W = X.copy()
    for g, s, k, r0, L in _reflector_list(N, nbw):
        W = dense_reflector(N, r0, hh_v[g, :L], hh_tau[g]) @ W
    assert np.abs(W - Y).max() > 1e-3
    if cplx:
        Yc = fortran(X)
        orc.back_transform(N, nbw, hh_v, np.conj(hh_tau), Yc)
        assert np.abs(Yc - Q2 @ X).max() > 1e-3
        Yv = fortran(X)
        orc.back_transform(N, nbw, np.conj(hh_v), hh_tau, Yv)
        assert np.abs(Yv - Q2 @ X).max() > 1e-3


@pytest.mark.parametrize("N,nbw,seed", [(64, 8, 1), (200, 32, 2), (512, 32, 1001)])
def test_end_to_end_eigen_residual_real(N, nbw, seed):
    """BASELINE.json configs 1-2 check: ||B Y - Y Lambda|| / ||B|| <= 1e-12 N with Y = Q2 X, X the
    tridiagonal eigenvectors; (512, 32, 1001) IS config 1."""
    B, hh_v, hh_tau, d, e = _chase(N, nbw, seed, False)
    lam, X = orc.tridiag_ql(d, e)
    Y = fortran(X)
    orc.back_transform(N, nbw, hh_v, hh_tau, Y)
    nB = np.linalg.norm(B, 2)
    assert np.abs(B @ Y - Y * lam).max() / nB <= 1e-12 * N
    assert np.abs(Y.T @ Y - np.eye(N)).max() <= 1e-12 * N
    assert np.abs(lam - np.linalg.eigvalsh(B)).max() <= 1e-12 * N * nB


def test_end_to_end_eigen_residual_complex():
    N, nbw = 96, 8
    B, hh_v, hh_tau, d, e = _chase(N, nbw, 9, True)
    lam, X = orc.tridiag_ql(d, e)
    Y = fortran(X.astype(np.complex128))
    orc.back_transform(N, nbw, hh_v, hh_tau, Y)
    nB = np.linalg.norm(B, 2)
    assert np.abs(B @ Y - Y * lam).max() / nB <= 1e-12 * N


@pytest.mark.parametrize("cplx", [False, True])
def test_valid_reorders_are_bit_identical(cplx):
    """DESIGN.md R5: chain-major order (k ascending outermost, s descending inside) applies the
    same reflectors to every row in the same relative order, so a plain numpy replay in that
    order must agree BIT FOR BIT with the oracle's reverse-generation order; k descending
    outermost is wrong at O(1)."""
    N, nbw = 41, 4
    B, hh_v, hh_tau, d, e = _chase(N, nbw, 12, cplx)
    rng = np.random.default_rng(4)
    X = rng.standard_normal((N, 3)) + (1j * rng.standard_normal((N, 3)) if cplx else 0)
    Y = fortran(X)
    orc.back_transform(N, nbw, hh_v, hh_tau, Y)

    def apply(order):
        Z = X.copy()
        for g, s, k, r0, L in order:
            if hh_tau[g] == 0:
                continue
            v = hh_v[g, :L]
            for j in range(Z.shape[1]):
                dot = 0.0
                for r in range(L):
                    dot = dot + np.conj(v[r]) * Z[r0 + r, j]
                td = hh_tau[g] * dot
                for r in range(L):
                    Z[r0 + r, j] = Z[r0 + r, j] - td * v[r]
        return Z

    refl = _reflector_list(N, nbw)
    rev_gen = sorted(refl, key=lambda t: (-t[1], t[2]))
    chain_major = sorted(refl, key=lambda t: (t[2], -t[1]))
    k_desc = sorted(refl, key=lambda t: (-t[2], -t[1]))
    Zr = apply(rev_gen)
    assert np.abs(Zr - Y).max() <= 1e-14          # same order; rounding of complex mul may differ
    assert np.array_equal(apply(chain_major), Zr)  # bit-identical reorder
    assert np.abs(apply(k_desc) - Zr).max() > 1e-3


# ---- FP32 (reading R16): orc_back_transform_{s,c} -------------------------------------
def tol32(N):
    """8 u sqrt(N) ||X||_max, u = 2^-24."""
    return 8.0 * 2.0 ** -24 * np.sqrt(max(N, 1))


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw,ncols", [(17, 4, 12), (64, 32, 20), (300, 32, 9), (700, 64, 5)])
def test_fp32_back_transform_pinned_to_dense_q2_and_fp64(N, nbw, ncols, cplx):
    """The FP32 oracle against (a) the dense closed form Q2 X built by numpy in FP64 from the SAME rounded
    reflectors (tiny N), (b) the FP64 oracle on the same rounded inputs, (c) column norms; (d) the
    generation-order application misses by O(1)."""
    _, hh_v, hh_tau, _, _ = _chase(N, nbw, 300 + N, cplx)
    f32, f64 = (np.complex64, np.complex128) if cplx else (np.float32, np.float64)
    v32, t32 = hh_v.astype(f32), hh_tau.astype(f32)
    rng = np.random.default_rng(N)
    X = (rng.standard_normal((N, ncols)) + (1j * rng.standard_normal((N, ncols)) if cplx else 0)).astype(f32)
    Y = fortran(X)
    orc.back_transform(N, nbw, v32, t32, Y)
    assert Y.dtype == f32
    xmax = np.abs(X).max()
    Y64 = fortran(X.astype(f64))
    orc.back_transform(N, nbw, v32.astype(f64), t32.astype(f64), Y64)
    assert np.abs(Y - Y64).max() <= tol32(N) * xmax
    if N <= 64:
        Q2 = _q2(N, nbw, v32.astype(f64), t32.astype(f64))
        assert np.abs(Y - Q2 @ X.astype(f64)).max() <= tol32(N) * xmax
    n0, n1 = np.linalg.norm(X.astype(f64), axis=0), np.linalg.norm(Y.astype(f64), axis=0)
    assert np.abs(n1 / n0 - 1.0).max() <= tol32(N) * 4
    # applied in generation order instead (forward over the slots): O(1) away
    Z = X.astype(f64)
    for g, s, k, r0, L in _reflector_list(N, nbw):
        v, t = v32[g, :L].astype(f64), f64(t32[g])
        Z[r0:r0 + L] -= t * np.outer(v, v.conj() @ Z[r0:r0 + L])
    if N >= 64:
        assert np.abs(Z - Y64).max() > 1e-2 * xmax
