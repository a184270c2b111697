"""Test-side helpers (numpy only).  Nothing here is imported by the product or by oracle/."""
from __future__ import annotations

import numpy as np


def dense_from_band(ab: np.ndarray, nbw: int) -> np.ndarray:
    """Full Hermitian matrix from the lower band storage ab[i-j, j] = B[i, j]."""
    N = ab.shape[1]
    B = np.zeros((N, N), dtype=ab.dtype)
    for j in range(N):
        for d in range(min(nbw, N - 1 - j) + 1):
            B[j + d, j] = ab[d, j]
            B[j, j + d] = np.conj(ab[d, j])
    return B


def tridiag_dense(d: np.ndarray, e: np.ndarray) -> np.ndarray:
    return np.diag(d) + np.diag(e, 1) + np.diag(e, -1)


def dense_reflector(N: int, r0: int, v: np.ndarray, tau) -> np.ndarray:
    """H = I - tau v v^H embedded at rows r0.. (textbook definition, Eq. 7)."""
    H = np.eye(N, dtype=np.result_type(v.dtype, np.float64))
    L = v.shape[0]
    H[r0:r0 + L, r0:r0 + L] -= tau * np.outer(v, np.conj(v))
    return H


def fortran(a: np.ndarray) -> np.ndarray:
    return np.array(a, order="F", copy=True)


def band_from_dense(B: np.ndarray, nbw: int) -> np.ndarray:
    """Lower band storage (2 nbw + 1, N), Fortran order, of a Hermitian band matrix given in full:
    ab[i-j, j] = B[i, j] for 0 <= i-j <= nbw (rows nbw+1 .. 2 nbw stay zero: room for the chase)."""
    N = B.shape[0]
    ab = np.zeros((2 * nbw + 1, N), dtype=B.dtype, order="F")
    for d in range(min(nbw, N - 1) + 1):
        ab[d, : N - d] = np.diagonal(B, -d)
    return ab
