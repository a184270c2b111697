"""Pins DESIGN.md reading R6 on the CPU: the aggregate the default CUDA path applies per block,
H_7 ... H_0 = I - V T V^H with T[j][j] = tau_j, T[j][:j] = -tau_j (v_j^H V[:, :j]) T[:j, :j], equals the product of
the eight dense textbook reflectors of a block of chase output (first rows 8b+7 .. 8b, applied in that order),
including blocks with identity slots (tau = 0) and the complex length-1 phase rotation (R4), and Y = V(-T)
reproduces x + Y (V^H x).  numpy only: no CUDA, no oracle arithmetic beyond producing the reflectors."""
import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import synth_inputs as si
from helpers import dense_reflector


def _block(N, nbw, hh_v, hh_tau, k, b):
    """(r0_i, v_i, tau_i) of the reflectors with first rows 8b+7 .. 8b of chain k, in application order."""
    out = []
    for i in range(8):
        r0 = 8 * b + 7 - i
        s = r0 - 1 - k * nbw
        if r0 > N - 1 or s < 0:
            out.append((r0, None, 0.0))
            continue
        g = orc.hh_offset(N, nbw, s) + k
        L = min(nbw, N - r0)
        out.append((r0, hh_v[g, :L].copy(), hh_tau[g]))
    return out


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw", [(70, 32), (150, 32), (200, 64)])
def test_compact_wy_equals_product_of_reflectors(N, nbw, cplx):
    ab = si.band_matrix(N, nbw, 31 + N, cplx)
    hh_v, hh_tau, _, _ = orc.bulge_chase(ab, nbw)
    K0 = (N - 2 + nbw) // nbw
    bhi = (N - 1) // 8
    rng = np.random.default_rng(5)
    checked = 0
    for k in range(K0):
        for b in (bhi, (bhi + k * nbw // 8) // 2, k * nbw // 8):       # first, middle and last block of the chain
            refl = _block(N, nbw, hh_v, hh_tau, k, b)
            W = nbw + 8
            V = np.zeros((W, 8), dtype=hh_v.dtype)
            tau = np.zeros(8, dtype=hh_v.dtype)
            P = np.eye(N + W, dtype=hh_v.dtype)                         # rows beyond N: zero padding of v
            for i, (r0, v, t) in enumerate(refl):
                if v is None:
                    continue
                V[7 - i:7 - i + len(v), i] = v
                tau[i] = t
                P = dense_reflector(N + W, r0, v, t) @ P                # H_i applied after H_{i-1}
            T = np.zeros((8, 8), dtype=hh_v.dtype)
            S = V.conj().T @ V
            for j in range(8):
                T[j, j] = tau[j]
                T[j, :j] = -tau[j] * (S[j, :j] @ T[:j, :j])
            Pw = np.eye(N + W, dtype=hh_v.dtype)
            Pw[8 * b:8 * b + W, 8 * b:8 * b + W] -= V @ T @ V.conj().T
            assert np.abs(Pw - P).max() <= 1e-13
            # the form the kernel evaluates: x += Y (V^H x), Y = V (-T)
            x = rng.standard_normal((N + W, 3)) + (1j * rng.standard_normal((N + W, 3)) if cplx else 0)
            y = x.copy()
            y[8 * b:8 * b + W] += (V @ -T) @ (V.conj().T @ x[8 * b:8 * b + W])
            assert np.abs(y - P @ x).max() <= 1e-12
            checked += 1
    assert checked >= 3
