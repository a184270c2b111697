"""Seeded synthetic inputs shared by the tests, the oracle legs and bench.py.

This module holds NONE of the method's arithmetic (no Householder generation, no reflector
application, no layout formulas): it only draws numbers.  It imports neither ``oracle`` nor the
CUDA binding.  Recipes:

* band matrix B ("random ... matrices"; after full->band reduction a random dense
  matrix leaves a band without special structure): entry (i, j), 0 <= i-j <= nbw, is a
  counter-based hash of (seed, j*(nbw+1) + (i-j), re/im) mapped to [-1, 1) with 53 bits; the
  diagonal is real.  Order-independent and reproducible.
* X for configs 3-5: i.i.d. N(0,1) (complex: re and im each N(0,1)), torch generator on the
  chosen device; sampled columns are copied out BEFORE the call, so host and device never have
  to agree bit for bit.
* synthetic reflector stream (full-size configs where the host bulge chase would take many
  minutes): v[0] = 1, v[1:L] uniform in a range that gives tau in about [1.1, 1.6] like chase
  output, zero padded to nbw; tau = 2/||v||^2 (real) or (1 + e^{i theta})/||v||^2 (complex), which
  makes every H = I - tau v v^H exactly unitary up to rounding.  The per-slot lengths L are an
  argument (the caller gets them from whichever side it is testing).
"""
from __future__ import annotations

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        x = ((x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        x = ((x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        x = x ^ (x >> np.uint64(31))
    return x


def hash_uniform(seed: int, counter: np.ndarray, stream: int = 0) -> np.ndarray:
    """Uniform [-1, 1) doubles from (seed, counter, stream), 53 random bits each."""
    c = np.asarray(counter, dtype=np.uint64)
    with np.errstate(over="ignore"):
        key = _splitmix64(np.uint64(seed) * np.uint64(0xD1342543DE82EF95) + np.uint64(stream))
        h = _splitmix64(c ^ key)
    u = (h >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)  # [0,1)
    return 2.0 * u - 1.0


def band_matrix(N: int, nbw: int, seed: int, cplx: bool = False) -> np.ndarray:
    """Lower band storage with room for the chase's fill: shape (2*nbw+1, N), Fortran order,
    ab[i-j, j] = B[i, j] for 0 <= i-j <= nbw and i < N; everything else zero."""
    dt = np.complex128 if cplx else np.float64
    ab = np.zeros((2 * nbw + 1, N), dtype=dt, order="F")
    jj, dd = np.meshgrid(np.arange(N, dtype=np.uint64), np.arange(nbw + 1, dtype=np.uint64))
    ctr = jj * np.uint64(nbw + 1) + dd
    re = hash_uniform(seed, ctr, 0)
    if cplx:
        im = hash_uniform(seed, ctr, 1)
        im[0, :] = 0.0  # real diagonal
        vals = re + 1j * im
    else:
        vals = re
    inside = (jj.astype(np.int64) + dd.astype(np.int64)) < N
    ab[: nbw + 1, :] = np.where(inside, vals, 0.0)
    return ab


def dense_hermitian(N: int, seed: int, cplx: bool = False) -> np.ndarray:
    """Full N x N symmetric / Hermitian matrix (Fortran order, both triangles) with lower-triangle
    entries hashed uniform in [-1, 1) (complex: both parts) and a real diagonal -- the "randomly
    generated" matrices of PAPER.md:196 before the full -> band reduction."""
    ii, jj = np.meshgrid(np.arange(N, dtype=np.uint64), np.arange(N, dtype=np.uint64), indexing="ij")
    lo, hi = np.minimum(ii, jj), np.maximum(ii, jj)
    ctr = hi * np.uint64(max(N, 1)) + lo
    re = hash_uniform(seed, ctr, 0)
    if cplx:
        im = hash_uniform(seed, ctr, 1)
        im = np.where(ii > jj, im, np.where(ii < jj, -im, 0.0))
        a = re + 1j * im
    else:
        a = re
    return np.asfortranarray(a)


def structured_band_matrix(N: int, nbw: int, seed: int, cplx: bool, kind: str) -> np.ndarray:
    """Degenerate variants of ``band_matrix`` (same storage) that make the chase produce identity
    reflectors in the middle of a chain -- the inputs a KS-DFT matrix with decoupled blocks or a
    narrower true band gives:

    * ``blockdiag``: couplings across the cuts at rows 20, N//2 and N//2 + nbw + 3 are zero
    * ``narrow2`` / ``narrow1``: true semi-bandwidth nbw//2 / 1 (already tridiagonal)
    * ``zero``, ``identity``: the zero matrix, the unit matrix
    * ``zerotail``: the last N//3 columns have no off-diagonal entries
    * ``sparsecols``: every third column has no off-diagonal entries
    """
    ab = band_matrix(N, nbw, seed, cplx)
    jj, dd = np.meshgrid(np.arange(N), np.arange(2 * nbw + 1))
    ii = jj + dd
    if kind == "blockdiag":
        for cut in (20, N // 2, N // 2 + nbw + 3):
            ab[(ii >= cut) & (jj < cut)] = 0.0
    elif kind == "narrow2":
        ab[dd > nbw // 2] = 0.0
    elif kind == "narrow1":
        ab[dd > 1] = 0.0
    elif kind == "zero":
        ab[:] = 0.0
    elif kind == "identity":
        ab[:] = 0.0
        ab[0, :] = 1.0
    elif kind == "zerotail":
        ab[(dd > 0) & (jj >= N - N // 3)] = 0.0
    elif kind == "sparsecols":
        ab[(dd > 0) & (jj % 3 == 1)] = 0.0
    else:
        raise ValueError(kind)
    return ab


def sample_columns(nev: int, count: int, seed: int) -> np.ndarray:
    """``count`` distinct column indices of [0, nev), seeded, sorted."""
    rng = np.random.default_rng(seed)
    count = min(count, nev)
    return np.sort(rng.choice(nev, size=count, replace=False)).astype(np.int64)


def gaussian_block(N: int, ncols: int, seed: int, cplx: bool = False, device: str = "cpu"):
    """Column-major N x ncols block of i.i.d. N(0,1) (complex: re, im ~ N(0,1)) as a torch tensor
    whose storage is Fortran order: returned as the transposed view of a (ncols, N) tensor."""
    import torch

    gen = torch.Generator(device=device)
    gen.manual_seed(seed)
    if cplx:
        t = torch.randn((ncols, N, 2), generator=gen, device=device, dtype=torch.float64)
        t = torch.view_as_complex(t)
    else:
        t = torch.randn((ncols, N), generator=gen, device=device, dtype=torch.float64)
    return t.t()  # shape (N, ncols), element (r, j) at r + j*N


def synthetic_reflectors(lengths, nbw: int, seed: int, cplx: bool = False, device: str = "cpu"):
    """Unitary synthetic reflector stream for a given per-slot length array (int, shape (G,)).
    Returns torch tensors (hh_v (G, nbw), hh_tau (G,)).  Slots of length 1 are identity (tau 0)."""
    import torch

    L = torch.as_tensor(np.asarray(lengths), device=device).to(torch.int64)
    G = L.shape[0]
    gen = torch.Generator(device=device)
    gen.manual_seed(seed)
    shape = (G, nbw, 2) if cplx else (G, nbw)
    v = torch.rand(shape, generator=gen, device=device, dtype=torch.float64) * 2.0 - 1.0
    scale = 1.3 / torch.sqrt(L.clamp(min=1).to(torch.float64))
    v = v * (scale[:, None, None] if cplx else scale[:, None])
    r = torch.arange(nbw, device=device)[None, :]
    mask = (r < L[:, None]) & (r > 0)
    if cplx:
        v = torch.view_as_complex(torch.where(mask[:, :, None], v, torch.zeros_like(v)).contiguous())
    else:
        v = torch.where(mask, v, torch.zeros_like(v))
    v[:, 0] = 1.0
    nrm2 = (v.real ** 2 + v.imag ** 2).sum(dim=1) if cplx else (v * v).sum(dim=1)
    if cplx:
        theta = (torch.rand(G, generator=gen, device=device, dtype=torch.float64) - 0.5) * 1.5
        tau = (1.0 + torch.polar(torch.ones_like(theta), theta)) / nrm2
    else:
        tau = 2.0 / nrm2
    tau = torch.where(L > 1, tau, torch.zeros_like(tau))
    return v.contiguous(), tau.contiguous()


def synthetic_full_reflectors(N: int, nbw: int, seed: int, cplx: bool = False, device: str = "cpu", ldv=None):
    """Unitary synthetic reflector set in the layout of the band -> full back-transformation (Eq. 6e;
    include/elpa2_bt.h): returns torch tensors (hv, tau) with hv of shape (N, Nv) stored column-major
    (the transposed view of a (Nv, ldv) tensor), Nv = max(N - nbw - 1, 0).  Column j: zeros in rows
    < j + nbw, 1 at row j + nbw, uniform entries scaled by 1.3 / sqrt(L) below (L = N - nbw - j: the range
    a QR of a random panel gives); tau = 2 / ||v||^2 (real) or (1 + e^{i theta}) / ||v||^2 (complex), so that
    every H = I - tau v v^H is unitary up to rounding.  Stands in for the output of a full -> band
    reduction at sizes where the oracle's O(N^3) reduction is out of reach."""
    import torch

    Nv = max(N - nbw - 1, 0)
    ldv = ldv or (N + (N & 1))
    dt = torch.complex128 if cplx else torch.float64
    back = torch.zeros((max(Nv, 1), ldv), dtype=dt, device=device)
    tau = torch.zeros((Nv,), dtype=dt, device=device)
    gen = torch.Generator(device=device)
    gen.manual_seed(seed)
    rows = torch.arange(N, device=device)[None, :]
    step = 1024
    for j0 in range(0, Nv, step):
        j1 = min(j0 + step, Nv)
        head = (torch.arange(j0, j1, device=device) + nbw)[:, None]
        L = (N - head).to(torch.float64)
        shape = (j1 - j0, N, 2) if cplx else (j1 - j0, N)
        v = torch.rand(shape, generator=gen, device=device, dtype=torch.float64) * 2.0 - 1.0
        scale = 1.3 / torch.sqrt(L)
        if cplx:
            v = torch.view_as_complex((v * scale[:, :, None]).contiguous())
        else:
            v = v * scale
        v = torch.where(rows > head, v, torch.zeros_like(v))
        v = torch.where(rows == head, torch.ones_like(v), v)
        nrm2 = (v.real ** 2 + v.imag ** 2).sum(dim=1) if cplx else (v * v).sum(dim=1)
        if cplx:
            theta = (torch.rand(j1 - j0, generator=gen, device=device, dtype=torch.float64) - 0.5) * 1.5
            tau[j0:j1] = (1.0 + torch.polar(torch.ones_like(theta), theta)) / nrm2
        else:
            tau[j0:j1] = 2.0 / nrm2
        back[j0:j1, :N] = v
    return back[:Nv].t()[:N, :], tau
