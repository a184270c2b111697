"""ctypes binding of the CPU oracle (oracle/elpa2_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs
may import this package.  It imports nothing from ``paper_2002_10991_b200`` and shares no code with
the CUDA path.  Array conventions (all numpy, float64 / complex128, column-major = Fortran order):

* band matrix ``ab``: shape ``(2*nbw+1, N)`` Fortran order, ``ab[i-j, j] = B[i, j]`` for
  ``0 <= i-j <= 2*nbw`` (entries at distance > nbw are zero on input).
* reflectors: ``hh_v`` shape ``(G, nbw)`` C order (slot-major), ``hh_tau`` shape ``(G,)``.
* ``q``: shape ``(N, ncols)`` Fortran order (leading dimension ``ldq = q.strides[1] / itemsize``).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "elpa2_oracle.c")
_LIB = os.path.join(_HERE, "libelpa2_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP, no fast-math).  Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        i64, i32, vp = ctypes.c_int64, ctypes.c_int, ctypes.c_void_p
        _lib.orc_hh_blocks.argtypes = [i64, i32, i64]
        _lib.orc_hh_blocks.restype = i32
        _lib.orc_hh_offset.argtypes = [i64, i32, i64]
        _lib.orc_hh_offset.restype = i64
        _lib.orc_hh_count.argtypes = [i64, i32]
        _lib.orc_hh_count.restype = i64
        _lib.orc_hh_rows.argtypes = [i64, i32, i64, i32, vp, vp]
        _lib.orc_hh_rows.restype = i32
        _lib.orc_larfg_d.argtypes = [i32, vp, vp, vp, vp]
        _lib.orc_larfg_d.restype = None
        _lib.orc_larfg_z.argtypes = [i32, vp, vp, vp, vp]
        _lib.orc_larfg_z.restype = None
        for nm in ("orc_bulge_chase_d", "orc_bulge_chase_z"):
            getattr(_lib, nm).argtypes = [i64, i32, vp, vp, vp, vp, vp]
            getattr(_lib, nm).restype = i32
        _lib.orc_tridiag_ql.argtypes = [i64, vp, vp, vp]
        _lib.orc_tridiag_ql.restype = i32
        for nm in ("orc_back_transform_d", "orc_back_transform_z", "orc_back_transform_s", "orc_back_transform_c"):
            getattr(_lib, nm).argtypes = [i64, i32, i64, vp, vp, vp, i64]
            getattr(_lib, nm).restype = None
        for nm in ("orc_full_to_band_d", "orc_full_to_band_z"):
            getattr(_lib, nm).argtypes = [i64, i32, vp, i64, vp, i64, vp]
            getattr(_lib, nm).restype = i32
        for nm in ("orc_band_to_full_back_d", "orc_band_to_full_back_z"):
            getattr(_lib, nm).argtypes = [i64, i32, i64, vp, i64, vp, vp, i64]
            getattr(_lib, nm).restype = None
        _lib.orc_num_threads.argtypes = []
        _lib.orc_num_threads.restype = i32
    return _lib


def _p(a: np.ndarray) -> int:
    return a.ctypes.data


def hh_blocks(N: int, nbw: int, s: int) -> int:
    return lib().orc_hh_blocks(N, nbw, s)


def hh_offset(N: int, nbw: int, s: int) -> int:
    return lib().orc_hh_offset(N, nbw, s)


def hh_count(N: int, nbw: int) -> int:
    return lib().orc_hh_count(N, nbw)


def hh_rows(N: int, nbw: int, s: int, k: int) -> tuple[int, int, int]:
    """(r0, r1, L) of reflector (s, k)."""
    r0, r1 = ctypes.c_int64(), ctypes.c_int64()
    L = lib().orc_hh_rows(N, nbw, s, k, ctypes.addressof(r0), ctypes.addressof(r1))
    return r0.value, r1.value, L


def larfg(x: np.ndarray):
    """(v, tau, beta) with H^H x = beta e1, H = I - tau v v^H, v[0] = 1."""
    cplx = np.iscomplexobj(x)
    x = np.ascontiguousarray(x, dtype=np.complex128 if cplx else np.float64)
    v = np.empty_like(x)
    tau = np.zeros(1, dtype=x.dtype)
    beta = np.zeros(1, dtype=np.float64)
    fn = lib().orc_larfg_z if cplx else lib().orc_larfg_d
    fn(x.shape[0], _p(x), _p(v), _p(tau), _p(beta))
    return v, tau[0], float(beta[0])


def bulge_chase(ab: np.ndarray, nbw: int):
    """Reduce the band matrix to tridiagonal form.  Returns (hh_v, hh_tau, d, e); ``ab`` is
    overwritten with T."""
    cplx = np.iscomplexobj(ab)
    dt = np.complex128 if cplx else np.float64
    assert ab.dtype == dt and ab.flags.f_contiguous and ab.shape[0] == 2 * nbw + 1
    N = ab.shape[1]
    G = hh_count(N, nbw)
    hh_v = np.zeros((G, nbw), dtype=dt)
    hh_tau = np.zeros(G, dtype=dt)
    d = np.zeros(N)
    e = np.zeros(max(N - 1, 0))
    fn = lib().orc_bulge_chase_z if cplx else lib().orc_bulge_chase_d
    rc = fn(N, nbw, _p(ab), _p(hh_v), _p(hh_tau), _p(d), _p(e))
    if rc != 0:
        raise RuntimeError(f"orc_bulge_chase failed: {rc}")
    return hh_v, hh_tau, d, e


def tridiag_ql(d: np.ndarray, e: np.ndarray):
    """Eigenpairs of the symmetric tridiagonal (d, e).  Returns (lam ascending, X columns)."""
    N = d.shape[0]
    lam = np.array(d, dtype=np.float64, copy=True)
    ee = np.array(e, dtype=np.float64, copy=True)
    X = np.zeros((N, N), dtype=np.float64, order="F")
    rc = lib().orc_tridiag_ql(N, _p(lam), _p(ee), _p(X))
    if rc != 0:
        raise RuntimeError(f"orc_tridiag_ql did not converge: {rc}")
    return lam, X


def back_transform(N: int, nbw: int, hh_v: np.ndarray, hh_tau: np.ndarray, q: np.ndarray) -> None:
    """q <- H(0,0) ... H(N-2,0) q in place (Eq. 6d), q Fortran-ordered N x ncols."""
    cplx = np.iscomplexobj(q)
    dt = q.dtype
    assert dt in (np.float64, np.complex128, np.float32, np.complex64)      # FP32: SURVEY 8(f) NEXT-4, reading R16
    assert hh_v.dtype == dt and hh_tau.dtype == dt
    assert q.ndim == 2 and q.shape[0] == N and q.strides[0] == q.itemsize
    assert hh_v.flags.c_contiguous and hh_tau.flags.c_contiguous
    assert hh_v.shape == (hh_count(N, nbw), nbw)
    ncols = q.shape[1]
    ldq = q.strides[1] // q.itemsize if ncols > 1 else max(N, 1)
    fn = {np.dtype(np.float64): lib().orc_back_transform_d, np.dtype(np.complex128): lib().orc_back_transform_z,
          np.dtype(np.float32): lib().orc_back_transform_s, np.dtype(np.complex64): lib().orc_back_transform_c}[np.dtype(dt)]
    fn(N, nbw, ncols, _p(hh_v), _p(hh_tau), _p(q), ldq)


def full_to_band(a: np.ndarray, nbw: int):
    """Eq. 6a (reading R15): reduce the full Hermitian matrix ``a`` (N x N, Fortran order, both
    triangles) to a band of semi-bandwidth nbw, in place.  Returns (hv, tau): hv is N x Nv Fortran
    order (column j = v_j at rows j+nbw.., unit head stored, zeros above), tau has Nv entries,
    Nv = max(N - nbw - 1, 0)."""
    cplx = np.iscomplexobj(a)
    dt = np.complex128 if cplx else np.float64
    assert a.dtype == dt and a.flags.f_contiguous and a.ndim == 2 and a.shape[0] == a.shape[1]
    N = a.shape[0]
    Nv = max(N - nbw - 1, 0)
    hv = np.zeros((N, max(Nv, 1)), dtype=dt, order="F")[:, :Nv]
    tau = np.zeros(Nv, dtype=dt)
    fn = lib().orc_full_to_band_z if cplx else lib().orc_full_to_band_d
    rc = fn(N, nbw, _p(a), max(N, 1), _p(hv), max(N, 1), _p(tau))
    if rc != 0:
        raise RuntimeError(f"orc_full_to_band failed: {rc}")
    return hv, tau


def band_to_full_back(N: int, nbw: int, hv: np.ndarray, tau: np.ndarray, q: np.ndarray) -> None:
    """Eq. 6e: q <- H_0 H_1 ... H_{Nv-1} q in place (q Fortran-ordered N x ncols)."""
    cplx = np.iscomplexobj(q)
    dt = np.complex128 if cplx else np.float64
    assert q.dtype == dt and hv.dtype == dt and tau.dtype == dt
    assert q.ndim == 2 and q.shape[0] == N and q.strides[0] == q.itemsize
    Nv = max(N - nbw - 1, 0)
    assert hv.shape == (N, Nv) and tau.shape == (Nv,) and tau.flags.c_contiguous
    if Nv == 0 or q.shape[1] == 0:
        return
    assert hv.strides[0] == hv.itemsize
    ldv = hv.strides[1] // hv.itemsize if Nv > 1 else max(N, 1)
    ncols = q.shape[1]
    ldq = q.strides[1] // q.itemsize if ncols > 1 else max(N, 1)
    fn = lib().orc_band_to_full_back_z if cplx else lib().orc_band_to_full_back_d
    fn(N, nbw, ncols, _p(hv), ldv, _p(tau), _p(q), ldq)


def num_threads() -> int:
    return lib().orc_num_threads()
