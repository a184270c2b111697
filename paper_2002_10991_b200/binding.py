"""Thin ctypes binding of the C-ABI library declared in ``include/elpa2_bt.h``.

Argument marshalling only: every step of the path runs in the CUDA kernels behind the C ABI.
torch is used for device memory and streams, nothing else.  There is no CPU fallback: if the
library is missing the import of any entry point raises, loudly.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libelpa2_bt.so")
SOURCES = [os.path.join(_HERE, "csrc", f) for f in ("elpa2_bt.cu", "fp64_probe.cu")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]

_lib = None

EXPORTS = (
    "elpa2_trans_ev_tridi_to_band_d", "elpa2_trans_ev_tridi_to_band_z",
    "elpa2_trans_ev_tridi_to_band_host", "elpa2_hh_count", "elpa2_hh_offset", "elpa2_hh_blocks",
    "elpa2_bt_last_launch_count", "elpa2_bt_set_variant", "elpa2_bt_version", "elpa2_bt_probe_fp64",
    "elpa2_bulge_chase_d", "elpa2_bulge_chase_z", "elpa2_bt_plan", "elpa2_bt_release_scratch",
    "elpa2_hh_lengths", "elpa2_trans_ev_band_to_full_d", "elpa2_trans_ev_band_to_full_z",
    "elpa2_trans_ev_band_to_full_host", "elpa2_bt_set_chain_parallel",
    "elpa2_trans_ev_tridi_to_band_s", "elpa2_trans_ev_tridi_to_band_c", "elpa2_trans_ev_tridi_to_band_host32",
    "elpa2_trans_ev_tridi_to_band_rows_d", "elpa2_trans_ev_tridi_to_band_rows_z",
    "elpa2_trans_ev_band_to_full_noalloc_d", "elpa2_noalloc_scratch_bytes",
)


def build(force: bool = False) -> str:
    """Compile the CUDA library in-tree with nvcc for sm_100a (no GPU needed)."""
    import subprocess

    deps = SOURCES + [os.path.join(_HERE, "csrc", f) for f in os.listdir(os.path.join(_HERE, "csrc"))]
    newest = max(os.path.getmtime(p) for p in deps)
    if force or not os.path.exists(LIB_PATH) or os.path.getmtime(LIB_PATH) < newest:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        subprocess.run([nvcc, *NVCC_FLAGS, "-o", LIB_PATH, *SOURCES], check=True)
    return LIB_PATH


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        i64, i32, vp = ctypes.c_int64, ctypes.c_int, ctypes.c_void_p
        for nm in ("elpa2_trans_ev_tridi_to_band_d", "elpa2_trans_ev_tridi_to_band_z",
                   "elpa2_trans_ev_tridi_to_band_s", "elpa2_trans_ev_tridi_to_band_c"):
            getattr(L, nm).argtypes = [i64, i32, i64, vp, vp, vp, i64, vp]
            getattr(L, nm).restype = i32
        for nm in ("elpa2_trans_ev_tridi_to_band_rows_d", "elpa2_trans_ev_tridi_to_band_rows_z"):
            getattr(L, nm).argtypes = [i64, i32, i64, vp, vp, vp, i64, i64, i64, i64, i64, i64, vp]
            getattr(L, nm).restype = i32
        L.elpa2_trans_ev_tridi_to_band_host32.argtypes = [i32, i64, i32, i64, vp, vp, vp, i64]
        L.elpa2_trans_ev_tridi_to_band_host32.restype = i32
        L.elpa2_trans_ev_tridi_to_band_host.argtypes = [i32, i64, i32, i64, vp, vp, vp, i64]
        L.elpa2_trans_ev_tridi_to_band_host.restype = i32
        for nm in ("elpa2_bulge_chase_d", "elpa2_bulge_chase_z"):
            getattr(L, nm).argtypes = [i64, i32, vp, vp, vp, vp, vp, vp]
            getattr(L, nm).restype = i32
        L.elpa2_noalloc_scratch_bytes.argtypes = []
        L.elpa2_noalloc_scratch_bytes.restype = i64
        for nm in ("elpa2_trans_ev_band_to_full_d", "elpa2_trans_ev_band_to_full_z", "elpa2_trans_ev_band_to_full_noalloc_d"):
            getattr(L, nm).argtypes = [i64, i32, i64, vp, i64, vp, vp, i64, vp]
            getattr(L, nm).restype = i32
        L.elpa2_trans_ev_band_to_full_host.argtypes = [i32, i64, i32, i64, vp, i64, vp, vp, i64]
        L.elpa2_trans_ev_band_to_full_host.restype = i32
        L.elpa2_bt_release_scratch.argtypes = []
        L.elpa2_bt_release_scratch.restype = i32
        L.elpa2_bt_plan.argtypes = [i32, i64, i32, i64, i32, ctypes.POINTER(i64)]
        L.elpa2_bt_plan.restype = i32
        L.elpa2_hh_count.argtypes = [i64, i32]
        L.elpa2_hh_count.restype = i64
        L.elpa2_hh_offset.argtypes = [i64, i32, i64]
        L.elpa2_hh_offset.restype = i64
        L.elpa2_hh_blocks.argtypes = [i64, i32, i64]
        L.elpa2_hh_blocks.restype = i32
        L.elpa2_hh_lengths.argtypes = [i64, i32, vp, i64]
        L.elpa2_hh_lengths.restype = i64
        L.elpa2_bt_last_launch_count.argtypes = []
        L.elpa2_bt_last_launch_count.restype = i32
        L.elpa2_bt_set_variant.argtypes = [i32]
        L.elpa2_bt_set_variant.restype = i32
        L.elpa2_bt_set_chain_parallel.argtypes = [i32]
        L.elpa2_bt_set_chain_parallel.restype = i32
        L.elpa2_bt_version.argtypes = []
        L.elpa2_bt_version.restype = ctypes.c_char_p
        L.elpa2_bt_probe_fp64.argtypes = [i32, i32, i32, ctypes.POINTER(ctypes.c_double)]
        L.elpa2_bt_probe_fp64.restype = i32
        _lib = L
    return _lib


class Elpa2BtError(RuntimeError):
    def __init__(self, rc: int):
        self.rc = rc
        what = f"argument {-rc} invalid" if rc < 0 else f"cudaError_t {rc}"
        if rc == -20:
            what = "the problem needs more scratch than the static no-alloc array holds (elpa2_noalloc_scratch_bytes)"
        super().__init__(f"elpa2_trans_ev_tridi_to_band failed: {what}")


def hh_count(N: int, nbw: int) -> int:
    return lib().elpa2_hh_count(N, nbw)


def hh_offset(N: int, nbw: int, s: int) -> int:
    return lib().elpa2_hh_offset(N, nbw, s)


def hh_blocks(N: int, nbw: int, s: int) -> int:
    return lib().elpa2_hh_blocks(N, nbw, s)


def hh_lengths(N: int, nbw: int):
    """Length L of every reflector slot, in slot order (int32 numpy array of G entries), from the
    library's ``elpa2_hh_lengths``."""
    import numpy as np

    G = max(int(lib().elpa2_hh_lengths(N, nbw, None, 0)), 0)
    out = np.zeros(G, dtype=np.int32)
    if G:
        lib().elpa2_hh_lengths(N, nbw, out.ctypes.data, G)
    return out


def plan(cplx: bool, N: int, nbw: int, nev: int, n_sm: int = 148) -> dict:
    """Launch plan of the default variant (host arithmetic only; works without a GPU)."""
    out = (ctypes.c_int64 * 6)()
    rc = lib().elpa2_bt_plan(int(cplx), N, nbw, nev, n_sm, out)
    if rc != 0:
        raise Elpa2BtError(rc)
    keys = ("grid", "warps_per_cta", "P", "slabs", "slabs_per_cta_max", "scratch_bytes")
    return dict(zip(keys, (int(x) for x in out)))


def release_scratch() -> None:
    """Free the library's cached device memory (host-entry buffers, unused scratch-pool blocks)."""
    rc = lib().elpa2_bt_release_scratch()
    if rc != 0:
        raise Elpa2BtError(rc)


def version() -> str:
    return lib().elpa2_bt_version().decode()


def set_variant(variant: int) -> int:
    return lib().elpa2_bt_set_variant(variant)


def set_chain_parallel(P: int) -> int:
    """Testing aid: force P warps per slab (0 = planned); see include/elpa2_bt.h."""
    return lib().elpa2_bt_set_chain_parallel(P)


def last_launch_count() -> int:
    return lib().elpa2_bt_last_launch_count()


def probe_fp64(kind: int, iters: int = 4096, reps: int = 20) -> float:
    out = ctypes.c_double(0.0)
    rc = lib().elpa2_bt_probe_fp64(kind, iters, reps, ctypes.byref(out))
    if rc != 0:
        raise Elpa2BtError(rc)
    return out.value


def _stream_ptr(stream) -> int:
    if stream is None:
        import torch

        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


def trans_ev_tridi_to_band_raw(cplx: bool, N: int, nbw: int, nev: int, hh_v_ptr: int, hh_tau_ptr: int,
                               q_ptr: int, ldq: int, stream_ptr: int, single: bool = False) -> int:
    """The C call itself, on raw device addresses; returns the C return code.  ``single``: the FP32 calls."""
    if single:
        fn = lib().elpa2_trans_ev_tridi_to_band_c if cplx else lib().elpa2_trans_ev_tridi_to_band_s
    else:
        fn = lib().elpa2_trans_ev_tridi_to_band_z if cplx else lib().elpa2_trans_ev_tridi_to_band_d
    return fn(N, nbw, nev, hh_v_ptr, hh_tau_ptr, q_ptr, ldq, stream_ptr)


def trans_ev_tridi_to_band(N: int, nbw: int, hh_v, hh_tau, q, stream=None) -> None:
    """q <- Q2 q in place (Eq. 6d).  ``q``: CUDA tensor of shape (N, nev), float64 or complex128 (or
    float32 / complex64: the FP32 calls), stored column-major (``q.stride(0) == 1``; ldq = ``q.stride(1)``).  ``hh_v`` (G, nbw) and
    ``hh_tau`` (G,) contiguous CUDA tensors of the same dtype, layout per include/elpa2_bt.h."""
    import torch

    if not (q.is_cuda and hh_v.is_cuda and hh_tau.is_cuda):
        raise ValueError("device tensors required (use trans_ev_tridi_to_band_host for numpy arrays)")
    cplx = q.dtype in (torch.complex128, torch.complex64)
    single = q.dtype in (torch.float32, torch.complex64)
    if (q.dtype not in (torch.float64, torch.complex128, torch.float32, torch.complex64) or hh_v.dtype != q.dtype
            or hh_tau.dtype != q.dtype):
        raise ValueError("one of float64, complex128, float32, complex64 throughout")
    if q.dim() != 2 or q.shape[0] != N or (q.shape[0] > 1 and q.stride(0) != 1):
        raise ValueError("q must be (N, nev) column-major")
    nev = q.shape[1]
    ldq = q.stride(1) if nev > 1 else max(N, 1)
    if not (hh_v.is_contiguous() and hh_tau.is_contiguous()):
        raise ValueError("hh_v / hh_tau must be contiguous")
    G = hh_count(N, nbw)
    if G > 0 and nev > 0 and (tuple(hh_v.shape) != (G, nbw) or tuple(hh_tau.shape) != (G,)):
        raise ValueError(f"hh_v must be ({G}, {nbw}) and hh_tau ({G},) for N = {N}, nbw = {nbw}")
    if not (hh_v.device == q.device and hh_tau.device == q.device):
        raise ValueError("hh_v, hh_tau and q must live on the same device")
    if torch.cuda.current_device() != q.device.index:
        raise ValueError("q's device must be the current CUDA device")
    rc = trans_ev_tridi_to_band_raw(cplx, N, nbw, nev, hh_v.data_ptr(), hh_tau.data_ptr(), q.data_ptr(),
                                    ldq, _stream_ptr(stream), single)
    if rc != 0:
        raise Elpa2BtError(rc)


def trans_ev_tridi_to_band_rows(N: int, nbw: int, hh_v, hh_tau, q_local, row0: int, nown: int, kb: int, ke: int,
                                stream=None) -> None:
    """Row-block form (include/elpa2_bt.h): ``q_local`` is a column-major CUDA tensor of
    shape (nloc, nev) holding the rows [row0, row0 + nloc) -- the ``nown`` owned rows and the halo rows
    below; applies the owned blocks of the chains [kb, ke)."""
    import torch

    if not (q_local.is_cuda and hh_v.is_cuda and hh_tau.is_cuda):
        raise ValueError("device tensors required")
    cplx = q_local.dtype == torch.complex128
    if q_local.dtype not in (torch.float64, torch.complex128) or hh_v.dtype != q_local.dtype or hh_tau.dtype != q_local.dtype:
        raise ValueError("float64 or complex128 throughout")
    if q_local.dim() != 2 or (q_local.shape[0] > 1 and q_local.stride(0) != 1):
        raise ValueError("q_local must be (nloc, nev) column-major")
    nloc, nev = q_local.shape
    ldq = q_local.stride(1) if nev > 1 else max(nloc, 1)
    G = hh_count(N, nbw)
    if not (hh_v.is_contiguous() and hh_tau.is_contiguous()) or tuple(hh_v.shape) != (G, nbw) or tuple(hh_tau.shape) != (G,):
        raise ValueError(f"hh_v must be contiguous ({G}, {nbw}) and hh_tau ({G},)")
    if not (hh_v.device == q_local.device and hh_tau.device == q_local.device
            and torch.cuda.current_device() == q_local.device.index):
        raise ValueError("hh_v, hh_tau and q_local must live on the current CUDA device")
    fn = lib().elpa2_trans_ev_tridi_to_band_rows_z if cplx else lib().elpa2_trans_ev_tridi_to_band_rows_d
    rc = fn(N, nbw, nev, hh_v.data_ptr(), hh_tau.data_ptr(), q_local.data_ptr(), ldq, row0, nown, nloc, kb, ke,
            _stream_ptr(stream))
    if rc != 0:
        raise Elpa2BtError(rc)


def noalloc_scratch_bytes() -> int:
    return int(lib().elpa2_noalloc_scratch_bytes())


def trans_ev_band_to_full_noalloc(N: int, nbw: int, hv, tau, q, stream=None) -> None:
    """``elpa2_trans_ev_band_to_full_noalloc_d``: Eq. 6e, real FP64, without any allocation -- the scratch is a
    static 16 MiB device array inside the library (N - nbw - 1 <= 32768, else Elpa2BtError with rc -20).  All
    calls share that array: calls that overlap on the GPU race.  Arguments as ``trans_ev_band_to_full``."""
    import torch

    if not (q.is_cuda and hv.is_cuda and tau.is_cuda):
        raise ValueError("device tensors required")
    if q.dtype != torch.float64 or hv.dtype != q.dtype or tau.dtype != q.dtype:
        raise ValueError("float64 throughout")
    Nv = max(N - nbw - 1, 0)
    if q.dim() != 2 or q.shape[0] != N or (N > 1 and q.stride(0) != 1):
        raise ValueError("q must be (N, nev) column-major")
    nev = q.shape[1]
    ldq = q.stride(1) if nev > 1 else max(N, 1)
    if Nv > 0 and (tuple(hv.shape) != (N, Nv) or hv.stride(0) != 1 or tuple(tau.shape) != (Nv,) or not tau.is_contiguous()):
        raise ValueError(f"hv must be ({N}, {Nv}) column-major and tau ({Nv},)")
    ldv = hv.stride(1) if Nv > 1 else max(N + (N & 1), 2)
    if not (hv.device == q.device and tau.device == q.device and torch.cuda.current_device() == q.device.index):
        raise ValueError("hv, tau and q must live on the current CUDA device")
    rc = lib().elpa2_trans_ev_band_to_full_noalloc_d(N, nbw, nev, hv.data_ptr(), ldv, tau.data_ptr(), q.data_ptr(), ldq,
                                                     _stream_ptr(stream))
    if rc != 0:
        raise Elpa2BtError(rc)


def trans_ev_band_to_full(N: int, nbw: int, hv, tau, q, stream=None) -> None:
    """q <- P* q in place (Eq. 6e).  ``hv``: CUDA tensor of shape (N, Nv) stored column-major
    (``hv.stride(0) == 1``, ldv = ``hv.stride(1)``), Nv = max(N - nbw - 1, 0); ``tau`` (Nv,); ``q`` (N, nev)
    column-major.  Layout per include/elpa2_bt.h."""
    import torch

    if not (q.is_cuda and hv.is_cuda and tau.is_cuda):
        raise ValueError("device tensors required")
    if q.dtype not in (torch.float64, torch.complex128) or hv.dtype != q.dtype or tau.dtype != q.dtype:
        raise ValueError("float64 or complex128 throughout")
    cplx = q.dtype == torch.complex128
    Nv = max(N - nbw - 1, 0)
    if q.dim() != 2 or q.shape[0] != N or (N > 1 and q.stride(0) != 1):
        raise ValueError("q must be (N, nev) column-major")
    nev = q.shape[1]
    ldq = q.stride(1) if nev > 1 else max(N, 1)
    if Nv > 0 and (tuple(hv.shape) != (N, Nv) or hv.stride(0) != 1 or tuple(tau.shape) != (Nv,) or not tau.is_contiguous()):
        raise ValueError(f"hv must be ({N}, {Nv}) column-major and tau ({Nv},)")
    ldv = hv.stride(1) if Nv > 1 else max(N + (N & 1), 2)
    if not (hv.device == q.device and tau.device == q.device and torch.cuda.current_device() == q.device.index):
        raise ValueError("hv, tau and q must live on the current CUDA device")
    fn = lib().elpa2_trans_ev_band_to_full_z if cplx else lib().elpa2_trans_ev_band_to_full_d
    rc = fn(N, nbw, nev, hv.data_ptr(), ldv, tau.data_ptr(), q.data_ptr(), ldq, _stream_ptr(stream))
    if rc != 0:
        raise Elpa2BtError(rc)


def trans_ev_band_to_full_host(N: int, nbw: int, hv, tau, q) -> None:
    """Eq. 6e with HOST numpy arrays: ``hv`` Fortran-ordered (ldv, Nv) block whose first N rows are the
    reflectors (ldv = hv.shape[0] even), ``tau`` (Nv,), ``q`` Fortran-ordered (N, nev), updated in place."""
    import numpy as np

    if q.dtype not in (np.float64, np.complex128) or hv.dtype != q.dtype or tau.dtype != q.dtype:
        raise ValueError("float64 or complex128 throughout")
    Nv = max(N - nbw - 1, 0)
    if q.ndim != 2 or q.shape[0] != N or not q.flags.f_contiguous:
        raise ValueError("q must be Fortran-contiguous (N, nev)")
    if Nv > 0 and (hv.ndim != 2 or hv.shape[1] != Nv or hv.shape[0] < N or not hv.flags.f_contiguous):
        raise ValueError("hv must be Fortran-contiguous (ldv >= N, Nv)")
    rc = lib().elpa2_trans_ev_band_to_full_host(int(np.iscomplexobj(q)), N, nbw, q.shape[1], hv.ctypes.data, hv.shape[0], tau.ctypes.data,
                                                q.ctypes.data, max(N, 1))
    if rc != 0:
        raise Elpa2BtError(rc)


def bulge_chase(N: int, nbw: int, ab, stream=None):
    """Band -> tridiagonal on the device (Eq. 6b).  ``ab``: CUDA float64 / complex128 tensor of shape
    (N, 2*nbw+1), row j = column j of the lower band storage (ab[j, i-j] = B[i, j]), overwritten
    with T.  Entries ab[:, nbw+1:] are room for the fill and MUST be zero on entry (not checked).  Returns CUDA tensors (hh_v (G, nbw), hh_tau (G,), d (N,), e (N-1,)); d, e are real."""
    import torch

    if (not ab.is_cuda or ab.dtype not in (torch.float64, torch.complex128) or not ab.is_contiguous()
            or tuple(ab.shape) != (N, 2 * nbw + 1)):
        raise ValueError("ab must be a contiguous CUDA float64/complex128 tensor of shape (N, 2*nbw+1)")
    G = hh_count(N, nbw)
    hh_v = torch.empty((G, nbw), dtype=ab.dtype, device=ab.device)
    hh_tau = torch.empty((G,), dtype=ab.dtype, device=ab.device)
    d = torch.empty((N,), dtype=torch.float64, device=ab.device)
    e = torch.empty((max(N - 1, 0),), dtype=torch.float64, device=ab.device)
    fn = lib().elpa2_bulge_chase_z if ab.dtype == torch.complex128 else lib().elpa2_bulge_chase_d
    rc = fn(N, nbw, ab.data_ptr(), hh_v.data_ptr(), hh_tau.data_ptr(), d.data_ptr(), e.data_ptr(),
            _stream_ptr(stream))
    if rc != 0:
        raise Elpa2BtError(rc)
    return hh_v, hh_tau, d, e


def trans_ev_tridi_to_band_host(N: int, nbw: int, hh_v, hh_tau, q) -> None:
    """Same with HOST numpy arrays (q Fortran-ordered (N, nev), updated in place); the library
    copies to the device, runs the kernel and copies back (synchronous)."""
    import numpy as np

    cplx = np.iscomplexobj(q)
    dt = q.dtype
    if dt not in (np.float64, np.complex128, np.float32, np.complex64) or hh_v.dtype != dt or hh_tau.dtype != dt:
        raise ValueError("one of float64, complex128, float32, complex64 throughout")
    single = dt in (np.float32, np.complex64)
    if q.ndim != 2 or q.shape[0] != N or (N > 1 and q.strides[0] != q.itemsize):
        raise ValueError("q must be (N, nev) column-major")
    nev = q.shape[1]
    ldq = q.strides[1] // q.itemsize if nev > 1 else max(N, 1)
    if nev > 1 and not q.flags.f_contiguous:
        raise ValueError("host q must be Fortran-contiguous (ldq == N)")
    fn = lib().elpa2_trans_ev_tridi_to_band_host32 if single else lib().elpa2_trans_ev_tridi_to_band_host
    rc = fn(int(cplx), N, nbw, nev, hh_v.ctypes.data, hh_tau.ctypes.data, q.ctypes.data, ldq)
    if rc != 0:
        raise Elpa2BtError(rc)
