"""Helpers for the -m gpu parity tests: run the CUDA path through the C ABI on seeded inputs and
compare with the oracle.  Test-side only."""
from __future__ import annotations

import numpy as np


def to_device_colmajor(x_np):
    """numpy (N, ncols) -> CUDA tensor of the same shape stored column-major (stride(0) == 1)."""
    import torch

    t = torch.from_numpy(np.ascontiguousarray(x_np.T)).cuda()
    return t.t()


def device_q(N, nev, ldq, dtype):
    """Uninitialised column-major (N, nev) view with leading dimension ldq, plus its backing."""
    import torch

    back = torch.full((nev, ldq), 7.25, dtype=dtype, device="cuda")
    return back, back.t()[:N, :]


def run_gpu(N, nbw, hh_v, hh_tau, x_np, ldq=None, variant=0):
    """Apply the CUDA back-transformation to a copy of x_np (N, nev); returns numpy result and the
    padding rows (to check they are untouched)."""
    import torch

    from paper_2002_10991_b200 import binding

    nev = x_np.shape[1]
    ldq = ldq or max(N, 1)
    dtype = torch.complex128 if np.iscomplexobj(x_np) else torch.float64
    back, q = device_q(N, nev, ldq, dtype)
    if N > 0 and nev > 0:
        q.copy_(torch.from_numpy(np.ascontiguousarray(x_np)).cuda())
    dv = torch.from_numpy(np.ascontiguousarray(hh_v)).cuda()
    dt = torch.from_numpy(np.ascontiguousarray(hh_tau)).cuda()
    if dv.numel() == 0:
        dv = torch.zeros((1, nbw), dtype=dtype, device="cuda")
        dt = torch.zeros((1,), dtype=dtype, device="cuda")
    old = binding.set_variant(variant)
    try:
        binding.trans_ev_tridi_to_band(N, nbw, dv, dt, q)
        torch.cuda.synchronize()
    finally:
        binding.set_variant(old)
    res = q.cpu().numpy()
    pad = back.t()[N:, :].cpu().numpy()
    return res, pad


def oracle_apply(N, nbw, hh_v, hh_tau, x_np):
    import oracle

    y = np.array(x_np, order="F", copy=True)
    if N >= 2 and y.shape[1] > 0:
        oracle.back_transform(N, nbw, hh_v, hh_tau, y)
    return y
