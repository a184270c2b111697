"""SURVEY.md 8(f) NEXT-1 (first version, real FP64): the GPU bulge chase against the oracle's chase,
against numpy's dense eigenvalues, and end to end with the GPU back-transform.

The tridiagonal form is unique (implicit Q) but ill-conditioned, so two correctly rounded chases
with different summation orders drift apart entry by entry (6e-10 at N = 1000 when the kernel used
FMAs and a tree reduction).  The kernel therefore follows SURVEY O3 operation by operation with
every product and sum rounded separately, and the comparison is BIT-EXACT at every size (the oracle
is built by gcc -O2 for baseline x86-64: no FMA contraction, no re-association)."""
import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import synth_inputs as si
from helpers import dense_from_band

pytestmark = pytest.mark.gpu


def _gpu_chase(ab, N, nbw):
    import torch

    from paper_2002_10991_b200 import binding

    dab = torch.from_numpy(np.ascontiguousarray(ab.T)).cuda()     # (N, 2 nbw + 1): row j = column j
    hv, ht, d, e = binding.bulge_chase(N, nbw, dab)
    torch.cuda.synchronize()
    assert binding.last_launch_count() >= 1
    return hv, ht, d, e, dab


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw", [(2, 32), (3, 32), (33, 32), (34, 32), (100, 32), (65, 64), (200, 64), (515, 64),
                                   (300, 128), (1000, 32), (2500, 64)])
def test_chase_matches_oracle(N, nbw, cplx):
    ab = si.band_matrix(N, nbw, 500 + N, cplx)
    ab_o = ab.copy(order="F")
    hv_o, ht_o, d_o, e_o = orc.bulge_chase(ab_o, nbw)
    hv, ht, d, e, dab = _gpu_chase(ab, N, nbw)
    scale = np.abs(ab).max()
    assert np.array_equal(ht.cpu().numpy(), ht_o)
    assert np.array_equal(hv.cpu().numpy(), hv_o)
    assert np.array_equal(d.cpu().numpy(), d_o)
    assert np.array_equal(e.cpu().numpy(), e_o)
    # layout conventions: v[0] = 1 stored, zero padding beyond the reflector's length
    hvn = hv.cpu().numpy()
    assert np.all(hvn[:, 0] == 1.0)
    from paper_2002_10991_b200 import binding

    Ls = binding.hh_lengths(N, nbw)
    mask = np.arange(nbw)[None, :] >= Ls[:, None]
    assert np.all(hvn[mask] == 0.0)
    # the band storage now holds T: nothing outside the tridiagonal
    t = dab.cpu().numpy()
    assert np.abs(t[:, 2:]).max(initial=0.0) <= 1e-12 * scale * max(N, 1)


DEGENERATE = ("blockdiag", "narrow2", "narrow1", "zero", "identity", "zerotail", "sparsecols")


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("nbw,N", [(32, 300), (64, 450), (128, 700)])
@pytest.mark.parametrize("kind", DEGENERATE)
def test_chase_degenerate_inputs_bit_exact(kind, nbw, N, cplx):
    """Identity reflectors in the middle of a chain (decoupled blocks, a narrower true band, zero /
    unit matrix, empty column tails): the steps `tau == 0` after a kept block, `ident` slots and L == 1
    slots inside a chain.  Bit for bit against the oracle, three runs each (the persistent schedule
    carries hand-written cross-CTA flags; a stale corner would show up as a run-to-run difference)."""
    ab = si.structured_band_matrix(N, nbw, 900 + N, cplx, kind)
    hv_o, ht_o, d_o, e_o = orc.bulge_chase(ab.copy(order="F"), nbw)
    for rep in range(3):
        hv, ht, d, e, dab = _gpu_chase(ab, N, nbw)
        assert np.array_equal(ht.cpu().numpy(), ht_o), (kind, rep)
        assert np.array_equal(hv.cpu().numpy(), hv_o), (kind, rep)
        assert np.array_equal(d.cpu().numpy(), d_o), (kind, rep)
        assert np.array_equal(e.cpu().numpy(), e_o), (kind, rep)
        t = dab.cpu().numpy()
        assert np.abs(t[:, 2:]).max(initial=0.0) <= 1e-12 * max(1.0, np.abs(ab).max()) * N


def test_wavefront_schedule_is_bit_identical():
    """ELPA2_BC_WAVEFRONT=1 (one launch per wavefront 3s + k) in a fresh process: same bits as the oracle."""
    import os
    import subprocess
    import sys

    code = (
        "import numpy as np, torch, oracle as orc\n"
        "from paper_2002_10991_b200 import binding, synth_inputs as si\n"
        "for cplx, N, nbw in ((False, 300, 64), (True, 200, 32), (False, 300, 128)):\n"
        "    ab = si.band_matrix(N, nbw, 9, cplx); ab_o = ab.copy(order='F')\n"
        "    hv_o, ht_o, d_o, e_o = orc.bulge_chase(ab_o, nbw)\n"
        "    hv, ht, d, e = binding.bulge_chase(N, nbw, torch.from_numpy(np.ascontiguousarray(ab.T)).cuda())\n"
        "    torch.cuda.synchronize()\n"
        "    assert binding.last_launch_count() > 100\n"
        "    assert np.array_equal(hv.cpu().numpy(), hv_o) and np.array_equal(ht.cpu().numpy(), ht_o)\n"
        "    assert np.array_equal(d.cpu().numpy(), d_o) and np.array_equal(e.cpu().numpy(), e_o)\n"
        "for kind in ('blockdiag', 'narrow2', 'zerotail', 'zero'):\n"
        "  for cplx, N, nbw in ((False, 300, 64), (True, 200, 32), (True, 300, 128)):\n"
        "    ab = si.structured_band_matrix(N, nbw, 9, cplx, kind)\n"
        "    hv_o, ht_o, d_o, e_o = orc.bulge_chase(ab.copy(order='F'), nbw)\n"
        "    hv, ht, d, e = binding.bulge_chase(N, nbw, torch.from_numpy(np.ascontiguousarray(ab.T)).cuda())\n"
        "    torch.cuda.synchronize()\n"
        "    assert np.array_equal(hv.cpu().numpy(), hv_o) and np.array_equal(ht.cpu().numpy(), ht_o), kind\n"
        "    assert np.array_equal(d.cpu().numpy(), d_o) and np.array_equal(e.cpu().numpy(), e_o), kind\n"
        "print('ok')\n")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, ELPA2_BC_WAVEFRONT="1", PYTHONPATH=root + os.pathsep + os.path.join(root, "tests"))
    out = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=900, cwd=root, env=env)
    assert out.returncode == 0 and out.stdout.strip().endswith("ok"), out.stderr[-2000:]


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw", [(64, 32), (257, 64)])
def test_chase_eigenvalues_and_end_to_end(N, nbw, cplx):
    import torch
    from scipy.linalg import eigh_tridiagonal

    from paper_2002_10991_b200 import binding

    ab = si.band_matrix(N, nbw, 77, cplx)
    B = dense_from_band(ab, nbw)
    hv, ht, d, e, _ = _gpu_chase(ab, N, nbw)
    lam, X = eigh_tridiagonal(d.cpu().numpy(), e.cpu().numpy())
    nB = np.linalg.norm(B, 2)
    assert np.abs(lam - np.linalg.eigvalsh(B)).max() <= 1e-12 * N * nB
    # back-transform the eigenvectors of T with the reflectors that never left the device
    Xc = X.astype(np.complex128) if cplx else X
    q = torch.from_numpy(np.ascontiguousarray(Xc.T)).cuda().t()
    binding.trans_ev_tridi_to_band(N, nbw, hv, ht, q)
    torch.cuda.synchronize()
    Y = q.cpu().numpy()
    assert np.abs(B @ Y - Y * lam).max() / nB <= 1e-12 * N
    assert np.abs(Y.conj().T @ Y - np.eye(N)).max() <= 1e-12 * N
