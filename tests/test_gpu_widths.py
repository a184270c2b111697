"""semi-bandwidths other than 32 / 64 / 128 ("multiples of 32";
PAPER.md:248: the block-size x semi-bandwidth study).  The back-transformation is instantiated for
every multiple of 32 up to 256 (real) and 160 (complex); reflectors come from the oracle's bulge chase,
which takes any nbw.  Same comparison and tolerance as tests/test_gpu_parity.py.
"""
import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import synth_inputs as si
from gpu_util import run_gpu, oracle_apply

pytestmark = pytest.mark.gpu

TOL = 1e-11
WIDTHS = [(False, w) for w in (96, 160, 192, 224, 256)] + [(True, w) for w in (96, 160)]


def _tight(N):
    return 2e-14 * max(1.0, (N / 64.0)) ** 0.5 * 8


def _x(N, nev, seed, cplx):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((N, nev))
    if cplx:
        x = x + 1j * rng.standard_normal((N, nev))
    return np.asfortranarray(x)


def _check(N, nbw, nev, cplx, ldq=None, variant=0):
    ab = si.band_matrix(N, nbw, 6000 + N + nbw, cplx)
    hh_v, hh_tau, _, _ = orc.bulge_chase(ab, nbw)
    x = _x(N, nev, 23 + N, cplx)
    want = oracle_apply(N, nbw, hh_v, hh_tau, x)
    got, pad = run_gpu(N, nbw, hh_v, hh_tau, x, ldq=ldq, variant=variant)
    err = np.abs(got - want).max(initial=0.0) / max(np.abs(x).max(initial=0.0), 1e-300)
    assert err <= TOL and err <= _tight(N), (N, nbw, nev, cplx, err)
    assert np.all(pad == 7.25)


@pytest.mark.parametrize("cplx,nbw", WIDTHS)
def test_edge_rows(cplx, nbw):
    for N in (2, 17, nbw - 1, nbw, nbw + 1, nbw + 2, 2 * nbw - 1, 2 * nbw + 1, 3 * nbw + 5):
        _check(N, nbw, 7, cplx)


@pytest.mark.parametrize("cplx,nbw", WIDTHS)
def test_columns_leading_dimension_and_many_ctas(cplx, nbw):
    _check(3 * nbw + 5, nbw, 33, cplx)
    _check(2 * nbw + 9, nbw, 19, cplx, ldq=2 * nbw + 9 + 3)     # 8-byte path (real)
    _check(4 * nbw + 3, nbw, 2500 + 13, cplx)                   # several CTAs, several warps each, ragged strip


@pytest.mark.parametrize("cplx,nbw", WIDTHS)
def test_chain_parallel_mode(cplx, nbw):
    _check(9 * nbw + 3, nbw, 5, cplx)            # K0 = 10: P = 2, one slab
    _check(17 * nbw + 1, nbw, 9, cplx)           # K0 = 18: P = 4 (real, 8 ring stages) / 2, two slabs


@pytest.mark.parametrize("cplx,nbw", [(False, 96), (True, 160), (False, 256)])
def test_plain_variant_on_other_widths(cplx, nbw):
    _check(2 * nbw + 11, nbw, 21, cplx, variant=1)


def test_unsupported_widths_are_rejected():
    import torch

    from paper_2002_10991_b200 import binding

    for nbw, dt in ((48, torch.float64), (288, torch.float64), (192, torch.complex128)):
        N = 300
        G = binding.hh_count(N, nbw)
        hv = torch.zeros((G, nbw), dtype=dt, device="cuda")
        ht = torch.zeros((G,), dtype=dt, device="cuda")
        with pytest.raises(binding.Elpa2BtError) as ei:
            binding.trans_ev_tridi_to_band(N, nbw, hv, ht, torch.zeros((4, N), dtype=dt, device="cuda").t())
        assert ei.value.rc == -2
