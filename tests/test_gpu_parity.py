"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, on the
same seeded inputs.  Tolerance from BASELINE.json north_star: max|dQ| <= 1e-11 * ||X||_max; a
tighter diagnostic bound is asserted too: the two sides differ only in
summation order, so the error must stay near 1e-15 * sqrt(N)-ish.
"""
import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import synth_inputs as si
from gpu_util import run_gpu, oracle_apply

pytestmark = pytest.mark.gpu

TOL = 1e-11


def _tight(N):
    return 2e-14 * max(1.0, (N / 64.0)) ** 0.5 * 8


def _reflectors(N, nbw, seed, cplx):
    ab = si.band_matrix(N, nbw, seed, cplx)
    hh_v, hh_tau, d, e = orc.bulge_chase(ab, nbw)
    return hh_v, hh_tau, d, e


def _x(N, nev, seed, cplx):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((N, nev))
    if cplx:
        x = x + 1j * rng.standard_normal((N, nev))
    return np.asfortranarray(x)


def _check(N, nbw, nev, cplx, ldq=None, variant=0, seed=0):
    hh_v, hh_tau, _, _ = _reflectors(N, nbw, 4000 + seed + N, cplx)
    x = _x(N, nev, 17 + seed, cplx)
    want = oracle_apply(N, nbw, hh_v, hh_tau, x)
    got, pad = run_gpu(N, nbw, hh_v, hh_tau, x, ldq=ldq, variant=variant)
    xmax = max(np.abs(x).max(initial=0.0), 1e-300)
    err = np.abs(got - want).max(initial=0.0) / xmax
    assert err <= TOL, (N, nbw, nev, cplx, err)
    assert err <= _tight(N), (N, nbw, nev, cplx, err)
    assert np.all(pad == 7.25)                       # rows N..ldq-1 untouched
    return err


# SURVEY.md section 4 tier T2: edge shapes around the window/tile/strip boundaries
def _edge_N(nbw):
    return [2, 3, 15, 16, 17, nbw - 1, nbw, nbw + 1, nbw + 2, 2 * nbw - 1, 2 * nbw + 1, 3 * nbw + 5]


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("nbw", [32, 64, 128])
def test_edge_rows(nbw, cplx):
    for N in _edge_N(nbw):
        _check(N, nbw, 7, cplx)


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("nbw", [32, 64, 128])
@pytest.mark.parametrize("nev", [1, 7, 33, 100])
def test_edge_columns(nbw, nev, cplx):
    _check(3 * nbw + 5, nbw, nev, cplx)


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("nbw", [32, 64, 128])
def test_ldq_padding_and_unaligned(nbw, cplx):
    N = 2 * nbw + 9
    _check(N, nbw, 19, cplx, ldq=N + 6)     # even ldq > N
    _check(N, nbw, 19, cplx, ldq=N + 3)     # ldq*8 not 16-byte aligned -> 8-byte path (real)
    _check(N + 1, nbw, 19, cplx, ldq=N + 1)


@pytest.mark.parametrize("cplx", [False, True])
def test_nev_equals_N_square(cplx):
    _check(200, 32, 200, cplx)
    _check(333, 64, 333, cplx)


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("nbw", [32, 64, 128])
def test_many_warps_and_ctas(nbw, cplx):
    # enough columns for several CTAs with several consumer warps each, ragged last strip
    _check(5 * nbw + 3, nbw, 2500 + 13, cplx)


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("nbw", [32, 64, 128])
def test_chain_parallel_mode(nbw, cplx):
    # few columns and many chains: P = 2 / 4 warps share a slab, each on its own chains, with the
    # hand-over of retired rows through global memory; ragged N, ragged last slab
    _check(9 * nbw + 3, nbw, 5, cplx)            # K0 = 10: P = 2, one slab
    _check(17 * nbw + 1, nbw, 9, cplx)           # K0 = 18: P = 4 (real) / 2 (complex), two slabs
    _check(16 * nbw, nbw, 200, cplx)             # 25 slabs on 25 CTAs
    _check(12 * nbw + 7, nbw, 148 * 8 * 3 + 5, cplx)   # 3-4 slabs per CTA: P = 2, ragged tail


@pytest.mark.parametrize("nbw,n", [(32, 5), (64, 6), (64, 7), (64, 10), (64, 12), (64, 13), (64, 14), (128, 3), (128, 7), (96, 4)])
def test_partial_spectrum_plans(nbw, n):
    # 5-16 slabs per CTA: the plan shares slab groups among P = 4 / 2 warps with SEVERAL slabs per warp
    # (the sub-partition balance of DESIGN.md 5.1); ragged last slab
    from paper_2002_10991_b200 import binding

    N, nev = 17 * nbw + 1, 148 * 8 * n - 3
    assert binding.plan(False, N, nbw, nev, 148)["P"] in (2, 4)
    _check(N, nbw, nev, False)


@pytest.mark.parametrize("nbw,n", [(32, 5), (64, 6), (64, 8)])
def test_partial_spectrum_plans_complex(nbw, n):
    # complex: P = 2 with two slabs per group of warps (5-8 slabs per CTA)
    from paper_2002_10991_b200 import binding

    N, nev = 17 * nbw + 1, 148 * 8 * n - 3
    assert binding.plan(True, N, nbw, nev, 148)["P"] == (2 if n < 8 else 1)
    _check(N, nbw, nev, True)
    old = binding.set_chain_parallel(2)                 # forced: also the shapes the plan leaves at P = 1
    try:
        _check(N, nbw, nev, True, seed=1)
    finally:
        binding.set_chain_parallel(old)


@pytest.mark.parametrize("cplx", [False, True])
def test_more_columns_than_one_wave(cplx):
    # more slabs than 148 CTAs x 8 warps x NGMAX: the grid becomes a multiple of the SM count > 1
    nev = 148 * 8 * 8 * (2 if cplx else 4) + 8 * 31 + 3
    _check(70, 32, nev, cplx)


def test_repeated_and_concurrent_calls_share_the_scratch_pool():
    """Two streams, interleaved calls on different problems: every call takes its scratch from the
    stream-ordered pool, so neither host synchronisation nor cross-talk may occur."""
    import torch

    from paper_2002_10991_b200 import binding
    from gpu_util import to_device_colmajor

    probs = []
    for (N, nbw, nev, seed) in ((300, 64, 64, 1), (17 * 32 + 1, 32, 9, 2), (260, 128, 40, 3)):
        hh_v, hh_tau, _, _ = _reflectors(N, nbw, 90 + seed, False)
        x = _x(N, nev, seed, False)
        probs.append((N, nbw, torch.from_numpy(hh_v).cuda(), torch.from_numpy(hh_tau).cuda(), x,
                      oracle_apply(N, nbw, hh_v, hh_tau, x)))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    outs = []
    for rep in range(3):
        for i, (N, nbw, dv, dt, x, want) in enumerate(probs):
            s = streams[(i + rep) % 2]
            with torch.cuda.stream(s):
                q = to_device_colmajor(x)
                binding.trans_ev_tridi_to_band(N, nbw, dv, dt, q, stream=s)
            outs.append((q, want, x))
    torch.cuda.synchronize()
    for q, want, x in outs:
        assert np.abs(q.cpu().numpy() - want).max() <= TOL * np.abs(x).max()


@pytest.mark.parametrize("cplx", [False, True])
def test_simple_variant_matches_oracle(cplx):
    _check(150, 32, 37, cplx, variant=1)
    _check(300, 64, 21, cplx, variant=1)
    _check(300, 128, 21, cplx, variant=1)


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("nbw", [32, 64, 128])
def test_register_window_variant_matches_oracle(nbw, cplx):
    # variant 2: one reflector at a time (DFMA), the A/B partner of the default compact-WY path
    _check(3 * nbw + 5, nbw, 100, cplx, variant=2)
    _check(2 * nbw + 9, nbw, 19, cplx, ldq=2 * nbw + 9 + 3, variant=2)


@pytest.mark.parametrize("nbw", [32, 64, 128])
def test_two_chains_per_pass_variant(nbw):
    # variant 3 (real): pairs of warps share their slabs and walk alternate chains, several slabs per warp
    _check(9 * nbw + 3, nbw, 148 * 8 * 2 + 21, False, variant=3)     # 2-3 slabs per CTA
    _check(8 * nbw, nbw, 5000, False, variant=3)
    _check(3 * nbw + 5, nbw, 100, False, variant=3)                  # too few chains: falls back to P = 1
    if nbw == 32:
        _check(9 * nbw + 3, nbw, 148 * 16 * 8 + 100, False, variant=3)  # more than one wave of CTAs, 4-slab warps


def test_degenerate_no_work():
    for N, nev in ((0, 5), (1, 5), (40, 0)):
        x = np.zeros((N, nev), order="F")
        got, _ = run_gpu(N, 32, np.zeros((0, 32)), np.zeros(0), x)
        assert got.shape == (N, nev)


def test_identity_reflectors_leave_q_bitwise():
    N, nbw, nev = 200, 64, 50
    G = orc.hh_count(N, nbw)
    hh_v = np.zeros((G, nbw))
    hh_v[:, 0] = 1.0
    hh_tau = np.zeros(G)
    x = _x(N, nev, 3, False)
    got, _ = run_gpu(N, nbw, hh_v, hh_tau, x)
    assert np.array_equal(got, x)


@pytest.mark.parametrize("cplx", [False, True])
def test_host_entry_point(cplx):
    from paper_2002_10991_b200 import binding

    N, nbw, nev = 260, 64, 45
    hh_v, hh_tau, _, _ = _reflectors(N, nbw, 77, cplx)
    x = _x(N, nev, 5, cplx)
    want = oracle_apply(N, nbw, hh_v, hh_tau, x)
    y = np.array(x, order="F", copy=True)
    binding.trans_ev_tridi_to_band_host(N, nbw, hh_v, hh_tau, y)
    assert np.abs(y - want).max() <= TOL * np.abs(x).max()
    assert binding.last_launch_count() == 2     # T-factor prepass + main kernel


def test_launch_on_side_stream():
    import torch

    from paper_2002_10991_b200 import binding
    from gpu_util import to_device_colmajor

    N, nbw, nev = 300, 64, 64
    hh_v, hh_tau, _, _ = _reflectors(N, nbw, 78, False)
    x = _x(N, nev, 6, False)
    want = oracle_apply(N, nbw, hh_v, hh_tau, x)
    s = torch.cuda.Stream()
    q = to_device_colmajor(x)
    dv, dt = torch.from_numpy(hh_v).cuda(), torch.from_numpy(hh_tau).cuda()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        binding.trans_ev_tridi_to_band(N, nbw, dv, dt, q, stream=s)
    s.synchronize()
    assert np.abs(q.cpu().numpy() - want).max() <= TOL * np.abs(x).max()


def test_release_scratch_and_reuse():
    """The cached scratch can be handed back and the next calls allocate again."""
    import torch

    from paper_2002_10991_b200 import binding

    before = torch.cuda.mem_get_info()[0]
    _check(300, 64, 40, False)
    N, nbw, nev = 260, 64, 45
    hh_v, hh_tau, _, _ = _reflectors(N, nbw, 77, True)
    x = _x(N, nev, 5, True)
    y = np.array(x, order="F", copy=True)
    binding.trans_ev_tridi_to_band_host(N, nbw, hh_v, hh_tau, y)
    binding.release_scratch()
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= before - (64 << 20)       # nothing sizeable is held back
    _check(300, 64, 40, True)                                          # and the library still works
    y2 = np.array(x, order="F", copy=True)
    binding.trans_ev_tridi_to_band_host(N, nbw, hh_v, hh_tau, y2)
    assert np.array_equal(y, y2)
