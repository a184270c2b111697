"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/elpa2_bt.h
declares, its integer layout helpers agree with the oracle's plain sums, and argument validation
(which runs before any CUDA call) returns the documented codes.  No compute calls."""
import ctypes
import os
import re

import pytest

import oracle as orc
from paper_2002_10991_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    binding.build()
    return binding.lib()


def test_header_symbols_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "elpa2_bt.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(elpa2_[a-z0-9_]+)\s*\(", hdr))
    assert names == set(binding.EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None
    assert b"sm_100a" in lib.elpa2_bt_version()


@pytest.mark.parametrize("N", [0, 1, 2, 3, 17, 33, 64, 65, 100, 129, 512, 1000])
@pytest.mark.parametrize("nbw", [4, 32, 48, 64, 96, 128, 160, 192, 224, 256])
def test_layout_helpers_match_oracle(lib, N, nbw):
    assert binding.hh_count(N, nbw) == orc.hh_count(N, nbw)
    for s in range(max(N - 1, 0)):
        assert binding.hh_offset(N, nbw, s) == orc.hh_offset(N, nbw, s)
        assert binding.hh_blocks(N, nbw, s) == orc.hh_blocks(N, nbw, s)
    if N >= 2:
        assert binding.hh_offset(N, nbw, N - 1) == orc.hh_count(N, nbw)
        assert binding.hh_offset(N, nbw, N) == -1
        assert binding.hh_blocks(N, nbw, N - 1) == 0


@pytest.mark.parametrize("N,nbw", [(2, 32), (17, 32), (17, 4), (33, 32), (100, 64), (130, 128), (515, 64), (1000, 32), (700, 96),
                                   (999, 160), (600, 256)])
def test_hh_lengths_match_oracle_rows(lib, N, nbw):
    """elpa2_hh_lengths (the only place the binding gets slot lengths from) against the oracle's
    row map, which the paper's worked example pins (tests/test_oracle_layout.py)."""
    got = binding.hh_lengths(N, nbw)
    want = [orc.hh_rows(N, nbw, s, k)[2] for s in range(N - 1) for k in range(orc.hh_blocks(N, nbw, s))]
    assert got.tolist() == want
    assert int(got.sum()) == N * (N - 1) // 2          # sum of L = N(N-1)/2
    assert lib.elpa2_hh_lengths(N, nbw, None, 0) == len(want)


def test_variant_selector_is_per_thread(lib):
    """elpa2_bt_set_variant in one thread changes neither another thread's variant nor its plan."""
    import threading

    args = (False, 4096, 64, 32768, 148)
    base = binding.plan(*args)
    assert binding.set_variant(0) == 0
    seen = {}

    def other():
        seen["old"] = binding.set_variant(3)          # this thread starts at the default, 0
        seen["plan3"] = binding.plan(*args)
        seen["now"] = binding.set_variant(3)

    t = threading.Thread(target=other)
    t.start()
    t.join()
    assert seen["old"] == 0 and seen["now"] == 3
    assert seen["plan3"]["P"] == 2                     # variant 3: two chains per pass
    assert binding.plan(*args) == base and base["P"] == 1
    assert binding.set_variant(0) == 0                 # still the default here


def test_layout_full_size_counts(lib):
    # G for the five configs
    assert binding.hh_count(512, 32) == 4336
    assert binding.hh_count(4096, 64) == 133056
    assert binding.hh_count(8192, 64) == 528256
    assert binding.hh_count(32768, 64) == 8404480
    assert binding.hh_count(16384, 128) == 1056640
    assert binding.hh_count(100, 48) == orc.hh_count(100, 48)      # the layout helpers take any nbw >= 1 (R13)
    assert binding.hh_count(100, 0) == 0


def test_argument_validation_codes(lib):
    buf = (ctypes.c_double * 64)()
    p = ctypes.addressof(buf)
    p16 = (p + 15) & ~15
    call = binding.trans_ev_tridi_to_band_raw
    for cplx in (False, True):
        assert call(cplx, -1, 64, 4, p16, p16, p16, 8, 0) == -1
        assert call(cplx, 8, 48, 4, p16, p16, p16, 8, 0) == -2        # not a multiple of 32
        assert call(cplx, 8, 288, 4, p16, p16, p16, 8, 0) == -2       # wider than the widest instantiated kernel
        assert call(cplx, 8, 64, -4, p16, p16, p16, 8, 0) == -3
        assert call(cplx, 8, 64, 4, 0, p16, p16, 8, 0) == -4
        assert call(cplx, 8, 64, 4, p16 + 8, p16, p16, 8, 0) == -4
        assert call(cplx, 8, 64, 4, p16, 0, p16, 8, 0) == -5
        assert call(cplx, 8, 64, 4, p16, p16, 0, 8, 0) == -6
        assert call(cplx, 8, 64, 4, p16, p16, p16 + 4, 8, 0) == -6
        assert call(cplx, 8, 64, 4, p16, p16, p16, 7, 0) == -7
        # no work: success without touching CUDA
        assert call(cplx, 0, 64, 4, 0, 0, 0, 1, 0) == 0
        assert call(cplx, 1, 64, 4, 0, 0, 0, 1, 0) == 0
        assert call(cplx, 8, 64, 0, 0, 0, 0, 8, 0) == 0
    assert lib.elpa2_trans_ev_tridi_to_band_host(0, 8, 40, 4, p16, p16, p16, 8) == -2
    assert lib.elpa2_trans_ev_tridi_to_band_host(1, 8, 32, 4, p16, p16, p16, 4) == -7
    assert binding.set_variant(7) == -1
    assert binding.set_variant(0) in (0, 1, 2, 3)


def test_no_gpu_fails_loudly(lib):
    """Without a device the compute call must fail with a cudaError_t (> 0), never silently."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    buf = (ctypes.c_double * 4096)()
    p16 = (ctypes.addressof(buf) + 15) & ~15
    rc = binding.trans_ev_tridi_to_band_raw(False, 8, 32, 2, p16, p16, p16, 8, 0)
    assert rc > 0


def test_missing_library_raises(monkeypatch):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", "/nonexistent/libelpa2_bt.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.lib()


def test_launch_plan_of_the_five_configs():
    """elpa2_bt_plan: host arithmetic of the decomposition, no device needed."""
    want = {
        (False, 512, 32, 512): (64, 16, 4),          # 64 slabs: one per CTA, 4 warps on each
        (False, 4096, 64, 4096): (148, 16, 4),       # 512 slabs: 3-4 per CTA, 16-warp build
        (True, 8192, 64, 4096): (148, 8, 2),         # complex: 8 warps, 2 per slab
        (False, 32768, 64, 32768): (148, 8, 1),      # 4096 slabs: 27-28 per CTA
        (True, 16384, 128, 8192): (148, 8, 1),       # 1024 slabs: 6-7 per CTA
    }
    for (cplx, N, nbw, nev), (grid, nw, P) in want.items():
        pl = binding.plan(cplx, N, nbw, nev, 148)
        assert (pl["grid"], pl["warps_per_cta"], pl["P"]) == (grid, nw, P), (cplx, N, nbw, nev, pl)
        assert pl["slabs"] == (nev + 7) // 8


def test_launch_plan_balances_sub_partitions_for_partial_spectra():
    """PAPER.md:218 (KS-DFT: 20-69 % of the eigenvectors): 5-16 slabs per SM.  The plan picks the number of
    warps per slab group that balances the four sub-partitions (measured table there)."""
    N, nbw = 32768, 64
    for frac, P in ((0.2, 4), (0.25, 4), (0.4, 2), (0.35, 2), (0.45, 2), (0.5, 2), (0.6, 1), (0.69, 1), (1.0, 1)):
        nev = int(round(frac * N))
        pl = binding.plan(False, N, nbw, nev, 148)
        assert pl["P"] == P and pl["grid"] == 148 and pl["warps_per_cta"] == 8, (frac, pl)
    # wider bands hold fewer slabs per warp: P = 4 needs n <= 2 * ngmax
    assert binding.plan(False, N, 128, 148 * 8 * 4, 148)["P"] == 4
    assert binding.plan(False, N, 128, 148 * 8 * 7, 148)["P"] == 2
    assert binding.plan(False, N, 256, 148 * 8 * 3, 148)["P"] == 2      # 4 ring stages: P <= 2
    assert binding.plan(True, 16384, 128, 8192, 148)["P"] == 1          # complex nbw 128: one slab per warp, 7 per SM
    assert binding.plan(True, 8192, 64, 148 * 8 * 6, 148)["P"] == 2     # complex nbw 64, 6 slabs per SM: 2 + 2 + 1 + 1 on pairs
    assert binding.plan(True, 8192, 64, 148 * 8 * 7, 148)["P"] == 1


def test_launch_plan_invariants():
    import itertools

    for cplx, nbw, N, nev, nsm in itertools.product((False, True), (32, 64, 128), (2, 70, 600, 5000),
                                                    (1, 8, 9, 1000, 9473, 40000, 100001), (1, 7, 148)):
        pl = binding.plan(cplx, N, nbw, nev, nsm)
        nslab = (nev + 7) // 8
        assert pl["slabs"] == nslab
        assert 1 <= pl["grid"] <= max(nslab, 1)
        assert pl["grid"] == nslab or pl["grid"] % nsm == 0          # a multiple of the SM count, or one slab per CTA
        assert pl["P"] in (1, 2, 4) and pl["warps_per_cta"] in (8, 16) and pl["warps_per_cta"] % pl["P"] == 0
        # every slab has a place: the fullest CTA gets ceil(nslab / grid) slabs
        assert -(-nslab // pl["grid"]) <= pl["slabs_per_cta_max"], (cplx, nbw, N, nev, nsm, pl)
        assert pl["scratch_bytes"] > 0
    assert binding.plan(False, 1, 64, 10) == dict.fromkeys(("grid", "warps_per_cta", "P", "slabs", "slabs_per_cta_max",
                                                           "scratch_bytes"), 0)


def test_release_scratch_without_anything_cached():
    binding.release_scratch()          # nothing cached, no device needed: success
