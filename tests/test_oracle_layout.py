"""Pins for the reflector row map / slot layout of the oracle (orc_hh_*).

Pinned to the paper's worked example N = 17, b = 4 (Figs. 1-4, text at :113, :130, :136,
:138, :164, :178; fixtures in tests/golden/ with citations) and to counting identities that hold
for any N, nbw (sum of reflector lengths = N(N-1)/2: every sub-diagonal entry position (i > j+... )
is hit exactly once per sweep row -- see test body).
"""
import os

import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import synth_inputs as si

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read(name):
    rows = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append([int(t) for t in line.split()])
    return rows


def test_paper_worked_example_rows():
    N, b = 17, 4
    for i, j, first, last in _read("paper_n17_b4_rows.txt"):
        r0, r1, L = orc.hh_rows(N, b, i - 1, j - 1)
        assert (r0 + 1, r1 + 1) == (first, last), (i, j)
        assert L == last - first + 1
        assert j - 1 < orc.hh_blocks(N, b, i - 1)


def test_paper_worked_example_xlocal_rows():
    # N_R = 7 rows for the four reflectors (8,1) (7,1) (6,1) (5,1) of length 4
    N, b = 17, 4
    rows = set()
    for i in (8, 7, 6, 5):
        r0, r1, _ = orc.hh_rows(N, b, i - 1, 0)
        rows.update(range(r0, r1 + 1))
    assert len(rows) == 7 == b + 4 - 1
    # window shifts upward by exactly one row per reflector
    tops = [orc.hh_rows(N, b, i - 1, 0)[0] for i in (8, 7, 6, 5)]
    assert tops == [tops[0] - t for t in range(4)]


def test_paper_worked_example_sweep_count():
    # PAPER.md:113 "The fourth stage consists of (N-i)/b = 3 sweeps": non-identity reflectors of
    # a generic band matrix in stage i, counted from an actual chase.
    N, b = 17, 4
    ab = si.band_matrix(N, b, 11)
    _, tau, _, _ = orc.bulge_chase(ab, b)
    for i, want in _read("paper_n17_b4_counts.txt"):
        s = i - 1
        off, K = orc.hh_offset(N, b, s), orc.hh_blocks(N, b, s)
        assert int(np.count_nonzero(tau[off:off + K])) == want
        assert K in (want, want + 1)  # at most one trailing identity slot (R3)


@pytest.mark.parametrize("N,nbw", [(2, 32), (3, 2), (17, 4), (33, 32), (65, 32), (100, 7), (257, 64),
                                   (512, 32), (129, 128)])
def test_layout_counting_identities(N, nbw):
    G = orc.hh_count(N, nbw)
    total_len = 0
    g = 0
    hit = np.zeros(N, dtype=np.int64)
    for s in range(N - 1):
        assert orc.hh_offset(N, nbw, s) == g
        K = orc.hh_blocks(N, nbw, s)
        assert K >= 1
        prev_r1 = s
        for k in range(K):
            r0, r1, L = orc.hh_rows(N, nbw, s, k)
            assert r0 == prev_r1 + 1 and r1 <= N - 1 and 1 <= L <= nbw
            assert L == nbw or k == K - 1          # only the last may be shorter
            prev_r1 = r1
            total_len += L
            hit[r0:r1 + 1] += 1
        assert prev_r1 == N - 1                    # one sweep tiles rows s+1 .. N-1 exactly
        g += K
    assert g == G
    assert total_len == N * (N - 1) // 2
    # row i is touched once per sweep s < i
    assert np.array_equal(hit, np.arange(N))


def test_layout_degenerate():
    assert orc.hh_count(0, 32) == 0
    assert orc.hh_count(1, 32) == 0
    assert orc.hh_count(2, 32) == 1
    assert orc.hh_blocks(5, 32, 4) == 0   # s beyond N-2
    assert orc.hh_blocks(5, 32, -1) == 0
