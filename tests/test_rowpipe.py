"""host logic of the row-pipelined multi-GPU variant (paper_2002_10991_b200/rowpipe.py)
on the CPU.  The schedule is executed (a) by R emulated ranks in one process and (b) by real processes
over gloo (world size 2 and 3) with messages of nbw rows; the row-block step is a numpy restatement of the
library call's definition (include/elpa2_bt.h: of chain k, the reflectors whose first row lies in the
owned rows, s descending).  The assembled rows must equal the oracle's back-transformation: the
partition, the split of a rank's rows into two calls, the order of the hand-overs and their sizes are
what is being pinned."""
import os
import socket

import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import rowpipe, synth_inputs as si


def _inputs(N, nbw, ncols, cplx, seed=3):
    ab = si.band_matrix(N, nbw, 40 + seed, cplx)
    hh_v, hh_tau, _, _ = orc.bulge_chase(ab, nbw)
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((N, ncols)) + (1j * rng.standard_normal((N, ncols)) if cplx else 0)
    x = np.asfortranarray(x)
    want = np.array(x, order="F", copy=True)
    orc.back_transform(N, nbw, hh_v, hh_tau, want)
    return hh_v, hh_tau, x, want


def _numpy_apply(N, nbw, hh_v, hh_tau, bounds):
    """The row-block call by definition: chain op.k, reflectors with first row in [row0, row0 + nown)
    (8-row blocks; to N if the range ends the matrix), applied s descending to the local rows."""

    def fn(r, buf, op):
        k = op.k
        b = np.asarray(buf)
        base = bounds[r]                       # global row of local row 0
        hi = N if op.row0 + op.nown >= N else op.row0 + op.nown
        for s in range(N - 2, -1, -1):
            if k >= orc.hh_blocks(N, nbw, s):
                continue
            r0 = s + 1 + k * nbw
            if not (op.row0 <= r0 < hi):
                continue
            L = min(nbw, N - r0)
            g = orc.hh_offset(N, nbw, s) + k
            v, t = hh_v[g, :L], hh_tau[g]
            lo = r0 - base
            b[lo:lo + L] -= t * np.outer(v, v.conj() @ b[lo:lo + L])

    return fn


def _bufs(x, N, nbw, bounds):
    R = len(bounds) - 1
    bufs = []
    for r in range(R):
        n = rowpipe.local_rows(N, nbw, bounds, r)
        buf = np.full((n, x.shape[1]), np.nan, dtype=x.dtype)      # halo rows: garbage on entry
        buf[: bounds[r + 1] - bounds[r]] = x[bounds[r]:bounds[r + 1]]
        bufs.append(buf)
    return bufs


@pytest.mark.parametrize("N,world,nbw", [(100, 1, 32), (64, 2, 32), (1000, 2, 32), (1000, 4, 64), (4096, 8, 64), (513, 3, 128),
                                         (32768, 8, 64)])
def test_partition_rows(N, world, nbw):
    b = rowpipe.partition_rows(N, world, nbw)
    assert b[0] == 0 and b[-1] == N and len(b) == world + 1
    for r in range(world):
        assert b[r + 1] - b[r] >= nbw and (b[r] % 8 == 0)
    if N == 32768:                             # equal work: rows i are touched by ~ i / nbw chains
        w = [b[r + 1] ** 2 - b[r] ** 2 for r in range(world)]
        assert max(w) / min(w) < 1.05
    with pytest.raises(ValueError):
        rowpipe.partition_rows(nbw * world - 8, world, nbw) if world > 1 else (_ for _ in ()).throw(ValueError())


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("N,nbw,R", [(70, 32, 2), (97, 32, 3), (200, 32, 4), (130, 64, 2), (300, 64, 3), (64, 32, 2), (96, 32, 3)])
def test_emulated_ranks_reproduce_the_oracle(N, nbw, R, cplx):
    hh_v, hh_tau, x, want = _inputs(N, nbw, 5, cplx)
    bounds = rowpipe.partition_rows(N, R, nbw)
    bufs = _bufs(x, N, nbw, bounds)
    rowpipe.run_emulated(N, nbw, bounds, bufs, _numpy_apply(N, nbw, hh_v, hh_tau, bounds))
    got = np.concatenate([bufs[r][: bounds[r + 1] - bounds[r]] for r in range(R)], axis=0)
    assert np.abs(got - want).max() <= 1e-12 * np.abs(x).max()


def test_schedule_message_sizes_and_pairing():
    """Every send has exactly one matching recv on the peer, in the same order per pair; all messages are
    nbw rows (the paper's "at most nbw rows exchanged with the neighbour")."""
    N, nbw, R = 1000, 64, 4
    bounds = rowpipe.partition_rows(N, R, nbw)
    progs = [rowpipe.schedule(N, nbw, bounds, r) for r in range(R)]
    for r in range(R):
        for peer in (r - 1, r + 1):
            if not 0 <= peer < R:
                continue
            sends = [(o.tag, o.k) for o in progs[r] if o.kind == "send" and o.peer == peer]
            recvs = [(o.tag, o.k) for o in progs[peer] if o.kind == "recv" and o.peer == r]
            assert sends == recvs and len(sends) > 0
    assert all(o.n == nbw for p in progs for o in p if o.kind != "apply")
    assert all(abs(o.peer - r) == 1 for r, p in enumerate(progs) for o in p if o.kind != "apply")
    # every (rank, chain) applies its rows exactly once, lower part before upper part
    for r, p in enumerate(progs):
        for k in range(rowpipe.chains_of(N, nbw, bounds, r)):
            parts = [(o.row0, o.nown) for o in p if o.kind == "apply" and o.k == k]
            assert sum(n for _, n in parts) == bounds[r + 1] - bounds[r]
            assert parts == sorted(parts, reverse=True)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, N, nbw, ncols, cplx, out_dir):
    import torch
    import torch.distributed as dist

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        hh_v, hh_tau, x, _ = _inputs(N, nbw, ncols, cplx)
        bounds = rowpipe.partition_rows(N, world, nbw)
        buf = _bufs(x, N, nbw, bounds)[rank]
        t = torch.from_numpy(np.ascontiguousarray(buf.T)).t()          # column-major torch view of a copy
        rowpipe.run(N, nbw, bounds, t, dist, _numpy_apply(N, nbw, hh_v, hh_tau, bounds))
        np.save(os.path.join(out_dir, f"rows{rank}.npy"), t.numpy()[: bounds[rank + 1] - bounds[rank]])
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,cplx", [(2, False), (3, True)])
def test_gloo_ranks_exchange_halos_and_match_the_oracle(tmp_path, world, cplx):
    import torch.multiprocessing as mp

    N, nbw, ncols = 230, 32, 6
    mp.spawn(_worker, args=(world, _free_port(), N, nbw, ncols, cplx, str(tmp_path)), nprocs=world, join=True)
    _, _, x, want = _inputs(N, nbw, ncols, cplx)
    got = np.concatenate([np.load(tmp_path / f"rows{r}.npy") for r in range(world)], axis=0)
    assert got.shape == want.shape
    assert np.abs(got - want).max() <= 1e-12 * np.abs(x).max()
