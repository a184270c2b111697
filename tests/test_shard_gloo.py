"""The N > 1 path on CPU (gloo, world_size 2): column shards are disjoint, cover every column, each
rank's result equals the corresponding columns of the single-process result (columns are
independent), and the timing reduction is the max over ranks."""
import os
import socket

import numpy as np
import pytest

import oracle as orc
from paper_2002_10991_b200 import shard, synth_inputs as si


@pytest.mark.parametrize("nev,world", [(0, 2), (5, 2), (8, 2), (9, 2), (100, 3), (4096, 8), (17, 4)])
def test_column_shard_partitions_every_column(nev, world):
    seen = []
    for rank in range(world):
        c0, n = shard.column_shard(nev, rank, world)
        assert n >= 0 and (c0 % 8 == 0 or n == 0)
        seen.extend(range(c0, c0 + n))
    assert seen == list(range(nev))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, N, nbw, nev, out_dir):
    import torch.distributed as dist

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ab = si.band_matrix(N, nbw, 11, False)
        hh_v, hh_tau, _, _ = orc.bulge_chase(ab, nbw)          # replicated reflector stream
        x = np.asfortranarray(si.gaussian_block(N, nev, 5, False, "cpu").numpy())
        c0, n = shard.column_shard(nev, rank, world)
        mine = np.array(x[:, c0:c0 + n], order="F", copy=True)
        if n:
            orc.back_transform(N, nbw, hh_v, hh_tau, mine)
        np.save(os.path.join(out_dir, f"shard{rank}.npy"), mine)
        t = shard.max_over_ranks(1.0 + rank, dist)             # "time" of this rank
        agg = shard.aggregate_throughput(10.0, world, t)
        np.save(os.path.join(out_dir, f"time{rank}.npy"), np.array([t, agg]))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_rank_column_shards_match_single_process(tmp_path):
    import torch.multiprocessing as mp

    N, nbw, nev, world = 150, 32, 21, 2
    mp.spawn(_worker, args=(world, _free_port(), N, nbw, nev, str(tmp_path)), nprocs=world, join=True)
    ab = si.band_matrix(N, nbw, 11, False)
    hh_v, hh_tau, _, _ = orc.bulge_chase(ab, nbw)
    want = np.asfortranarray(si.gaussian_block(N, nev, 5, False, "cpu").numpy())
    orc.back_transform(N, nbw, hh_v, hh_tau, want)
    got = np.concatenate([np.load(tmp_path / f"shard{r}.npy") for r in range(world)], axis=1)
    assert got.shape == want.shape
    assert np.array_equal(got, want)          # same arithmetic per column: bit-identical
    for r in range(world):
        t, agg = np.load(tmp_path / f"time{r}.npy")
        assert t == float(world)              # max over ranks of 1 + rank
        assert agg == world * 10.0 / world
