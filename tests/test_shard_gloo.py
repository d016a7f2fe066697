"""N > 1 host logic on CPU: world_size-2 gloo.

The path shards by contiguous flat-index ranges with NO data-path collective: rank r scans
workloads.shard_range(G, r, world) through first_index/count.  Checked here with the CPU oracle standing in for
the per-rank scan (it takes the same first_index/count): the shards tile [0, G) exactly, every rank's slice is
bit-identical to the same slice of the unsharded scan (results are keyed by the GLOBAL flat index), and the only
collectives are the ones bench.py uses -- a barrier and a MAX all-reduce of the step time.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import zmc_oracle as orc
from paper_1910_01965_b200 import binding as zb
from paper_1910_01965_b200 import workloads as wl


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, tmpdir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = wl.config(5, scale=[3, 5, 4, 3, 7], n_samples=64)        # G = 1260, not divisible by the batch size below
        first, count = wl.shard_range(w.G, rank, world)
        # the library's own batch cutting of this rank's range (pure host helper, no GPU needed)
        nb, _, _ = zb.zmc_batch_range(first, count, 100, 0)
        covered = 0
        for b in range(nb):
            _, bf, bc = zb.zmc_batch_range(first, count, 100, b)
            assert bf == first + covered
            covered += bc
        assert covered == count
        rc, mean, err = orc.scan_workload(w, first, count)
        assert rc == 0
        # gather the (first, count) pairs and the step "time" the way bench.py does
        spans = [None] * world
        dist.all_gather_object(spans, (first, count))
        t = torch.tensor([10.0 + rank], dtype=torch.float64)
        dist.barrier()
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert float(t) == 10.0 + world - 1
        np.save(os.path.join(tmpdir, f"mean{rank}.npy"), mean)
        np.save(os.path.join(tmpdir, f"err{rank}.npy"), err)
        if rank == 0:
            pos = 0
            for f, c in spans:                      # contiguous, ordered, gap-free tiling of [0, G)
                assert f == pos
                pos += c
            assert pos == w.G
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_shards_tile_the_grid_and_reproduce_the_unsharded_scan(tmp_path, world):
    port = _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    w = wl.config(5, scale=[3, 5, 4, 3, 7], n_samples=64)
    rc, mean_all, err_all = orc.scan_workload(w)
    assert rc == 0
    mean = np.concatenate([np.load(tmp_path / f"mean{r}.npy") for r in range(world)])
    err = np.concatenate([np.load(tmp_path / f"err{r}.npy") for r in range(world)])
    assert np.array_equal(mean, mean_all) and np.array_equal(err, err_all)      # bit-identical


def test_shard_range_properties():
    for G in (1, 7, 1000, 10**10):
        for world in (1, 2, 3, 8):
            pos = 0
            sizes = []
            for r in range(world):
                f, c = wl.shard_range(G, r, world)
                assert f == pos
                pos += c
                sizes.append(c)
            assert pos == G and max(sizes) - min(sizes) <= 1
