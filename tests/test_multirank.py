"""World-size-2 gloo tests (CPU) of the multi-GPU host logic: antennas shard across ranks with no data-path
collective; the only reduction is the max of the timing scalar."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import synth_inputs as si
from paper_2303_09886_b200 import sharding


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, A, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = si.custom_workload(A=A, n=64, T=4, S=6, P=2, seed=5, random_weights=True, coarse_range=(-10, 200))
        mine = sharding.shard_antennas(A, world, rank)
        sel = list(mine)
        # the product-side slicing: exactly what a rank hands to FEngine(...) / the setters / fengine_process
        rs = sharding.rank_slice(world, rank, w.packed, w.coarse, w.fine_delay, w.phase, w.gains)
        assert rs["n_antennas"] == len(sel) and list(rs["antennas"]) == sel
        for key, full in (("packed", w.packed), ("coarse", w.coarse), ("fine_delay", w.fine_delay), ("phase", w.phase),
                          ("gains", w.gains)):
            assert rs[key].flags["C_CONTIGUOUS"] and rs[key].dtype == full.dtype
            np.testing.assert_array_equal(rs[key], full[sel])
        # each rank runs the path on its own antennas only (here: the oracle stands in for the GPU, CPU test)
        res = oracle.process(rs["packed"], rs["n_antennas"], w.n, w.T, w.P, w.weights, w.S, coarse=rs["coarse"],
                             fine_delay=rs["fine_delay"], phase=rs["phase"], gains=rs["gains"])
        np.save(os.path.join(out_dir, f"out_{rank}.npy"), res["out"])
        t = sharding.max_over_ranks(1.0 + rank, dist)            # slowest rank decides
        assert t == float(world)
        assert sharding.aggregate_rate(100, world, t) == pytest.approx(100 * world / world)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("A", [3, 4])
def test_antenna_shards_reassemble_to_the_full_result(tmp_path, A):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), A, str(tmp_path)), nprocs=world, join=True)
    w = si.custom_workload(A=A, n=64, T=4, S=6, P=2, seed=5, random_weights=True, coarse_range=(-10, 200))
    full = oracle.process(w.packed, w.A, w.n, w.T, w.P, w.weights, w.S, coarse=w.coarse, fine_delay=w.fine_delay,
                          phase=w.phase, gains=w.gains)["out"]
    parts = [np.load(tmp_path / f"out_{r}.npy") for r in range(world)]
    np.testing.assert_array_equal(np.concatenate(parts, axis=0), full)


def test_shards_partition_the_antennas():
    for A in range(0, 20):
        for world in range(1, 9):
            got = [a for r in range(world) for a in sharding.shard_antennas(A, world, r)]
            assert got == list(range(A))
            sizes = [len(sharding.shard_antennas(A, world, r)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_antennas(4, 2, 2)
