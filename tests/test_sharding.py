"""World-size-2 gloo test of the multi-GPU plumbing (CPU): ranks own disjoint seeded cell ranges whose
union is the single-process workload, timings reduce with MAX, counters with SUM.
The update itself needs no collective (cells are independent)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2407_18304_b200 import sharding, workloads as W


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, n: int, out_dir: str) -> None:
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = W.workload(4, ncells=n)
        start, count = sharding.rank_cell_range(n, rank)
        st = wl.make_state(device="cpu", cell_start=start, ncells=count)
        np.save(os.path.join(out_dir, f"erad_{rank}.npy"), st["Erad"].numpy())
        np.save(os.path.join(out_dir, f"mom_{rank}.npy"), st["mom"].numpy())
        slowest = sharding.max_over_ranks(1.0 + rank, dist)
        total = sharding.sum_over_ranks([count, rank], dist)
        assert slowest == float(world)
        assert total == [n * world, sum(range(world))]
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_rank_shards_match_single_process(tmp_path):
    n, world = 257, 2
    mp.spawn(_worker, args=(world, _free_port(), n, str(tmp_path)), nprocs=world, join=True)
    ref = W.workload(4, ncells=n * world).make_state(device="cpu")
    erad = np.concatenate([np.load(tmp_path / f"erad_{r}.npy") for r in range(world)], axis=1)
    mom = np.concatenate([np.load(tmp_path / f"mom_{r}.npy") for r in range(world)], axis=1)
    # same counter-based draws; torch's vectorised exp/log may differ in the last bit between a vector
    # body and a scalar tail, so compare to a few ulp rather than bit for bit
    np.testing.assert_allclose(erad, ref["Erad"].numpy(), rtol=1e-13, atol=0.0)
    np.testing.assert_allclose(mom, ref["mom"].numpy(), rtol=1e-13, atol=0.0)


def test_split_cells_covers_everything():
    for total, world in ((0, 1), (10, 3), (16777216, 8), (5, 8)):
        parts = sharding.split_cells(total, world)
        assert len(parts) == world and parts[0][0] == 0
        assert all(parts[i][0] + parts[i][1] == parts[i + 1][0] for i in range(world - 1))
        assert parts[-1][0] + parts[-1][1] == total
        sizes = [p[1] for p in parts]
        assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.split_cells(4, 0)
    assert sharding.rank_cell_range(100, 3) == (300, 100)
    assert sharding.max_over_ranks(2.5) == 2.5 and sharding.sum_over_ranks([1, 2]) == [1, 2]
