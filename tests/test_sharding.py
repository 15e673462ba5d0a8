"""N > 1 host logic on CPU (gloo, world_size 2): history ranges tile the job exactly and the tally exchange is an
exact integer sum, so a sharded run equals the single-rank run bit for bit (checked here with the oracle as the
per-rank worker, since no GPU is present)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2605_25963_b200.sharding import allreduce_tallies, history_range

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_history_ranges_tile_exactly():
    for n, world, first in [(10, 3, 0), (0, 2, 5), (10 ** 8, 8, 7), (7, 8, 0), (1, 1, 99)]:
        nxt = first
        for r in range(world):
            s, c = history_range(n, r, world, first)
            assert s == nxt and c >= 0
            nxt = s + c
        assert nxt == first + n
    with pytest.raises(ValueError):
        history_range(5, 2, 2)


def _worker(rank, world, port, n, out_dir):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import detmesh as dm
    from oracle import gadep_oracle as orc
    os.environ["OMP_NUM_THREADS"] = "2"
    w = dm.make_config(0)
    s = orc.OracleScene(w)
    first, count = history_range(n, rank, world)
    spec, em, pk, _ = s.run(count, 1, first=first)
    t = torch.from_numpy(np.concatenate([spec, em, pk]).astype(np.int64))
    allreduce_tallies(t)
    if rank == 0:
        np.save(os.path.join(out_dir, "sum.npy"), t.numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharded_run_equals_single_rank(tmp_path):
    n, port = 300_000, 29000 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, n, str(tmp_path)), nprocs=2, join=True)
    got = np.load(tmp_path / "sum.npy")
    sys.path.insert(0, ROOT)
    import detmesh as dm
    from oracle import gadep_oracle as orc
    s = orc.OracleScene(dm.make_config(0))
    spec, em, pk, _ = s.run(n, 1)
    assert np.array_equal(got, np.concatenate([spec, em, pk]).astype(np.int64))
