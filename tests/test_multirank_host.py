"""The N > 1 path of bench.py on CPU: world_size-2 `gloo` processes (one process per GPU in production; here the
host-side logic only).  The path shards by particles with no data-path collective: every
rank traces its own seeded ensemble, and the only exchange is the reduction of the timing and the counters."""
import os
import socket
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    from paper_2604_07617_b200 import workloads as W
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # every rank draws its own ensemble of the same distribution (weak scaling)
        cfg = W.config(1, n=257, with_nodes=False, ensemble=rank)
        ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
        counts = [100.0 * (rank + 1), 7.0, float(cfg["x0"].shape[1])]
        t, c = bench.reduce_over_ranks(ms, counts, world, "cpu")
        np.save(os.path.join(out_dir, f"x0_{rank}.npy"), cfg["x0"])
        np.save(os.path.join(out_dir, f"red_{rank}.npy"), np.array([t] + c))
    finally:
        dist.destroy_process_group()


def test_two_ranks_reduce_and_own_ensembles(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    red = [np.load(tmp_path / f"red_{r}.npy") for r in range(world)]
    # time = max over ranks, counts = sums over ranks, identical on every rank
    assert np.array_equal(red[0], red[1])
    assert red[0][0] == 15.0 and red[0][1] == 300.0 and red[0][2] == 14.0 and red[0][3] == 2 * 257
    x = [np.load(tmp_path / f"x0_{r}.npy") for r in range(world)]
    assert x[0].shape == x[1].shape == (4, 257)
    assert not np.array_equal(x[0], x[1])                       # independent ensembles ...
    for r in range(world):                                      # ... that are reproducible
        from paper_2604_07617_b200 import workloads as W
        assert np.array_equal(x[r], W.config(1, n=257, with_nodes=False, ensemble=r)["x0"])
    # rank 0's ensemble is the single-GPU workload
    from paper_2604_07617_b200 import workloads as W
    assert np.array_equal(x[0], W.config(1, n=257, with_nodes=False)["x0"])


def test_single_rank_reduce_is_identity():
    import bench
    t, c = bench.reduce_over_ranks(3.5, [1, 2.5], 1, "cpu")
    assert t == 3.5 and c == [1.0, 2.5]
