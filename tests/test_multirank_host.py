"""The N > 1 path on CPU: world_size-2 `gloo` processes (one process per GPU in production; here the host-side
logic only).  SURVEY.md 8(e): ONE seeded ensemble, interleaved index split, tables replicated, no data-path
collective; the only exchange is one all-reduce of (sum g, sum g^2, n) = 24 bytes, plus the reduction of bench.py's
timing (max) and counters (sum).  Oracle-free: the per-particle "results" are a deterministic function of the
initial state, which is all the split and the reduce can see."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

N_ENSEMBLE = 1001          # odd: the two shards have different sizes


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _fake_result(x0: np.ndarray):
    """stand-in for a trace: 'lost' flag and 'stop time' as fixed functions of the initial state"""
    lost = (np.abs(x0[3]) < 0.31 * np.abs(x0[3]).max()).astype(np.float64)
    tstop = 1e-3 * (0.1 + np.abs(np.sin(x0[1])))
    return lost, tstop


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2604_07617_b200 import sharding as S
    from paper_2604_07617_b200 import workloads as W
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = W.config(1, n=N_ENSEMBLE, with_nodes=False)          # the SAME ensemble on every rank
        idx = S.shard_indices(N_ENSEMBLE, rank, world)
        mine = S.shard_columns(cfg["x0"], rank, world)
        assert np.array_equal(mine, cfg["x0"][:, idx])
        lost, tstop = _fake_result(cfg["x0"])                      # decided on the whole ensemble, used per shard
        out = {}
        for name, g in (("lost", lost[idx]), ("tstop", tstop[idx])):
            out[name] = S.reduce_estimate(float(np.sum(g)), float(np.sum(g * g)), len(idx))
        t, c = S.reduce_timing(10.0 + 5.0 * rank, [100.0 * (rank + 1), 7.0, float(len(idx))])
        np.save(os.path.join(out_dir, f"idx_{rank}.npy"), idx)
        with open(os.path.join(out_dir, f"red_{rank}.json"), "w") as fh:
            json.dump(dict(lost=out["lost"], tstop=out["tstop"], t=t, c=c), fh)
    finally:
        dist.destroy_process_group()


def test_two_ranks_split_one_ensemble_and_reduce_24_bytes(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    from paper_2604_07617_b200 import sharding as S
    from paper_2604_07617_b200 import workloads as W
    idx = [np.load(tmp_path / f"idx_{r}.npy") for r in range(world)]
    # the shards partition the ensemble: disjoint, interleaved, union = everything
    assert np.array_equal(np.sort(np.concatenate(idx)), np.arange(N_ENSEMBLE))
    assert np.array_equal(idx[0], np.arange(0, N_ENSEMBLE, 2)) and np.array_equal(idx[1], np.arange(1, N_ENSEMBLE, 2))
    assert np.array_equal(S.gather_order(N_ENSEMBLE, world), np.concatenate(idx))
    red = [json.load(open(tmp_path / f"red_{r}.json")) for r in range(world)]
    assert red[0] == red[1]                                         # identical on every rank
    cfg = W.config(1, n=N_ENSEMBLE, with_nodes=False)
    lost, tstop = _fake_result(cfg["x0"])
    single = S.reduce_estimate(float(lost.sum()), float((lost * lost).sum()), N_ENSEMBLE)   # no process group here
    # the indicator's count is an integer: the sharded estimate equals the single-rank one bit for bit
    assert tuple(red[0]["lost"]) == single
    assert red[0]["lost"][2] == float(int(lost.sum())) and red[0]["lost"][4] == N_ENSEMBLE
    assert red[0]["lost"][0] == lost.sum() / N_ENSEMBLE
    # a floating-point g: same to rounding of the two partial sums
    s1 = S.reduce_estimate(float(tstop.sum()), float((tstop * tstop).sum()), N_ENSEMBLE)
    assert np.allclose(red[0]["tstop"], s1, rtol=1e-14)
    assert abs(s1[1] - tstop.std(ddof=1) / np.sqrt(N_ENSEMBLE)) <= 1e-12 * s1[1] * 50
    # timing: max over ranks; counters: sums
    assert red[0]["t"] == 15.0 and red[0]["c"] == [300.0, 14.0, float(N_ENSEMBLE)]


def test_single_rank_reduce_is_identity():
    from paper_2604_07617_b200 import sharding as S
    t, c = S.reduce_timing(3.5, [1, 2.5])
    assert t == 3.5 and c == [1.0, 2.5]
    assert S.reduce_estimate(3.0, 3.0, 12)[:3] == (0.25, np.sqrt((3.0 / 12 - 0.0625) / 11), 3.0)
    with pytest.raises(ValueError):
        S.shard_indices(10, 2, 2)


def test_bench_gpus_n_spawns_n_ranks_without_torchrun(tmp_path):
    """`python bench.py --gpus 2` (no torchrun) must itself start two rank processes with RANK / LOCAL_RANK /
    WORLD_SIZE / MASTER_* set; `--dry-run-ranks` makes every rank report its environment and exit before it
    touches a GPU."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-run-ranks"],
                       capture_output=True, text=True, timeout=120, env=env)
    assert r.returncode == 0, r.stderr[-500:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    ranks = sorted((l["rank"], l["local_rank"], l["world_size"]) for l in lines if "rank" in l)
    assert ranks == [(0, 0, 2), (1, 1, 2)]
    assert all(l["master_addr"] == "127.0.0.1" for l in lines)
    assert len({l["master_port"] for l in lines}) == 1
