#!/usr/bin/env python
"""bench.py -- throughput of the CATAPULT hot path on B200 (contract: see the task statement).

    python bench.py --gpus 1 --steps K --warmup W                 # this library (CUDA, C-ABI)
    python bench.py --impl reference --steps K --warmup W         # the CPU oracle, timed as it stands
    torchrun --nproc-per-node N ... bench.py --gpus N ...         # N ranks, one ensemble per rank (weak)

Workload (default cfg4 = BASELINE.json configs[4], the 10^6-particle config north_star's roofline
target is quoted on): 64^3-cell random-Fourier Boozer field + shear Alfven wave, 10^6 alphas.
One "step" = one pass of the whole hot path over one batch: field build (a1) -> DP5 tracing of the
WHOLE ensemble across one time window of `--window` seconds (a2-a9) -> loss-fraction estimate (a10).
Consecutive steps trace consecutive windows [j*w, (j+1)*w] of the same job with the state carried on
the device (catapult_trace_continue), so K steps are K*w seconds of the T = 1e-2 s trace; the full
job is `--window 1e-2 --steps 1`.  The metric (accepted DP5 steps per second) is intensive.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2604_07617_b200 import workloads as W  # noqa: E402

METRIC = "fp64 accepted DP5 steps/sec"
UNIT = "accepted steps/s"

# Algorithmic FP64 work per right-hand-side evaluation: FMA = 2,
# add/mul = 1, division/sqrt/atan2/sincos/exp = 1 each.  Tricubic contraction 84 FMA per quantity.
FLOPS_PER_EVAL = {"boozer_vac": 4 * 168 + 39 + 30 + 46, "boozer_saw": 4 * 168 + 39 + 30 + 110,
                  "cart": 7 * 168 + 39 + 24 + 75}
FLOPS_STAGE_ALGEBRA_PER_ATTEMPT = 2 * 4 * (1 + 2 + 3 + 4 + 5 + 5) + 2 * 4 * 6 + 4 * 6 + 12
BYTES_PER_EVAL = {"boozer_vac": 4 * 512, "boozer_saw": 4 * 512, "cart": 7 * 512}


def model_of(cfg) -> str:
    if cfg["field"]["coord"] == 1:
        return "cart"
    return "boozer_saw" if cfg["params"]["saw_on"] else "boozer_vac"


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                parts = [p.strip() for p in line.split(",")]
                if len(parts) < 7:
                    continue
                try:
                    sm.append(float(parts[0]))
                    mx.append(float(parts[1]))
                except ValueError:
                    continue
                for nm, val in zip(names, parts[3:7]):
                    if val.lower().startswith("active"):
                        reasons.add(nm)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


# ------------------------------------------------------------------------------------------------
def oracle_sample(cfg, window: float, nsample: int, nthreads: int = 0) -> dict:
    """Times the CPU oracle, as it stands, on the first `nsample` particles of the workload over
    [0, window]: the reported CPU baseline (not the target)."""
    from oracle import catapult_oracle as O
    f = O.Field(cfg["field"])
    p = O.make_params(dict(cfg["params"], T=window))
    x0 = np.ascontiguousarray(cfg["x0"][:, :nsample])
    t0 = time.perf_counter()
    r = O.trace(f, p, x0, nthreads)
    dt = time.perf_counter() - t0
    acc = int(r["nacc"].sum())
    return dict(value=acc / dt, seconds=dt, accepted=acc, attempts=acc + int(r["nrej"].sum()),
                cores=nthreads if nthreads > 0 else O.max_threads(),
                sample=f"first {x0.shape[1]} particles of {cfg['name']} over [0, {window:g}] s")


def reduce_over_ranks(time_value: float, counts, world: int, device):
    """Whole-job figures of a weak-scaling run: the time is the MAX over ranks, every count the SUM over ranks
    (each rank traces its own ensemble; there is no data-path collective, only this).  Returns (time, [counts])."""
    if world <= 1:
        return float(time_value), [float(c) for c in counts]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(time_value)], dtype=torch.float64, device=device)
    c = torch.tensor([float(v) for v in counts], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), [float(v) for v in c.tolist()]


def run_reference(args, cfg_idx: int):
    """--impl reference: the oracle on the host cores (rank 0 only under torchrun)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = W.config(cfg_idx, n=args.ref_particles)
    vals, secs = [], []
    for i in range(args.warmup + args.steps):
        r = oracle_sample(cfg, args.window, args.ref_particles)
        if i >= args.warmup:
            vals.append(r["accepted"])
            secs.append(r["seconds"])
    tot_t = sum(secs)
    value = sum(vals) / tot_t
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "window_s": args.window,
                   "sample": f"first {args.ref_particles} particles per step, each step [0, window]"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=W.CONFIG_NAMES)
    ap.add_argument("--window", type=float, default=1e-5, help="seconds of physical time traced per step")
    ap.add_argument("--particles", type=int, default=0, help="override the particle count (0 = full size)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-particles", type=int, default=2048, help="oracle sample for cpu_baseline (0 = skip)")
    ap.add_argument("--ref-particles", type=int, default=1024)
    ap.add_argument("--no-peaks", action="store_true")
    ap.add_argument("--ncell", type=int, default=0,
                    help="cells per dimension instead of the workload's grid (0 = the workload's): a coarser grid "
                         "changes cells less often, which separates the cost of cell fetches from the rest")
    args = ap.parse_args()
    cfg_idx = W.CONFIG_NAMES.index(args.workload)
    if args.impl == "reference":
        run_reference(args, cfg_idx)
        return

    import torch
    import torch.distributed as dist

    from paper_2604_07617_b200 import binding as K

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    K.load()

    # ---- inputs: seeded, synthetic, resident in HBM before the timed region ---------------------
    n = args.particles if args.particles > 0 else None
    ncell = [args.ncell] * 3 if args.ncell > 0 else None
    cfg = W.config(cfg_idx, n=n, ncell=ncell, ensemble=rank)     # every rank traces its own ensemble (weak scaling)
    fd, pd = cfg["field"], cfg["params"]
    model = model_of(cfg)
    npart = cfg["x0"].shape[1]
    d_nodes = torch.from_numpy(fd["nodes"]).cuda()
    d_x = torch.from_numpy(cfg["x0"]).cuda()
    field = K.catapult_field_build(fd, d_nodes)
    state = K.catapult_trace_init(field, pd, d_x)
    torch.cuda.synchronize()
    table_bytes = field.table_bytes
    blocks, threads = K.catapult_trace_launch_shape(field, pd)
    field.destroy()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    trace_events = []

    def one_step(j: int, timed: bool):
        f = K.catapult_field_build(fd, d_nodes)                         # a1
        p = dict(pd, T=(j + 1) * args.window)
        if timed:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
        K.catapult_trace_continue(f, p, state)                          # a2-a9
        if timed:
            e1.record()
            trace_events.append((e0, e1))
        est = K.catapult_estimate(0, d_status=state["status"], to_host=False)   # a10
        return f, est

    fields = []
    for j in range(args.warmup):
        f, _ = one_step(j, False)
        fields.append(f)
    barrier()
    for f in fields:
        f.destroy()
    fields = []
    cnt0 = state["counters"].clone()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    est = None
    for j in range(args.warmup, args.warmup + args.steps):
        f, est = one_step(j, True)
        fields.append(f)        # destroyed after the timed region (cudaFree synchronises)
    ev1.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms = ev0.elapsed_time(ev1)
    trace_ms = [a.elapsed_time(b) for a, b in trace_events]
    for f in fields:
        f.destroy()
    cnt = (state["counters"] - cnt0).cpu().numpy().astype(np.float64)
    ms_all, (acc_all, att_all, evals_all) = reduce_over_ranks(ms, [cnt[0], cnt[0] + cnt[1], cnt[6]], world, "cuda")
    value = acc_all / (ms_all * 1e-3)
    loss_fraction = float(est[0].item())
    alive = int((state["status"] == 0).sum().item())

    # ---- roofline of the dominant kernel (trace_kernel), measured live with CUDA events ------------
    trace_s = sum(trace_ms) * 1e-3
    flops = cnt[6] * FLOPS_PER_EVAL[model] + (cnt[0] + cnt[1]) * FLOPS_STAGE_ALGEBRA_PER_ATTEMPT
    roof = None
    if rank == 0:
        peak_fp64 = l2_bw = None
        if not args.no_peaks:
            peak_fp64 = K.catapult_measure_fp64_peak()
            l2_bw = K.catapult_measure_l2_bandwidth(48 << 20)
        nominal = 148 * 64 * 2 * 1.965e9          # 64 DFMA/clk/SM at clocks.max.sm (B200_PROFILING.md)
        achieved = flops / trace_s / 1e12
        peak = (peak_fp64 or nominal) / 1e12
        alg_bytes = cnt[6] * BYTES_PER_EVAL[model]
        roof = {"bound": "alu", "kernel": "trace_kernel", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak,
                "peak_source": "measured DFMA micro-benchmark (catapult_measure_fp64_peak)" if peak_fp64 else
                "nominal 148 SM x 64 DFMA/clk x 1.965 GHz",
                "traffic": _ncu_traffic(model, cnt[6] / max(1, args.steps)),
                "flops_per_rhs_eval": FLOPS_PER_EVAL[model], "rhs_evals_per_launch": cnt[6] / max(1, args.steps),
                "launch_ms": sum(trace_ms) / max(1, len(trace_ms)),
                "trace_share_of_step": sum(trace_ms) / ms,
                "l2": {"algorithmic_bytes_per_rhs_eval": BYTES_PER_EVAL[model],
                       "achieved_gbs": alg_bytes / trace_s / 1e9,
                       "peak_gbs": (l2_bw / 1e9) if l2_bw else None,
                       "frac": (alg_bytes / trace_s / l2_bw) if l2_bw else None,
                       "note": "coefficient bytes touched per evaluation / measured L2 read bandwidth"},
                "hbm_peak_gbs": _measured_peaks().get("hbm_gbs")}

    # ---- end to end: HOST buffers, H2D + D2H inside the timed region, same windows continuing --------
    e2e = None
    if args.e2e_steps > 0:
        f = K.catapult_field_build(fd, d_nodes)
        host = {}
        for k in ("x", "t", "dt", "mu", "status", "nacc", "nrej", "counters"):
            t = state[k]
            dt_ = {torch.int32: torch.int32, torch.int64: torch.int64}.get(t.dtype, t.dtype)
            pin = torch.empty(t.shape, dtype=dt_, pin_memory=True)
            pin.copy_(t)
            host[k] = pin.numpy()
        host["nacc"] = host["nacc"].view(np.uint32)
        host["nrej"] = host["nrej"].view(np.uint32)
        host["counters"] = host["counters"].view(np.uint64)
        c0 = host["counters"].copy()
        h2d = sum(host[k].nbytes for k in host)
        d2h = h2d
        barrier()
        j0 = args.warmup + args.steps
        K.catapult_trace_continue_host(f, dict(pd, T=(j0 + 1) * args.window), host)   # warm-up of the host path
        c0 = host["counters"].copy()
        barrier()
        t0 = time.perf_counter()
        for j in range(j0 + 1, j0 + 1 + args.e2e_steps):
            K.catapult_trace_continue_host(f, dict(pd, T=(j + 1) * args.window), host)
            _loss = float(np.mean(host["status"] == 1))      # the step's result, read on the host
        torch.cuda.synchronize()
        dt_e2e = time.perf_counter() - t0
        acc_e2e = float(host["counters"][0] - c0[0])
        dt_e2e, (acc_e2e,) = reduce_over_ranks(dt_e2e, [acc_e2e], world, "cuda")
        e2e = {"value": acc_e2e / dt_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "steps": args.e2e_steps, "ms_per_step": 1e3 * dt_e2e / args.e2e_steps,
               "api": "catapult_trace_continue_host (pinned host buffers)"}
        f.destroy()

    # ---- CPU oracle beside it (rank 0, N = 1 only) ---------------------------------------------------
    cpu = None
    if rank == 0 and world == 1 and args.cpu_particles > 0:
        r = oracle_sample(W.config(cfg_idx, n=min(args.cpu_particles, npart), ncell=ncell), args.window,
                          args.cpu_particles)
        cpu = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"],
               "seconds": r["seconds"]}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_all / max(1, args.steps), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "particles_per_gpu": npart, "window_s": args.window,
                       "T_full_s": W.FULL_T[cfg_idx], "ncell": fd["ncell"], "model": model,
                       "rtol": pd["rtol"], "atol": pd["atol"], "table_bytes": table_bytes,
                       "l2_policy": "inputs larger than L2 (512 MiB tables, 126 MB L2)" if table_bytes > (126 << 20)
                       else "tables fit in L2 (resident by design)",
                       "launch": {"blocks": blocks, "threads": threads},
                       "parallelism": f"dp{world} (one ensemble per GPU, no data-path collective)"},
            "attempted_steps_per_s": att_all / (ms_all * 1e-3),
            "rhs_evals_per_s": evals_all / (ms_all * 1e-3),
            "particle_windows_per_s": world * npart * args.steps / (ms_all * 1e-3),
            "loss_fraction_so_far": loss_fraction, "particles_alive": alive,
            "clocks": clocks, "e2e": e2e, "gpu_launches": 4 * args.steps,
            "roofline": roof, "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def _ncu_traffic(model: str, evals_per_launch: float):
    """DRAM bytes of one trace launch: `dram__bytes_read.sum + dram__bytes_write.sum` per right-hand-side
    evaluation of the committed `ncu --set full` capture (profiles/r1_traffic_v5.md; cfg4 recipe) times the
    evaluations of one timed launch.  None for the models that were not captured."""
    if model != "boozer_saw":
        return None
    try:
        for line in open(os.path.join(ROOT, "profiles", "r1_traffic_v5.csv")):
            f = line.strip().split(",")
            if f[0] == "dram_bytes_per_rhs_eval":
                return float(f[1]) * evals_per_launch
    except Exception:
        pass
    return None


def _measured_peaks() -> dict:
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


if __name__ == "__main__":
    main()
