#!/usr/bin/env python
"""bench.py -- throughput of the CATAPULT hot path on B200 (contract: see the task statement).

    python bench.py --gpus 1 --steps K --warmup W                 # this library (CUDA, C-ABI)
    python bench.py --gpus N ...                                  # spawns N ranks itself (one per GPU)
    torchrun --nproc-per-node N ... bench.py --gpus N ...         # or under torchrun
    python bench.py --impl reference --steps K --warmup W         # the CPU oracle, timed as it stands

Workload (default cfg4 = BASELINE.json configs[4], the 10^6-particle config north_star's roofline target is quoted
on): 64^3-cell random-Fourier Boozer field + shear Alfven wave, 10^6 alphas per GPU.

WINDOW LEG (the timed K steps; `value`).  One "step" = one pass of the whole hot path over one batch: field build
(a1) -> DP5 tracing of the WHOLE ensemble across one time window of `--window` seconds (a2-a9) -> loss-fraction
estimate (a10).  Consecutive steps trace consecutive windows [j*w, (j+1)*w] of the same job with the state carried
on the device (catapult_trace_continue).  The metric (accepted DP5 steps per second) is intensive.

JOB LEG (`full_job`, the second half of BASELINE.json's metric: particles-to-T per second).  The ensemble traced from
t = 0 to the config's own T (1e-2 s) in ONE catapult_trace launch: the population thins as particles are lost and
the tail runs under-filled, so the job-level rate is what a user sees.  The default (`--job-particles -1`) is the
WHOLE ensemble, the config the metric is quoted on (cfg4: 10^6 particles, ~10 GPU-minutes, which dominates the run
time of the default command); `--job-particles 65536` is the quick form (slot efficiency 0.83 instead of 0.98, so
its particles-to-T/s is ~15 % lower), `--job-particles 0` skips the leg.

N > 1: ONE seeded ensemble of N x particles, split over the ranks by interleaved index, tables
replicated, no data-path collective; one 24-byte all-reduce of (sum g, sum g^2, n) gives the estimate.  Per-GPU work
is fixed as N grows ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import math
import os
import socket
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2604_07617_b200 import sharding as S  # noqa: E402
from paper_2604_07617_b200 import workloads as W  # noqa: E402

METRIC = "fp64 accepted DP5 steps/sec"
UNIT = "accepted steps/s"

# ---- the flop model, in ONE place (DESIGN.md section 7.1 quotes these numbers) ----------------------------------
# ALGORITHMIC work: per right-hand-side evaluation the tricubic contraction of m quantities at
# 84 FMA each (FMA = 2 flops), ~30 flops of Lagrange basis, and locate + right-hand side (sqrt / atan2 / sincos /
# exp / division = 1 flop each): ~100 (Boozer vacuum), ~150 (Boozer + wave), ~120 (Cartesian); per attempted step
# ~150 flops of stage / error algebra.  `roofline.achieved` and `roofline.frac` use these.
ALG_FLOPS_PER_EVAL = {"boozer_vac": 4 * 168 + 30 + 100, "boozer_saw": 4 * 168 + 30 + 150, "cart": 7 * 168 + 30 + 120}
# derivative-of-interpolant mode (R1c; not one of SURVEY 8(d)'s figures): value and gradient of ONE tricubic by
# the simultaneous value / derivative Horner scheme, 112 FMA, + locate and right-hand side as above
ALG_FLOPS_PER_EVAL.update({"boozer_vac_doi": 224 + 100, "boozer_saw_doi": 224 + 150})
ALG_FLOPS_PER_ATTEMPT = 150
# EXECUTED work of the tracer kernels (their own arithmetic: 63-FMA Horner per quantity in the monomial basis, no
# Lagrange basis; the scalar warp's and the stage sums' DFMA / DMUL / DADD per evaluation from the ncu instruction mix
# of the committed capture, profiles/r2_ncu_trace_pair.md: 391 DFMA + 75 DMUL + 22 DADD thread instructions per
# evaluation, lanes without a particle included).  `roofline.executed` uses these; stage algebra included.
EXEC_FLOPS_PER_EVAL = {"boozer_vac": 4 * 126 + 275, "boozer_saw": 4 * 126 + 375, "cart": 7 * 126 + 260}
EXEC_FLOPS_PER_EVAL.update({"boozer_vac_doi": 224 + 290, "boozer_saw_doi": 224 + 390})
# The part of the executed work that is known EXACTLY, without any capture: the contraction's 63 FMA per quantity
# (m quantities; derivative-of-interpolant mode: 112 FMA for value and gradient).  `roofline.contraction_only` uses
# these and leaves the scalar side out: a lower bound of the executed rate that no hand-entered constant enters.
# (`roofline.frac` stays the ALGORITHMIC figure: that is the bench contract's definition of `achieved`, SURVEY 8(d);
# the scalar-side constants of EXEC_FLOPS_PER_EVAL come from ONE capture of cfg4 and are not re-derived per build.)
CONTRACTION_FLOPS_PER_EVAL = {"boozer_vac": 4 * 126, "boozer_saw": 4 * 126, "cart": 7 * 126, "boozer_vac_doi": 224,
                              "boozer_saw_doi": 224}
# particle slots served by one thread block (tracer_pair.cu: two warp pairs; tracer.cu: one scalar warp)
SLOTS_PER_BLOCK = {"boozer_vac": 64, "boozer_saw": 64, "cart": 32, "boozer_vac_doi": 64, "boozer_saw_doi": 64}
BYTES_PER_CELL_VISIT = {"boozer_vac": 4 * 512, "boozer_saw": 4 * 512, "cart": 7 * 512, "boozer_vac_doi": 512, "boozer_saw_doi": 512}
KERNELS_PER_STEP = {"catapult_field_build": 1, "catapult_trace_continue": 1, "catapult_trace": 1, "catapult_estimate": 2}


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
    return dict(value=acc / dt, seconds=dt, accepted=acc, attempts=acc + int(r["nrej"].sum()), status=r["status"],
                cores=nthreads if nthreads > 0 else O.max_threads(),
                sample=f"first {x0.shape[1]} particles of {cfg['name']} over [0, {window:g}] s")


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


def spawn_ranks(args) -> int:
    """`python bench.py --gpus N` without torchrun: starts N rank processes (one per GPU) with the torchrun
    environment (RANK, LOCAL_RANK, WORLD_SIZE, MASTER_ADDR = 127.0.0.1, MASTER_PORT) and waits for them."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    procs = []
    for r in range(args.gpus):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(args.gpus), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), NCCL_DEBUG=os.environ.get("NCCL_DEBUG", "WARN"))
        procs.append(subprocess.Popen([sys.executable, os.path.abspath(__file__), *sys.argv[1:]], env=env))
    rc = 0
    for p in procs:
        rc = rc or p.wait()
    return rc


def committed_capture(model: str) -> dict:
    """Per-evaluation DRAM / L2 bytes of trace_kernel from the committed `ncu --set full` capture of this kernel
    (profiles/r2_traffic_pair.csv; the command is in the .md beside it).  bench.py does not run ncu: the traffic
    it reports is that capture's per-evaluation figure times the evaluations of its own timed launches."""
    out = {}
    for name in ("r2_traffic_pair.csv", "r3_traffic.csv"):   # boozer_saw (round 2); cart, boozer_vac (round 3)
        try:
            for line in open(os.path.join(ROOT, "profiles", name)):
                f = line.strip().split(",")
                if len(f) >= 3 and f[0] == model:
                    out[f[1]] = float(f[2])
        except Exception:
            pass
    return out


def measured_peaks() -> dict:
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=W.CONFIG_NAMES)
    ap.add_argument("--window", type=float, default=1e-5, help="seconds of physical time traced per step")
    ap.add_argument("--particles", type=int, default=0, help="particles per GPU (0 = the config's full size)")
    ap.add_argument("--cells", type=int, default=0, help="cells per dimension of the same field (0 = the config's grid): "
                    "the grid-resolution axis of the paper's sweeps (PAPER.md:100-102)")
    ap.add_argument("--derivative-of-interpolant", action="store_true", help="Boozer configs: tabulate |B| only (nquant = 1) and "
                    "take its derivatives from the interpolant (DESIGN.md R1c, SURVEY 8(f) f2): a quarter of the table")
    ap.add_argument("--rtol", type=float, default=0.0, help="tracing tolerance (0 = the config's 1e-9): PAPER.md:100-102")
    ap.add_argument("--e2e-steps", type=int, default=-1, help="steps of the host-buffer leg (-1 = --steps, 0 = skip)")
    ap.add_argument("--job-particles", type=int, default=-1,
                    help="particles of the full-T job leg (-1 = the whole ensemble, the config BASELINE.json's metric is "
                         "quoted on: ~10 min for cfg4's 10^6 particles; 65536 = a quick run; 0 = skip)")
    ap.add_argument("--job-T", type=float, default=0.0, help="end time of the job leg (0 = the config's own T)")
    ap.add_argument("--job-oracle", type=int, default=0, help="fidelity leg of the sweep (PAPER.md:98-102): the oracle traces "
                    "the first N particles of the job leg to the same end time; loss fractions and per-particle loss "
                    "flags are compared (0 = skip)")
    ap.add_argument("--cpu-particles", type=int, default=2048, help="oracle sample for cpu_baseline (0 = skip)")
    ap.add_argument("--ref-particles", type=int, default=2048, help="oracle sample of --impl reference: the same sample "
                    "as the cpu_baseline leg of the GPU arm (first N particles, [0, window])")
    ap.add_argument("--no-peaks", action="store_true")
    ap.add_argument("--dry-run-ranks", action="store_true", help="every rank prints its environment and exits")
    args = ap.parse_args()
    cfg_idx = W.CONFIG_NAMES.index(args.workload)
    if args.impl == "reference":
        run_reference(args, cfg_idx)
        return
    if args.gpus > 1 and "RANK" not in os.environ:
        sys.exit(spawn_ranks(args))
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.dry_run_ranks:
        print(json.dumps({"rank": rank, "local_rank": local, "world_size": world,
                          "master_addr": os.environ.get("MASTER_ADDR", "127.0.0.1"),
                          "master_port": os.environ.get("MASTER_PORT")}), flush=True)
        return

    import torch
    import torch.distributed as dist

    from paper_2604_07617_b200 import binding as K

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    K.load()
    launches = {"n": 0}

    def count(name):
        launches["n"] += KERNELS_PER_STEP[name]

    # ---- inputs: seeded, synthetic, resident in HBM before the timed region ---------------------
    per_gpu = args.particles if args.particles > 0 else W.FULL_N[cfg_idx]
    ncell = [args.cells] * 3 if args.cells > 0 else None
    cfg = W.config(cfg_idx, n=per_gpu * world, ncell=ncell)          # ONE ensemble of world x per_gpu particles
    if args.rtol > 0:
        cfg["params"]["rtol"] = args.rtol
    if args.derivative_of_interpolant:
        if cfg["field"]["coord"] != 0:
            raise SystemExit("--derivative-of-interpolant is a Boozer mode")
        cfg["field"] = dict(cfg["field"], nquant=1, nodes=np.ascontiguousarray(cfg["field"]["nodes"][:1]))
    fd, pd = cfg["field"], cfg["params"]
    model = model_of(cfg) + ("_doi" if args.derivative_of_interpolant else "")
    x0 = S.shard_columns(cfg["x0"], rank, world)                     # this rank's share: rank, rank + world, ...
    npart = x0.shape[1]
    d_nodes = torch.from_numpy(fd["nodes"]).cuda()
    d_x = torch.from_numpy(x0).cuda()
    field = K.catapult_field_build(fd, d_nodes)
    state = K.catapult_trace_init(field, pd, d_x.clone())
    torch.cuda.synchronize()
    table_bytes = field.table_bytes
    blocks, threads = K.catapult_trace_launch_shape(field, pd)
    field.destroy()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- window leg -----------------------------------------------------------------------------
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
            count("catapult_field_build"), count("catapult_trace_continue"), count("catapult_estimate")
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
    ms_all, red = S.reduce_timing(ms, [cnt[0], cnt[0] + cnt[1], cnt[6], cnt[7], cnt[8], cnt[9]], device="cuda")
    acc_all, att_all, evals_all, loads_all, blocking_all, rounds_all = red
    value = acc_all / (ms_all * 1e-3)
    e = est.cpu().numpy()
    loss_fraction, loss_se, n_lost, _, n_all = S.reduce_estimate(e[2], e[3], npart, device="cuda")   # the 24-byte reduce
    alive = int((state["status"] == 0).sum().item())

    # ---- roofline of the dominant kernel (trace_kernel), measured live with CUDA events ------------
    trace_s = sum(trace_ms) * 1e-3
    roof = None
    if rank == 0:
        peak_fp64 = l2_bw = None
        if not args.no_peaks:
            peak_fp64 = K.catapult_measure_fp64_peak()
            l2_bw = K.catapult_measure_l2_bandwidth(48 << 20)
        nominal = 148 * 64 * 2 * 1.965e9          # 64 DFMA/clk/SM at clocks.max.sm (B200_PROFILING.md)
        peak = (peak_fp64 or nominal) / 1e12
        alg = (cnt[6] * ALG_FLOPS_PER_EVAL[model] + (cnt[0] + cnt[1]) * ALG_FLOPS_PER_ATTEMPT) / trace_s / 1e12
        exe = cnt[6] * EXEC_FLOPS_PER_EVAL[model] / trace_s / 1e12
        cap = committed_capture(model)
        evals_per_launch = cnt[6] / max(1, args.steps)
        dram_b, l2_b = cap.get("dram_bytes_per_rhs_eval"), cap.get("l2_bytes_per_rhs_eval")
        roof = {"bound": "alu", "kernel": "trace_kernel" if model == "cart" else "trace_pair_kernel", "achieved": alg, "peak": peak, "unit": "TFLOP/s",
                "frac": alg / peak,
                "peak_source": "measured DFMA micro-benchmark (libcatapult_probe.so)" if peak_fp64 else
                "nominal 148 SM x 64 DFMA/clk x 1.965 GHz",
                "flops_per_rhs_eval": ALG_FLOPS_PER_EVAL[model], "flops_per_attempt": ALG_FLOPS_PER_ATTEMPT,
                "executed": {"achieved": exe, "frac": exe / peak, "flops_per_rhs_eval": EXEC_FLOPS_PER_EVAL[model],
                             "note": "the kernel's own arithmetic (63-FMA Horner per quantity, no Lagrange basis); the "
                                     "scalar-side constant is from one ncu capture of cfg4 (profiles/r2_ncu_trace_pair.md)"},
                "contraction_only": {"achieved": cnt[6] * CONTRACTION_FLOPS_PER_EVAL[model] / trace_s / 1e12,
                                     "frac": cnt[6] * CONTRACTION_FLOPS_PER_EVAL[model] / trace_s / 1e12 / peak,
                                     "flops_per_rhs_eval": CONTRACTION_FLOPS_PER_EVAL[model],
                                     "note": "exactly known flops of the tricubic contraction alone; locate, right-hand "
                                             "side and stage algebra excluded"},
                "traffic": dram_b * evals_per_launch if dram_b else None,
                "traffic_source": "profiles/r2_traffic_pair.csv / r3_traffic.csv (committed ncu --set full captures, bytes per evaluation) "
                                  "x the evaluations of one timed launch" if dram_b else None,
                "rhs_evals_per_launch": evals_per_launch,
                "launch_ms": sum(trace_ms) / max(1, len(trace_ms)),
                "trace_share_of_step": sum(trace_ms) / ms,
                "cell_fetches_per_rhs_eval": cnt[7] / max(1.0, cnt[6]),
                "blocking_fetches_per_rhs_eval": cnt[8] / max(1.0, cnt[6]),
                "slot_efficiency": cnt[6] / max(1.0, 32.0 * cnt[9]),
                "hbm": {"gbs": dram_b * cnt[6] / trace_s / 1e9 if dram_b else None, "peak_gbs": measured_peaks().get("hbm_gbs")},
                "l2": {"bytes_per_rhs_eval": l2_b, "algorithmic_bytes_per_rhs_eval":
                       BYTES_PER_CELL_VISIT[model] * cnt[7] / max(1.0, cnt[6]),
                       "gbs": l2_b * cnt[6] / trace_s / 1e9 if l2_b else None,
                       "peak_gbs": (l2_bw / 1e9) if l2_bw else None,
                       "frac": (l2_b * cnt[6] / trace_s / l2_bw) if (l2_b and l2_bw) else None}}

    # ---- end to end: HOST buffers, H2D + D2H inside the timed region, same windows continuing --------
    e2e = None
    e2e_steps = args.steps if args.e2e_steps < 0 else args.e2e_steps
    if e2e_steps > 0:
        f = K.catapult_field_build(fd, d_nodes)
        host = {}
        for k in ("x", "t", "dt", "mu", "status", "nacc", "nrej", "counters"):
            t = state[k]
            pin = torch.empty(t.shape, dtype=t.dtype, pin_memory=True)
            pin.copy_(t)
            host[k] = pin.numpy()
        host["nacc"] = host["nacc"].view(np.uint32)
        host["nrej"] = host["nrej"].view(np.uint32)
        host["counters"] = host["counters"].view(np.uint64)
        h2d = sum(host[k].nbytes for k in host)
        d2h = h2d
        barrier()
        j0 = args.warmup + args.steps
        K.catapult_trace_continue_host(f, dict(pd, T=(j0 + 1) * args.window), host)   # warm-up of the host path
        c0 = host["counters"].copy()
        barrier()
        t0 = time.perf_counter()
        for j in range(j0 + 1, j0 + 1 + e2e_steps):
            K.catapult_trace_continue_host(f, dict(pd, T=(j + 1) * args.window), host)
            _loss = float(np.mean(host["status"] == 1))      # the step's result, read on the host
        torch.cuda.synchronize()
        dt_e2e = time.perf_counter() - t0
        acc_e2e = float(host["counters"][0] - c0[0])
        dt_e2e, (acc_e2e,) = S.reduce_timing(dt_e2e, [acc_e2e], device="cuda")
        e2e = {"value": acc_e2e / dt_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "steps": e2e_steps, "ms_per_step": 1e3 * dt_e2e / e2e_steps,
               "api": "catapult_trace_continue_host (pinned host buffers)"}
        f.destroy()
        K.catapult_release_host_cache()

    # ---- job leg: t = 0 -> the config's T in ONE launch (population thins, tail under-filled) ----------
    job = None
    if args.job_particles != 0:
        nj = npart if args.job_particles < 0 else min(args.job_particles, npart)
        Tj = args.job_T if args.job_T > 0 else W.FULL_T[cfg_idx]
        f = K.catapult_field_build(fd, d_nodes)
        xj = d_x[:, :nj].contiguous()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g = K.catapult_trace(f, dict(pd, T=Tj), xj)
        e1.record()
        barrier()
        job_s = e0.elapsed_time(e1) * 1e-3
        c = g["counters"].cpu().numpy().astype(np.float64)
        ej = K.catapult_estimate(0, d_status=g["status"])
        job_s_all, (jacc, jatt, jev, jrounds, jn) = S.reduce_timing(job_s, [c[0], c[0] + c[1], c[6], c[9], nj], device="cuda")
        jloss = S.reduce_estimate(ej[2], ej[3], nj, device="cuda")
        ts = g["tstop"][g["status"] == 1].cpu().numpy()
        edges = Tj * np.array([0.0, 1e-3, 3e-3, 1e-2, 3e-2, 0.1, 0.3, 1.0])
        job = {"particles": int(jn), "T_s": Tj, "seconds": job_s_all,
               "particles_to_T_per_s": jn / job_s_all, "accepted_steps_per_s": jacc / job_s_all,
               "rhs_evals_per_s": jev / job_s_all, "loss_fraction": jloss[0], "loss_fraction_se": jloss[1],
               "rejected_share_of_attempts": 1.0 - jacc / max(1.0, jatt),
               "slot_efficiency": jev / max(1.0, 32.0 * jrounds),
               "resident_slots": SLOTS_PER_BLOCK[model] * blocks, "gpu_launches": KERNELS_PER_STEP["catapult_trace"],
               "loss_time_histogram": {"edges_s": edges.tolist(), "counts_rank0": np.histogram(ts, bins=edges)[0].tolist()},
               "note": "one catapult_trace launch from t = 0; slot_efficiency = evaluations / (32 x block rounds): the share "
                       "of slot-rounds doing useful work (idle lanes at refill and in the under-filled tail lower it)"}
        if rank == 0 and world == 1 and args.job_oracle > 0:
            # the CPU oracle on the first particles of the same job (same field, tolerance and end time): what the
            # paper's fidelity axis measures (loss fraction against cells per dimension and tolerance)
            no = min(args.job_oracle, nj)
            r = oracle_sample(dict(cfg, x0=cfg["x0"][:, :no]), Tj, no)
            lost_o = r["status"] == 1
            lost_g = (g["status"][:no] == 1).cpu().numpy()
            job["oracle"] = {"particles": no, "seconds": r["seconds"], "cores": r["cores"],
                             "loss_fraction_oracle": float(lost_o.mean()), "loss_fraction_gpu_same_particles": float(lost_g.mean()),
                             "loss_flags_agree": float((lost_o == lost_g).mean()),
                             "binomial_sigma": float(math.sqrt(max(lost_o.mean() * (1 - lost_o.mean()), 1e-12) / no))}
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
                       "l2_policy": f"inputs larger than L2 ({table_bytes >> 20} MiB tables, 126 MB L2)" if table_bytes > (126 << 20)
                       else "tables fit in L2 (resident by design)",
                       "launch": {"blocks": blocks, "threads": threads},
                       "parallelism": f"dp{world} (one ensemble of {npart * world} particles split by interleaved "
                                      "index, tables replicated, one 24-byte all-reduce of the estimate)"},
            "attempted_steps_per_s": att_all / (ms_all * 1e-3),
            "rhs_evals_per_s": evals_all / (ms_all * 1e-3),
            "particle_windows_per_s": world * npart * args.steps / (ms_all * 1e-3),
            "particles_to_T_per_s": job["particles_to_T_per_s"] if job else None,
            "loss_fraction_so_far": loss_fraction, "loss_fraction_se": loss_se, "particles_alive": alive,
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches["n"],
            "roofline": roof, "full_job": job, "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
