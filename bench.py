#!/usr/bin/env python
"""bench.py -- throughput of the zmc_scan hot path on B200 (driver contract in the task prompt).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl reference]

A "step" is one pass of the whole hot path (H1-H8: stage lists, decode, Philox, integrand, fp64
reduce, finalise, store) over one synthetic workload of BASELINE.json `configs` (default
configs[1] = cfg2; cfg5 streams its 80 GB of results to pinned host memory).  `value` is
integrand evaluations/s with device-resident outputs; `e2e` is the same metric through the C ABI
with HOST output buffers (list H2D and result D2H inside the timed region).  `roofline` is the
measured-dispatch-cost ALU bound of DESIGN.md section 6 ("bound": "alu"); `cpu_baseline` is the CPU oracle, as it
stands, on a bounded sample of the same workload.  With N > 1 (torchrun) the grid's first list is
lengthened N-fold and each rank scans its own contiguous flat range -- no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1910_01965_b200 import workloads as wl  # noqa: E402

METRIC = "integrand_evals_per_s"
UNIT = "evals/s"

# ALU roofline.  The loop is bound by the SM sub-partition's dispatch of half-width (16-lane)
# pipes, measured by `python -m paper_1910_01965_b200.pipe_rates` (profiles/r01_pipe_rates.txt): every integer
# instruction (IMAD.WIDE, LOP3, SHF, IADD3) costs 2 SMSP-cycles per warp, every FP32 instruction 1, and the two
# classes serialise on one port ("main"); FP64 instructions cost 2 on their own pipe, MUFU and F2F 8 each on the XU pipe.
# W_MIN[cfg] = max over those resources of the ALGORITHMIC instruction list of one evaluation (Philox4x32-10 with the
# t-only rounds hoisted = 16 IMAD.WIDE + 18 LOP3 per block, one bit-op per uniform (two for fp64), one FMA per
# dimension, the integrand's own arithmetic, F2F + 2 fp64 accumulate ops), in SMSP-cycles per warp = lane-cycles per
# thread.  (integer, FP32, FP64, XU) instructions per evaluation:
ALG_OPS = {
    "cfg1": (0.25 * 34 + 2 + 2, 0, 1 + 12 + 2, 0),        # fp64 sinpi(z) - K: 12 fp64 + 2 integer (sign); phase FMA; 2 accumulate
    "cfg2": (0.50 * 34 + 4 + 2, 0, 2 + 12 + 2, 0),
    "cfg3": (1.00 * 34 + 4, 4 + 4, 2, 3),                 # 4 FFMA; FADD+FMUL (exact reduction), FMUL.RZ, FADD (shift); FRND, MUFU.SIN, F2F
    "cfg4": (1.50 * 34 + 6, 12 + 1, 2, 2),                # 2 FFMA per dimension + FADD (shift); MUFU.EX2, F2F
    "cfg5": (0.75 * 34 + 3, 15 + 3, 2, 4),                # 15 FP32 of the integrand + reduction; FRND, MUFU.SIN, MUFU.EX2, F2F
    "eq4": (1.50 * 34 + 12 + 2, 0, 6 + 12 + 2, 0),        # paper Eq. (4), N = 6, fp64: one batch of Table 2
}
# Workloads that scan only part of their grid per step: the paper's Table 2 batch is 10^6 of the
# 10^8 grid points x 10^5 samples; its V100 "GPU evaluation time per batch" 18.19497 s = 5.50e9 evals/s is the one
# published number for exactly this workload, hence the one non-null vs_baseline.
ALG_OPS["cfg2_user"] = ALG_OPS["cfg2"]     # same method, same minimum; the generic user path executes more
SCAN_POINTS = {"eq4": 10**6}
# NEXT-3: the cfg2 inputs with the integrand handed over as a user body and compiled with NVRTC at run time
USER_BODIES = {"cfg2_user": ("cfg2", "return sin(x[0] * y[0] + x[1] * y[1]);")}
PUBLISHED_EVALS_PER_S = {"eq4": 1e6 * 1e5 / 18.19497}


def w_min(name):
    i, f, d, xu = ALG_OPS[name]
    res = {"main(int*2+fp32)": 2 * i + f, "fp64": 2 * d, "xu": 8 * xu, "issue": i + f + d + xu}
    bound = max(res, key=res.get)
    return res[bound], bound, res


SM_COUNT, LANES_PER_SM_CLK, SM_MAX_MHZ = 148, 128, 1965.0
PEAK_GLANE = SM_COUNT * LANES_PER_SM_CLK * SM_MAX_MHZ * 1e6 / 1e9      # 37 225 G lane-cycles/s


def build_workload(name: str, world: int):
    base = USER_BODIES[name][0] if name in USER_BODIES else name
    w = wl.paper_eq4() if base == "eq4" else wl.config(int(base[3:]))
    w.name = name
    if world > 1:       # weak scaling: N-fold longer first list, one contiguous shard per rank
        lo, hi = float(w.lists[0][0]), float(w.lists[0][-1])
        w.lists[0] = wl.linspace(lo, hi, len(w.lists[0]) * world)
    return w


class ClockSampler:
    """nvidia-smi clocks/throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.gpu), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm = [float(r[1]) for r in self.rows if len(r) >= 9 and r[1].replace(".", "").isdigit()]
        mx = [float(r[2]) for r in self.rows if len(r) >= 9 and r[2].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows if len(r) >= 9 for n, v in zip(names, r[5:9]) if v == "Active"})
        # the busiest half of the samples = under load (idle samples sit at the floor clock)
        load = sorted(sm)[len(sm) // 2:] if sm else []
        return {"sm_mhz": float(np.median(load)) if load else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def cpu_oracle_rate(w, seconds: float = 1.5):
    """The oracle as it stands on all host cores, on a bounded contiguous slice from the middle of the grid."""
    from oracle import zmc_oracle as orc
    if w.name in USER_BODIES:
        orc.set_user_integrand(USER_BODIES[w.name][1], w.N, w.M, len(w.consts))
        w.integrand_id = max(w.integrand_id, 1000)
    cores = os.cpu_count() or 1
    first = (w.G // 2 // 1000) * 1000
    probe = max(cores * 4, min(w.G - first, max(cores * 4, int(2e6 // w.n_samples))))
    t0 = time.perf_counter()
    rc, _, _ = orc.scan_workload(w, first, probe, n_threads=cores)
    dt = max(time.perf_counter() - t0, 1e-4)
    assert rc == 0
    pts = int(min(w.G - first, max(probe, probe * seconds / dt)))
    t0 = time.perf_counter()
    rc, _, _ = orc.scan_workload(w, first, pts, n_threads=cores)
    dt = time.perf_counter() - t0
    assert rc == 0
    return pts * w.n_samples / dt, cores, f"{pts} contiguous grid points from flat index {first} x {w.n_samples} samples"


def run_reference(args, rank: int):
    """--impl reference: the CPU oracle on the box's host cores (this tier has no reference code)."""
    if rank != 0:
        return
    w = build_workload(args.workload, 1)
    vals = []
    for i in range(args.warmup + args.steps):
        v, cores, sample = cpu_oracle_rate(w, seconds=1.0)
        if i >= args.warmup:
            vals.append(v)
    value = float(np.mean(vals))
    evals_per_step = value * 1.0
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * evals_per_step / value,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "grid_points": w.G, "n_samples": w.n_samples, "N": w.N, "M": w.M},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg2", choices=sorted(ALG_OPS))
    ap.add_argument("--impl", default="zmc", choices=["zmc", "reference"])
    ap.add_argument("--schedule", type=int, default=0, help="0 auto, 1 thread, 2 warp, 3 cta")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--adaptive", default="", help="n_first,n_max,target_stderr: also time zmc_scan_adaptive (N=1 only)")
    ap.add_argument("--farm-devices", default="", help="e.g. 0,1,2,3: also time zmc_scan_farm over these devices (N=1 only)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "zmc" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_1910_01965_b200 import binding as zb

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the zmc_scan hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    zb.load()

    w = build_workload(args.workload, world)
    if w.name in USER_BODIES:
        w.integrand_id = zb.zmc_register_integrand(w.name, USER_BODIES[w.name][1], w.N, w.M, len(w.consts))
    G_scan = SCAN_POINTS.get(w.name, w.G) * (world if w.name in SCAN_POINTS else 1)
    first, count = wl.shard_range(G_scan, rank, world)
    stream = torch.cuda.current_stream()
    out_dtype = torch.float32 if w.out_f32 else torch.float64
    elem = 4 if w.out_f32 else 8
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, warmup):
        """K steps, each bracketed by CUDA events on the launching stream, L2 flushed in between."""
        for _ in range(warmup):
            fn()
        barrier()
        total_ms, infos = 0.0, []
        for _ in range(steps):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            infos.append(fn())
            b.record(stream)
            b.synchronize()
            total_ms += a.elapsed_time(b)
        barrier()
        if world > 1:
            t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            total_ms = float(t.item())
        return total_ms, infos

    # ---- device-resident arm: `value` ---------------------------------------------------------------
    # cfg5's 80 GB of results cannot stay in HBM next to nothing else on every pool GPU; like every
    # config it is written to a device buffer here when that fits, else per-batch staging only (host arm).
    device_fits = count * elem * 2 <= 100e9
    if device_fits:
        d_mean = torch.empty(count, dtype=out_dtype, device="cuda")
        d_err = torch.empty(count, dtype=out_dtype, device="cuda")

        def step_dev():
            return zb.zmc_scan_ex(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, d_mean, d_err, stream,
                                  precision=w.precision, schedule=args.schedule, batch_points=w.batch_points,
                                  first_index=first, count=count, consts=w.consts, timing=True)
        sampler = ClockSampler(local_rank)
        sampler.start()
        total_ms, infos = timed(step_dev, args.steps, args.warmup)
        clocks = sampler.stop()
        kernel_ms = float(np.mean([i["kernel_ms"] for i in infos]))
        launches = int(sum(i["gpu_launches"] for i in infos))
        sched = infos[-1]["schedule"]
    else:
        raise SystemExit("workload does not fit the device-resident arm")

    ms_per_step = total_ms / args.steps
    evals_all = G_scan * w.n_samples                   # all ranks together
    value = evals_all / (ms_per_step * 1e-3)
    evals_rank = count * w.n_samples

    # ---- end-to-end arm: HOST (pinned) outputs, D2H inside the timed region ------------------------------
    e2e = None
    if not args.no_e2e:
        h_mean = torch.empty(count, dtype=out_dtype, pin_memory=True)
        h_err = torch.empty(count, dtype=out_dtype, pin_memory=True)
        bp = w.batch_points or max(1, min(count, 1 << 22))      # stream in batches so copies overlap compute

        def step_host():
            return zb.zmc_scan_ex(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, h_mean, h_err, stream,
                                  precision=w.precision, schedule=args.schedule, batch_points=bp,
                                  first_index=first, count=count, consts=w.consts, timing=True)
        e_steps = max(2, min(args.steps, 5))
        e_ms, e_infos = timed(step_host, e_steps, 1)
        e2e = {"value": evals_all / (e_ms / e_steps * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": int(e_infos[-1]["h2d_bytes"]) * world,
               "d2h_bytes_per_step": int(e_infos[-1]["d2h_bytes"]) * world,
               "ms_per_step": e_ms / e_steps,
               "kernel_ms": float(np.mean([i["kernel_ms"] for i in e_infos])),
               "d2h_ms": float(np.mean([i["d2h_ms"] for i in e_infos])),
               "exposed_d2h_ms": float(np.mean([i["exposed_d2h_ms"] for i in e_infos])),
               "n_batches": int(e_infos[-1]["n_batches"]),
               "d2h_gbs": float(np.mean([i["d2h_bytes"] / max(i["d2h_ms"], 1e-9) * 1e-6 for i in e_infos]))}
        launches += int(sum(i["gpu_launches"] for i in e_infos))

    # ---- NEXT-4: adaptive sample count; throughput counts the samples actually drawn (sum of out_n) -----------------
    adaptive = None
    if args.adaptive and world == 1:
        n_first, n_max, target = args.adaptive.split(",")
        n_first, n_max, target = int(n_first), int(n_max), float(target)
        a_n = torch.zeros(count, dtype=torch.int32, device="cuda")

        def step_adaptive():
            return zb.zmc_scan_adaptive(w.integrand_id, w.bounds, w.lists, n_first, n_max, target, w.seed, d_mean, d_err,
                                        a_n, stream, precision=w.precision, first_index=first, count=count,
                                        batch_points=w.batch_points, consts=w.consts, timing=True)
        a_ms, a_infos = timed(step_adaptive, 3, 2)
        drawn = int(a_n.to(torch.int64).sum().item())
        adaptive = {"n_first": n_first, "n_max": n_max, "target_stderr": target, "ms_per_step": a_ms / 3,
                    "samples_drawn": drawn, "value": drawn / (a_ms / 3 * 1e-3), "unit": UNIT,
                    "mean_n": drawn / count, "frac_at_n_max": float((a_n == n_max).float().mean().item()),
                    "fixed_n_max_evals": count * n_max}

    # ---- NEXT-2: the single-node batch farm over --farm-devices (host outputs, synchronous, host wall clock) -------
    farm = None
    if args.farm_devices and world == 1 and not args.no_e2e:
        devs = [int(d) for d in args.farm_devices.split(",")]
        f_ms = []
        for _ in range(3):
            tmf = zb.zmc_scan_farm(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, h_mean, h_err, devs,
                                   precision=w.precision, schedule=args.schedule, first_index=first, count=count,
                                   batch_points=w.batch_points, consts=w.consts)
            f_ms.append(tmf["wall_ms"])
        farm = {"devices": devs, "value": evals_all / (min(f_ms[1:]) * 1e-3), "unit": UNIT, "wall_ms": min(f_ms[1:]),
                "n_batches": tmf["n_batches"], "batches_done": tmf["batches_done"], "busy_ms": tmf["busy_ms"]}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    w_cyc, w_bound, w_res = w_min(w.name)
    achieved = w_cyc * evals_rank / (kernel_ms * 1e-3) / 1e9
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": (value / PUBLISHED_EVALS_PER_S[w.name] if w.name in PUBLISHED_EVALS_PER_S and world == 1 else None),
        "dtype": "f64" if w.precision == wl.PREC_F64 else "f32", "data": "synthetic",
        "config": {"workload": w.name, "grid_points": w.G, "scanned_points": G_scan, "n_samples": w.n_samples,
                   "N": w.N, "M": w.M, "evals_per_step": evals_all, "schedule": {1: "thread", 2: "warp", 3: "cta"}[sched],
                   "accumulate": "f64", "l2_flush_between_steps": True, "seed": w.seed,
                   "parallelism": f"index-range shards x{world}, no collective"},
        "points_per_s": G_scan / (ms_per_step * 1e-3),
        "kernel_ms_per_step": kernel_ms,
        "clocks": clocks,
        "e2e": e2e,
        "farm": farm,
        "adaptive": adaptive,
        "gpu_launches": launches,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": PEAK_GLANE, "unit": "G lane-cycles/s",
                     "frac": achieved / PEAK_GLANE, "traffic": None,
                     "lane_cycles_per_eval": w_cyc, "binding_resource": w_bound, "resources": w_res,
                     "measured_lane_cycles_per_eval": PEAK_GLANE * 1e9 * (clocks["sm_mhz"] or SM_MAX_MHZ) / SM_MAX_MHZ
                     / (evals_rank / (kernel_ms * 1e-3)),
                     "peak_source": "148 SMs x 4 SMSPs x 32 lanes x 1965 MHz dispatch; per-class costs measured by "
                                    "paper_1910_01965_b200.pipe_rates (profiles/r01_pipe_rates.txt), DESIGN.md section 6",
                     "frac_at_measured_clock": (achieved / (PEAK_GLANE * clocks["sm_mhz"] / SM_MAX_MHZ)
                                                if clocks.get("sm_mhz") else None)},
    }
    if not args.no_cpu_baseline and world == 1:
        v, cores, sample = cpu_oracle_rate(w)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
