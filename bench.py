#!/usr/bin/env python
"""bench.py -- throughput of the zmc_scan hot path on B200 (driver contract in the task prompt).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--impl reference]

A "step" is one pass of the whole hot path (H1-H8: stage lists, decode, Philox, integrand, fp64 reduce, finalise,
store) over one synthetic workload of BASELINE.json `configs`.  The default workload is cfg5, the largest
single-GPU configuration (10^10 grid points x 256 samples): `value` is integrand
evaluations/s with the 80 GB of results device-resident, `e2e` the same scan through the C ABI with pinned HOST
outputs (list H2D forced, result D2H streamed in 2^28-point batches, `exposed_d2h_ms` = what compute did not hide).
`per_config_detail` carries the same record for cfg1-cfg4 (the north_star target is on cfg2-cfg4) and `per_config`, near
the end of the line, their headline numbers; `roofline.frac` is measured against the busiest physical unit (ncu-measured pipe occupancy per
instruction class), `frac_dispatch_model` the round-2 dispatch model, `frac_survey` SURVEY.md 8(d)'s own table; `pipe_rates` the
dispatch costs measured in this very run (bench_probe.py, its own libzmc_probe.so) that the ALU roofline is built from, `cpu_baseline`
the unoptimised CPU oracle on a bounded slice.  With N > 1 (torchrun) the grid's first list is lengthened N-fold and
each rank scans its own contiguous flat range -- no data-path collective.
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

# ALU roofline.  The loop is bound by the SM sub-partition's dispatch: every integer instruction
# (IMAD.WIDE, LOP3, SHF, IADD3) costs 2 SMSP-cycles per warp, every FP32 instruction 1, and the two classes serialise
# on one port ("main"); FP64 instructions cost 2 on their own pipe, MUFU and F2F 8 each on the XU pipe (`pipe_rates`
# in the output re-measures these on every run).  W_MIN[cfg] = max over those resources of the ALGORITHMIC instruction
# list of one evaluation (Philox4x32-10 with the t-only rounds hoisted = 16 IMAD.WIDE + 18 LOP3 per block, one bit-op
# per uniform (two for fp64), one FMA per dimension, the integrand's own arithmetic, F2F + 2 fp64 accumulate ops), in
# SMSP-cycles per warp = lane-cycles per thread.  (integer, FP32, FP64, XU) instructions per evaluation:
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
ALG_OPS["eq4_all"] = ALG_OPS["eq4"]        # the whole Table 2 experiment: all 10^8 grid points in the paper's 100 batches of 10^6
ALG_OPS["cfg2_user"] = ALG_OPS["cfg2"]     # same method, same minimum; the generic user path executes more
ALG_OPS["cfg2_user_libdevice"] = ALG_OPS["cfg2"]
SCAN_POINTS = {"eq4": 10**6}
# NEXT-3: the cfg2 inputs with the integrand handed over as a user body and compiled with NVRTC at run time
USER_BODIES = {"cfg2_user": ("cfg2", "return zmc_sin(x[0] * y[0] + x[1] * y[1]);"),
               "cfg2_user_libdevice": ("cfg2", "return sin(x[0] * y[0] + x[1] * y[1]);")}
# eq4_all: the paper's "total evaluation time" 721.20234 s for 10^8 points x 10^5 samples on its 3-node, 7-GPU cluster
# = 1.39e10 evals/s -- another machine's number for the same experiment: context
PUBLISHED_EVALS_PER_S = {"eq4": 1e6 * 1e5 / 18.19497, "eq4_all": 1e8 * 1e5 / 721.20234}
PER_CONFIG = ["cfg1", "cfg2", "cfg3", "cfg4"]
# roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum of the scan kernel, per launch, from the one
# `ncu --set full` capture of each kernel (profiles/r02_kernel.md).  cfg5: per 2^28-point batch launch (algorithmic:
# 2^28 x 8 B = 2.147e9 written); cfg4: 1e8 x 16 B = 1.6e9; cfg2: its 16 MB of results never leave L2 during the kernel.
NCU_TRAFFIC_BYTES = {"cfg5": 28.094464e6 + 2.096151e9, "cfg4": 37.298176e6 + 1.556428e9, "cfg2": 40.96e3 + 0.0}
NCU_TRAFFIC_SOURCE = "stored constant: one `ncu --set full` capture of this kernel (profiles/r02_kernel.md), NOT measured in this run"
# SURVEY.md 8(d) as written: I_min thread-instructions per evaluation and the IMAD.WIDE count per evaluation of its table
# (Philox with all 20 IMAD.WIDE per block), for `roofline.frac_survey` = max(I_min, 4 n_IMAD.WIDE) lane-cycles per evaluation:
# the issue bound (128 thread-instructions per clock per SM) or, by the survey's own sensitivity clause, the FMA-heavy pipe at
# 32 IMAD.WIDE per clock per SM (= 4 lane-cycles each; ncu shows 3.3-3.9 FMA-heavy cycles per instruction, profiles/r02_kernel.md section 3).
SURVEY_I_MIN = {"cfg1": (45.0, 5), "cfg2": (57.0, 10), "cfg3": (54.0, 20), "cfg4": (84.5, 30), "cfg5": (53.0, 15)}
IMAD_WIDE_LANE_CYCLES = 4.0


def w_min(name):
    i, f, d, xu = ALG_OPS[name]
    res = {"main(int*2+fp32)": 2 * i + f, "fp64": 2 * d, "xu": 8 * xu, "issue": i + f + d + xu}
    bound = max(res, key=res.get)
    # what the same list costs if FP64 / XU instructions do NOT hide behind the integer stream but take one dispatch
    # cycle each (what zmc_measure_pipes' "same warp" rows and every kernel of this library show on sm_100)
    return res[bound], bound, res, 2 * i + f + d + xu


# The PHYSICAL units, with the occupancy ncu reads for one warp-instruction of each class (profiles/r03_probe_ncu.md: each
# single-class probe kernel drives its pipe to 97-99.8 % busy at exactly these rates): IMAD.WIDE / IMAD.HI hold the
# FMA-heavy pipe 4 SMSP-cycles, FP32 instructions 1 cycle on FMA-heavy or FMA-lite (half each), LOP3 / SHF / IADD3 the ALU pipe
# 2 cycles, FP64 its pipe 2 cycles, MUFU / F2F the XU 8 cycles; every instruction takes one issue slot.  16 of a hoisted
# Philox block's 34 integer instructions are IMAD.WIDE.  Lane-cycles per evaluation on the busiest unit:
PHILOX_BLOCKS = {"cfg1": 0.25, "cfg2": 0.5, "cfg3": 1.0, "cfg4": 1.5, "cfg5": 0.75, "eq4": 1.5}


def pipe_bound(name):
    base = USER_BODIES[name][0] if name in USER_BODIES else ("eq4" if name.startswith("eq4") else name)
    i, f, d, xu = ALG_OPS[name]
    wide = 16.0 * PHILOX_BLOCKS[base]
    res = {"fma_heavy(4*IMAD.WIDE+fp32/2)": 4 * wide + f / 2, "alu(2*other int)": 2 * (i - wide), "fp64": 2 * d, "xu": 8 * xu,
           "issue": i + f + d + xu}
    bound = max(res, key=res.get)
    return res[bound], bound, res


SM_COUNT, LANES_PER_SM_CLK, SM_MAX_MHZ = 148, 128, 1965.0
PEAK_GLANE = SM_COUNT * LANES_PER_SM_CLK * SM_MAX_MHZ * 1e6 / 1e9      # 37 225 G lane-cycles/s


def build_workload(name: str, world: int):
    base = USER_BODIES[name][0] if name in USER_BODIES else name
    w = wl.paper_eq4() if base.startswith("eq4") else wl.config(int(base[3:]))
    w.name = name
    if name == "eq4_all":
        w.batch_points = 10 ** 6            # PAPER.md:132 "100 batches"
    if world > 1:       # weak scaling: N-fold longer first list, one contiguous shard per rank
        lo, hi = float(w.lists[0][0]), float(w.lists[0][-1])
        w.lists[0] = wl.linspace(lo, hi, len(w.lists[0]) * world)
    return w


def config_of(w, world: int):
    """The `config` object: the workload, identical for the zmc arm and the reference arm."""
    G_scan = SCAN_POINTS.get(w.name, w.G) * (world if w.name in SCAN_POINTS else 1)
    return {"workload": w.name, "grid_points": w.G, "scanned_points": G_scan, "n_samples": w.n_samples, "N": w.N, "M": w.M,
            "evals": G_scan * w.n_samples, "precision": "f64" if w.precision == wl.PREC_F64 else "f32 evaluate / f64 accumulate",
            "out_dtype": "f32" if w.out_f32 else "f64", "seed": w.seed, "schedule": "auto",
            "l2_flush_between_steps": True, "parallelism": f"index-range shards x{world}, no collective"}


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
            t0 = time.time()                 # wait for the first sample: nvidia-smi's start-up (NVML initialisation) must
            while not self.rows and time.time() - t0 < 3.0:      # not fall into a timed region that lasts milliseconds
                time.sleep(0.01)
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


def oracle_slice(w, n_threads: int, seconds: float, min_points: int):
    """Time the CPU oracle, as it stands, on a contiguous slice from the middle of the grid: at least `min_points` grid
    points and about `seconds` of work.  Returns (evals/s, seconds taken, points)."""
    from oracle import zmc_oracle as orc
    first = (w.G // 2 // 1000) * 1000
    avail = w.G - first
    probe = int(min(avail, max(n_threads * 4, 2e6 * n_threads / 16 // w.n_samples)))
    t0 = time.perf_counter()
    rc, _, _ = orc.scan_workload(w, first, probe, n_threads=n_threads)
    dt = max(time.perf_counter() - t0, 1e-4)
    assert rc == 0
    pts = int(min(avail, max(min_points, probe * seconds / dt)))
    t0 = time.perf_counter()
    rc, _, _ = orc.scan_workload(w, first, pts, n_threads=n_threads)
    dt = time.perf_counter() - t0
    assert rc == 0
    return pts * w.n_samples / dt, dt, pts, first


def cpu_baseline(w, seconds: float = 5.0, single_core: bool = True):
    """BASELINE.md "CPU-baseline plan": the oracle on all host cores and on one core, each on a slice of
    >= 10^5 grid points and >= `seconds` of work.  The oracle is deliberately plain (one Philox block per 32-bit word,
    two-pass long-double estimator): a reported baseline, not a tuned CPU implementation -- no speed-up is claimed."""
    from oracle import zmc_oracle as orc
    if w.name in USER_BODIES:
        orc.set_user_integrand(USER_BODIES[w.name][1], w.N, w.M, len(w.consts))
        w.integrand_id = max(w.integrand_id, 1000)
    cores = os.cpu_count() or 1
    min_pts = min(w.G // 2, 10 ** 5)
    v, dt, pts, first = oracle_slice(w, cores, seconds, min_pts)
    out = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle (unoptimised reference implementation)",
           "sample": f"{pts} contiguous grid points from flat index {first} x {w.n_samples} samples", "seconds": dt}
    if single_core:
        v1, dt1, pts1, _ = oracle_slice(w, 1, seconds, max(1, min_pts // cores))
        out["single_core"] = {"value": v1, "seconds": dt1, "points": pts1}
    return out


def run_reference(args, rank: int):
    """--impl reference: the CPU oracle on the box's host cores (this tier has no reference code).  Each step is one
    timed slice of the workload (>= 10^5 grid points, about 4 s of work); ms_per_step is that slice's real time."""
    if rank != 0:
        return
    from oracle import zmc_oracle as orc
    w = build_workload(args.workload, 1)
    if w.name in USER_BODIES:
        orc.set_user_integrand(USER_BODIES[w.name][1], w.N, w.M, len(w.consts))
        w.integrand_id = max(w.integrand_id, 1000)
    cores = os.cpu_count() or 1
    vals, secs, sample = [], [], ""
    budget = max(1.0, min(4.0, 150.0 / max(1, args.warmup + args.steps)))
    for i in range(args.warmup + args.steps):
        v, dt, pts, first = oracle_slice(w, cores, budget, min(w.G // 2, 10 ** 5))
        sample = f"{pts} contiguous grid points from flat index {first} x {w.n_samples} samples per step"
        if i >= args.warmup:
            vals.append(v)
            secs.append(dt)
    value = float(np.mean(vals))
    v1, dt1, pts1, _ = oracle_slice(w, 1, 3.0, max(1, min(w.G // 2, 10 ** 5) // cores))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(secs)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if w.precision == wl.PREC_F64 else "f32", "data": "synthetic",
        "config": config_of(w, 1),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle (unoptimised reference implementation)",
                         "sample": sample, "single_core": {"value": v1, "seconds": dt1, "points": pts1}},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg5", choices=sorted(ALG_OPS))
    ap.add_argument("--impl", default="zmc", choices=["zmc", "reference"])
    ap.add_argument("--schedule", type=int, default=0, help="0 auto, 1 thread, 2 warp, 3 cta")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the cfg1-cfg4 sub-records")
    ap.add_argument("--no-pipe-rates", action="store_true")
    ap.add_argument("--adaptive", default="", help="n_first,n_max,target_stderr: also time zmc_scan_adaptive (N=1 only)")
    ap.add_argument("--farm-devices", default="", help="e.g. 0,1,2,3: also time zmc_scan_farm over these devices (N=1 only; "
                    "default: all visible devices when there is more than one)")
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
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, warmup):
        """K steps, each bracketed by its own pair of CUDA events on the launching stream, L2 flushed in between (the
        flush is outside the brackets).  The host does not synchronise between steps unless the step itself does
        (timing=True): the queue stays full, so a bracket holds the step's device time, not the host's enqueue latency."""
        t0 = time.perf_counter()
        done = 0
        while done < warmup or time.perf_counter() - t0 < 0.25:      # at least W steps AND a quarter second of work: a
            fn()                                                      # 25-us step does not bring an idle GPU's clocks up
            done += 1
            if done % 64 == 0:
                torch.cuda.synchronize()
        barrier()
        infos, events = [], []
        for _ in range(steps):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            infos.append(fn())
            b.record(stream)
            events.append((a, b))
        barrier()
        total_ms = sum(a.elapsed_time(b) for a, b in events)

        if world > 1:
            t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            total_ms = float(t.item())
        return total_ms, infos

    def measure(name, steps, warmup, want_e2e, e2e_steps):
        """One workload: the device-resident arm (`value`), the HOST-output arm (`e2e`) and the roofline record."""
        w = build_workload(name, world)
        if w.name in USER_BODIES:
            w.integrand_id = zb.zmc_register_integrand(w.name, USER_BODIES[w.name][1], w.N, w.M, len(w.consts))
        cfg = config_of(w, world)
        G_scan = cfg["scanned_points"]
        first, count = wl.shard_range(G_scan, rank, world)
        out_dtype = torch.float32 if w.out_f32 else torch.float64
        elem = 4 if w.out_f32 else 8
        common = dict(precision=w.precision, schedule=args.schedule, first_index=first, count=count, consts=w.consts)
        shard_flags = zb.ZMC_OPT_EXPLICIT_COUNT if world > 1 else 0        # a rank's shard may be empty: count is meant literally

        # ---- device-resident arm: `value` (cfg5: its 80 GB of results fit a B200's 180 GB) ---------------------
        if count * elem * 2 > 120e9:
            raise SystemExit("workload does not fit the device-resident arm")
        d_mean = torch.empty(count, dtype=out_dtype, device="cuda")
        d_err = torch.empty(count, dtype=out_dtype, device="cuda")
        plan = zb.ScanPlan(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, d_mean, d_err,
                           batch_points=w.batch_points, flags=shard_flags, **common)
        # A step is the plain enqueue-only call a user makes.  For steps of a millisecond or more the library's own
        # per-kernel events ride along in the timed steps (timing=True: negligible there); for tiny grids (cfg1: 25 us)
        # that report's forced synchronisation would be most of the step, so the kernel time is taken in a second set of
        # steps, timed the same way, right after.
        plan(stream, timing=True)                   # first call: module load, list upload
        probe = plan(stream, timing=True)
        tiny = probe["kernel_ms"] < 1.0
        sampler = ClockSampler(local_rank)
        sampler.start()
        total_ms, infos = timed((lambda: plan(stream)) if tiny else (lambda: plan(stream, timing=True)), steps, warmup)
        if tiny:
            _, infos = timed(lambda: plan(stream, timing=True), min(steps, 10), 1)
        clocks = sampler.stop()
        kernel_ms = float(np.mean([i["kernel_ms"] for i in infos]))
        launches = int(probe["gpu_launches"]) * steps + (int(sum(i["gpu_launches"] for i in infos)) if tiny else 0)
        sched = infos[-1]["schedule"]
        ms_per_step = total_ms / steps
        evals_all = G_scan * w.n_samples                   # all ranks together
        evals_rank = count * w.n_samples

        adaptive = None
        if args.adaptive and world == 1 and name == args.workload:
            # NEXT-4: adaptive sample count; throughput counts the samples actually drawn (sum of out_n)
            n_first, n_max, target = args.adaptive.split(",")
            n_first, n_max, target = int(n_first), int(n_max), float(target)
            a_n = torch.zeros(count, dtype=torch.int32, device="cuda")

            def step_adaptive():
                return zb.zmc_scan_adaptive(w.integrand_id, w.bounds, w.lists, n_first, n_max, target, w.seed, d_mean, d_err,
                                            a_n, stream, precision=w.precision, first_index=first, count=count,
                                            batch_points=w.batch_points, consts=w.consts, timing=True)
            a_ms, _ = timed(step_adaptive, 3, 2)
            drawn = int(a_n.to(torch.int64).sum().item())
            adaptive = {"n_first": n_first, "n_max": n_max, "target_stderr": target, "ms_per_step": a_ms / 3,
                        "samples_drawn": drawn, "value": drawn / (a_ms / 3 * 1e-3), "unit": UNIT,
                        "mean_n": drawn / count, "frac_at_n_max": float((a_n == n_max).float().mean().item()),
                        "fixed_n_max_evals": count * n_max}
            del a_n
        del plan, d_mean, d_err
        torch.cuda.empty_cache()

        # ---- end-to-end arm: HOST (pinned) outputs, list H2D forced and result D2H inside the timed region -------
        e2e = farm = None
        if want_e2e:
            e_count = count if world == 1 else min(count, 1 << 31)       # bounded per rank when several ranks share one host
            t0 = time.perf_counter()
            while True:          # 80 GB of page-locked memory for cfg5: if this host cannot pin that much, scan (and say) less
                try:
                    h_mean = h_err = None
                    h_mean = zb.pinned_empty(e_count, out_dtype)
                    h_err = zb.pinned_empty(e_count, out_dtype)
                    break
                except (RuntimeError, MemoryError, OSError):
                    if e_count <= (1 << 28):
                        raise
                    e_count = max(1 << 28, e_count // 2)
            pin_s = time.perf_counter() - t0
            bp = w.batch_points or max(1, min(e_count, 1 << 22))      # stream in batches so copies overlap compute
            hplan = zb.ScanPlan(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, h_mean, h_err, batch_points=bp,
                                flags=zb.ZMC_OPT_FRESH_LISTS | shard_flags, **dict(common, count=e_count))
            if tiny:        # as in the device arm: the timing report's synchronisation would be most of a sub-millisecond step
                e2e_steps = max(e2e_steps, 10)
                e_ms, _ = timed(lambda: hplan(stream), e2e_steps, 1)
                _, e_infos = timed(lambda: hplan(stream, timing=True), min(e2e_steps, 3), 1)
            else:
                e_ms, e_infos = timed(lambda: hplan(stream, timing=True), e2e_steps, 1)
            e_evals_all = evals_all if e_count == count else e_count * w.n_samples * world
            e2e = {"value": e_evals_all / (e_ms / e2e_steps * 1e-3), "unit": UNIT,
                   "h2d_bytes_per_step": int(e_infos[-1]["h2d_bytes"]) * world,
                   "d2h_bytes_per_step": int(e_infos[-1]["d2h_bytes"]) * world,
                   "steps": e2e_steps, "ms_per_step": e_ms / e2e_steps,
                   "scanned_points_per_rank": e_count,
                   "kernel_ms": float(np.mean([i["kernel_ms"] for i in e_infos])),
                   "d2h_ms": float(np.mean([i["d2h_ms"] for i in e_infos])),
                   "exposed_d2h_ms": float(np.mean([i["exposed_d2h_ms"] for i in e_infos])),
                   "n_batches": int(e_infos[-1]["n_batches"]), "host_out_pinned": int(e_infos[-1]["host_out_pinned"]),
                   "pin_seconds_not_timed": pin_s,
                   # results written by the kernel itself (host_out_pinned == 2: small one-batch scans) have no copy to rate
                   "d2h_gbs": (float(np.mean([i["d2h_bytes"] / i["d2h_ms"] * 1e-6 for i in e_infos]))
                               if all(i["d2h_ms"] > 0 for i in e_infos) else None)}
            launches += int(sum(i["gpu_launches"] for i in e_infos)) + (int(e_infos[-1]["gpu_launches"]) * e2e_steps if tiny else 0)
            # ---- NEXT-2: the single-node batch farm (host outputs, synchronous, host wall clock) -------------------
            devs = [int(d) for d in args.farm_devices.split(",")] if args.farm_devices else \
                (list(range(torch.cuda.device_count())) if torch.cuda.device_count() > 1 else [])
            if devs and world == 1 and name == args.workload:
                f_count = min(e_count, 1 << 31)
                f_ms = []
                try:            # an extra record: a failure here (it has never run on more than one device) must not cost the line
                    for _ in range(3):
                        tmf = zb.zmc_scan_farm(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, h_mean[:f_count], h_err[:f_count],
                                               devs, precision=w.precision, schedule=args.schedule, first_index=first,
                                               count=f_count, batch_points=min(w.batch_points or f_count, max(1, f_count // (4 * len(devs)))),
                                               consts=w.consts)
                        f_ms.append(tmf["wall_ms"])
                    farm = {"devices": devs, "value": f_count * w.n_samples / (min(f_ms[1:]) * 1e-3), "unit": UNIT,
                            "wall_ms": min(f_ms[1:]), "scanned_points": f_count, "n_batches": tmf["n_batches"],
                            "batches_done": tmf["batches_done"], "busy_ms": tmf["busy_ms"]}
                except Exception as exc:        # noqa: BLE001 -- reported, not swallowed
                    farm = {"devices": devs, "error": f"{type(exc).__name__}: {exc}"}
                    torch.cuda.set_device(local_rank)
            del hplan, h_mean, h_err

        w_cyc, w_bound, w_res, w_add = w_min(w.name)
        rate = evals_rank / (kernel_ms * 1e-3)
        achieved = w_cyc * rate / 1e9
        pb_cyc, pb_bound, pb_res = pipe_bound(w.name)
        sv = SURVEY_I_MIN.get(USER_BODIES[w.name][0] if w.name in USER_BODIES else w.name)
        sv_cyc = max(sv[0], IMAD_WIDE_LANE_CYCLES * sv[1]) if sv else None
        return {
            "config": cfg, "w": w,
            "value": evals_all / (ms_per_step * 1e-3), "points_per_s": G_scan / (ms_per_step * 1e-3),
            "ms_per_step": ms_per_step, "kernel_ms_per_step": kernel_ms, "steps": steps, "warmup": warmup,
            "schedule_used": {1: "thread", 2: "warp", 3: "cta"}[sched], "clocks": clocks, "e2e": e2e, "farm": farm,
            "kernel_ms_from": "separate timed steps (library events force a sync)" if tiny else "the timed steps",
            "adaptive": adaptive, "gpu_launches": launches,
            # `frac` is the PHYSICAL-UNIT bound: algorithmic instruction counts x the pipe occupancy ncu measured per class, busiest
            # unit (round 3; rounds 1-2 headlined the dispatch model, kept as frac_dispatch_model: ncu shows the FMA-heavy pipe
            # only 82 % busy on a pure Philox block where that model claims the ceiling -- a fitted cost model, not a peak)
            "roofline": {"bound": "alu", "achieved": pb_cyc * rate / 1e9, "peak": PEAK_GLANE, "unit": "G lane-cycles/s",
                         "frac": pb_cyc * rate / 1e9 / PEAK_GLANE, "binding_unit": pb_bound, "unit_lane_cycles_per_eval": pb_res,
                         "frac_dispatch_model": achieved / PEAK_GLANE, "traffic": NCU_TRAFFIC_BYTES.get(w.name),
                         "traffic_source": NCU_TRAFFIC_SOURCE if w.name in NCU_TRAFFIC_BYTES else None,
                         # the same rate against SURVEY.md 8(d)'s own instruction table (see SURVEY_I_MIN above)
                         "frac_survey": sv_cyc * rate / 1e9 / PEAK_GLANE if sv else None,
                         "survey_lane_cycles_per_eval": sv_cyc,
                         "survey_binding": (None if not sv else "issue (I_min)" if sv[0] >= IMAD_WIDE_LANE_CYCLES * sv[1]
                                            else "FMA-heavy pipe (4 lane-cycles per IMAD.WIDE)"),
                         "lane_cycles_per_eval": w_cyc, "binding_resource": w_bound, "resources": w_res,
                         "measured_lane_cycles_per_eval": PEAK_GLANE * 1e9 * (clocks["sm_mhz"] or SM_MAX_MHZ) / SM_MAX_MHZ / rate,
                         "lane_cycles_per_eval_no_overlap": w_add, "frac_no_overlap": w_add * rate / 1e9 / PEAK_GLANE,
                         "peak_source": "peak = 148 SMs x 4 SMSPs x 32 lanes x 1965 MHz (sm_max_mhz of MEASURED_PEAKS.json; its HBM / bf16 "
                                        "figures do not apply: ALU-bound, no contraction). `frac`: algorithmic instruction list x per-class pipe "
                                        "occupancy measured with ncu (profiles/r03_probe_ncu.md), busiest physical unit. `frac_dispatch_model`: "
                                        "the builder's W_min (integer 2 + FP32 1 lane-cycles on one port; pipe_rates of this run; DESIGN.md "
                                        "section 6). `frac_survey`: SURVEY.md 8(d)'s own table, max(I_min, 4 x IMAD.WIDE)",
                         "frac_at_measured_clock": (pb_cyc * rate / 1e9 / (PEAK_GLANE * clocks["sm_mhz"] / SM_MAX_MHZ)
                                                    if clocks.get("sm_mhz") else None)},
        }

    main_rec = measure(args.workload, args.steps, args.warmup, not args.no_e2e, max(2, min(args.steps, 3)))
    per_config = {}
    if args.workload == "cfg5" and world == 1 and not args.no_per_config:
        for name in PER_CONFIG:
            r = measure(name, 10, 3, not args.no_e2e, 3)
            r.pop("w")
            per_config[name] = {k: r[k] for k in ("value", "points_per_s", "ms_per_step", "kernel_ms_per_step", "steps", "warmup",
                                                  "schedule_used", "kernel_ms_from", "clocks", "roofline", "e2e", "gpu_launches")}
            per_config[name]["grid_points"] = r["config"]["grid_points"]
            per_config[name]["n_samples"] = r["config"]["n_samples"]
    pipes = None
    if not args.no_pipe_rates and rank == 0:
        import bench_probe                       # a tool beside bench.py with its own libzmc_probe.so: not part of libzmc.so
        rep = bench_probe.measure_pipes(stream.cuda_stream)
        pipes = {"sm_mhz": round(rep["sm_mhz"], 1), "unit": "SMSP-cycles per group per warp: [measured, if independent pipes, if one shared pipe]",
                 "rows": {r["name"]: [round(r["cycles"], 2), round(r["parallel"], 2), round(r["serial"], 2)] for r in rep["rows"]}}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    w = main_rec.pop("w")
    launches = main_rec["gpu_launches"] + sum(p["gpu_launches"] for p in per_config.values())
    # Key order: the bulky records first, the contract keys after them, and a compact per-config table plus the CPU baseline
    # last -- whoever keeps only the tail of this line still sees every headline number.
    out = {
        "pipe_rates": pipes, "per_config_detail": per_config or None,
        "metric": METRIC, "value": main_rec["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": main_rec["ms_per_step"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": (main_rec["value"] / PUBLISHED_EVALS_PER_S[w.name] if w.name in PUBLISHED_EVALS_PER_S and world == 1 else None),
        "dtype": "f64" if w.precision == wl.PREC_F64 else "f32", "data": "synthetic",
        "config": main_rec["config"],
        "points_per_s": main_rec["points_per_s"], "kernel_ms_per_step": main_rec["kernel_ms_per_step"],
        "schedule_used": main_rec["schedule_used"], "clocks": main_rec["clocks"], "e2e": main_rec["e2e"],
        "farm": main_rec["farm"], "adaptive": main_rec["adaptive"], "gpu_launches": launches,
        "roofline": main_rec["roofline"],
    }
    if per_config:
        out["per_config"] = {"columns": ["evals_per_s", "kernel_ms", "roofline_frac", "frac_dispatch_model", "frac_survey", "e2e_evals_per_s"],
                             **{k: [float("%.4g" % v["value"]), round(v["kernel_ms_per_step"], 4), round(v["roofline"]["frac"], 3),
                                    round(v["roofline"]["frac_dispatch_model"], 3), round(v["roofline"]["frac_survey"], 3),
                                    float("%.4g" % v["e2e"]["value"]) if v["e2e"] else None]
                                for k, v in per_config.items()}}
    if not args.no_cpu_baseline and world == 1:
        out["cpu_baseline"] = cpu_baseline(w)
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
