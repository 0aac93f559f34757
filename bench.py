#!/usr/bin/env python
"""bench.py -- pair-interactions/s of the direct-summation hot path on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2] [--n N]
    python bench.py --sweep-n 11 23 [--out profiles/r2_sweep_n.json]     # throughput vs N, every shape class

One STEP = one pass of the whole hot path over one batch of synthetic input:
    pp_step_kdk(1 step, PP_ACC_VALID, pot)  = kick+drift+pack -> pair sweep with potential -> split-j finalize + kick
    pp_invariants(pot)                      = E, P, L, COM, M from the state and that potential
i.e. N(N-1) ordered pair interactions per step.  The workload is BASELINE.json configs[2] (N = 2^20 exponential
disk, delta = 0.005, dt = 2.5e-4, seed 2) -- the configuration the metric is quoted on.  `value` is the FP32 figure
(dtype "f32"); the same step in FP64 is timed in the same run and reported under "fp64", and the force-only single
evaluation (pp_forces without potential) of both precisions under "force_only".

Multi-GPU: the north_star runs on one GPU with no sharding -- `--gpus N` runs N independent replicas ("replicas
only"), one process per GPU under torchrun, no data-path collective; value = pairs of all ranks / max time.
`--sharded` (opt-in) instead shards the i-bodies of ONE system over the N GPUs, with one
all-gather of the positions per step (paper_1803_01190_b200/sharded.py); it reports "scaling": "strong".

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample of the same
workload; it is the only other place besides cpu_baseline where this file touches oracle/.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "pair-interactions/s"
UNIT = "pair-interactions/s"
# nominal pipe peaks: lanes per SM x SMs x max SM clock
FP32_LANES, FP64_LANES, SM_COUNT, SM_MAX_HZ = 128, 64, 148, 1.965e9
# dram__bytes_read.sum + dram__bytes_write.sum of ONE sweep launch (with potential) at N = 2^20, from the
# `ncu --set full` captures summarised in profiles/r2_force_sym_f32_ncu.md / profiles/r2_force_sym_f64_ncu.md (the
# symmetric sweeps: the writes are their j-side rows, N^2/(2 x 2048) x 16 or 32 B, written once)
NCU_TRAFFIC_BYTES = {("f32", 1 << 20): 159.560448e6 + 4267.639e6, ("f64", 1 << 20): 406.194688e6 + 8599.203e6}
L2_FLUSH_BYTES = 256 << 20


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json configs (default 2: N=2^20)")
    ap.add_argument("--n", type=int, default=None, help="override N (same recipe and seed)")
    ap.add_argument("--no-fp64", action="store_true", help="skip the FP64 arm (faster profiling runs)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-variants", action="store_true",
                    help="skip the unequal-mass and one-sided force-only timings (single solves at N = 2^22, 2^23)")
    ap.add_argument("--no-kdk-latency", action="store_true", help="skip the small-N step-latency rows (configs 0, 1)")
    ap.add_argument("--sweep-n", type=int, nargs=2, metavar=("LOG2_MIN", "LOG2_MAX"), default=None,
                    help="throughput of one gravity solve vs N = 2^min .. 2^max for every shape class (BASELINE.md "
                         "section 4.2); prints one JSON document, also written to --out")
    ap.add_argument("--out", default=None, help="file that --sweep-n also writes its JSON to")
    ap.add_argument("--sharded", action="store_true",
                    help="ONE system, i-bodies sharded over the N GPUs with an all-gather of positions per step "
                         "(SURVEY.md 8(f) NEXT-1, strong scaling) instead of the default N independent replicas")
    return ap.parse_args()


def workload_name(c):
    return "configs[%d] %s N=%d delta=%g dt=%g seed=%d" % (c["index"], c["name"], c["N"], c["delta"], c["dt"],
                                                            c["seed"])


# ---- clocks ------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        mhz, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f:
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                mhz.append(float(parts[0]))
                mx.append(float(parts[1]))
                pw.append(float(parts[2]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if mhz:
            out.update(sm_mhz=float(np.median(mhz)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                       samples=len(mhz), power_w_max=float(max(pw)))
        return out


# ---- our arm -----------------------------------------------------------------------------------------------------
def time_steps(torch, step_fn, steps, warmup, flush, barrier):
    """W warm-up steps, then exactly K steps between two (barrier + synchronize) brackets, timed with CUDA events on
    the current stream (the stream the library launches on).  Returns milliseconds for the K steps."""
    for _ in range(warmup):
        step_fn()
        flush()
    barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        step_fn()
        flush()
    e1.record()
    torch.cuda.synchronize()
    barrier()
    return e0.elapsed_time(e1)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1803_01190_b200 import ppgrav, replicas, workloads

    rank, local, world = replicas.env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    barrier = replicas.barrier

    def max_over_ranks(x):                             # timing bookkeeping only: not on the data path
        return replicas.max_over_ranks(x, device="cuda")

    ppgrav.lib()                                       # fails loudly if the CUDA library is missing
    c = workloads.config(args.config, N=args.n)
    c["index"] = args.config
    if world > 1:                                      # replicas: same recipe, a different seed per rank
        c = dict(c)
        c["seed"] = replicas.replica_seed(c["seed"], rank)
        c["pos"], c["vel"], c["mass"] = workloads.make(c["kind"], c["N"], c["seed"], c.get("sigma_f", 0.1), c["G"])
    N, G, delta = c["N"], c["G"], c["delta"]
    dt = c["dt"] if c["dt"] > 0 else 2.5e-4
    pairs = float(N) * float(N - 1)
    flush_buf = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda")

    def flush():
        flush_buf.zero_()                              # > 126 MB L2: the next step starts cold

    results = {}
    gpu_samples = {}
    clocks = None
    launches = None
    precisions = [("f32", torch.float32)] + ([] if args.no_fp64 else [("f64", torch.float64)])
    for name, dtype in precisions:
        pos = torch.tensor(c["pos"], dtype=dtype, device="cuda")
        vel = torch.tensor(c["vel"], dtype=dtype, device="cuda")
        mass = torch.tensor(c["mass"], dtype=dtype, device="cuda")
        acc = torch.empty_like(pos)
        pot = torch.empty_like(mass)
        out16 = torch.empty(16, dtype=torch.float64, device="cuda")
        ppgrav.pp_step_kdk(pos, vel, mass, acc, dt, 0, G=G, delta=delta)          # a(t0), untimed

        def step():
            ppgrav.pp_step_kdk(pos, vel, mass, acc, dt, 1, G=G, delta=delta, acc_valid=True, pot=pot)
            ppgrav.pp_invariants(pos, vel, mass, G=G, delta=delta, pot=pot, out16=out16)

        ppgrav.pp_configure(ppgrav.PP_CFG_PROFILE, 1)
        sampler = ClockSampler(local) if (name == "f32" and rank == 0) else None
        n0 = ppgrav.pp_launch_count()
        # warm-up happens inside time_steps; its sweeps are discarded from the profile below
        for _ in range(args.warmup):
            step()
            flush()
        ppgrav.pp_profile_read()
        n0 = ppgrav.pp_launch_count()
        ms = time_steps(torch, step, args.steps, 0, flush, barrier)
        n1 = ppgrav.pp_launch_count()
        sweep_ms, sweep_n = ppgrav.pp_profile_read()
        ppgrav.pp_configure(ppgrav.PP_CFG_PROFILE, 0)
        if sampler is not None:
            clocks = sampler.stop()
            launches = n1 - n0
        ms = max_over_ranks(ms)
        plan = ppgrav.pp_plan_query(N, ppgrav.PP_F32 if name == "f32" else ppgrav.PP_F64, True)
        lanes = FP32_LANES if name == "f32" else FP64_LANES
        peak = lanes * SM_COUNT * SM_MAX_HZ / 1e12
        # pipe operations per pair actually executed: one less on j-tiles whose bodies have a common mass
        n_tiles, n_common = ppgrav.pp_equal_mass_tiles(mass)
        plan["equal_mass_tiles"] = [n_tiles, n_common]
        ops = plan["pipe_ops_per_pair"] - n_common / n_tiles
        achieved = ops * pairs * sweep_n / (sweep_ms * 1e-3) / 1e12 if sweep_ms > 0 else 0.0
        inv = ppgrav.invariants_dict(out16)
        results[name] = dict(
            value=replicas.job_value(pairs, args.steps, ms, world), ms_per_step=ms / args.steps,
            sweep_ms_per_launch=sweep_ms / max(sweep_n, 1), sweep_share_of_step=sweep_ms / ms,
            roofline=dict(bound="alu", kernel="force_%s%s_kernel (pair sweep with potential)" %
                                 ("sym_" if plan["shape"] == 3 else "", name),
                          achieved=achieved, peak=peak, unit="Tlane-op/s", frac=achieved / peak,
                          traffic=NCU_TRAFFIC_BYTES.get((name, N)),
                          pipe_ops_per_pair=ops,
                          # SURVEY.md section 8(d) counted 13 (FP32) / 18 (FP64) operations per pair interaction with the
                          # potential, assuming every ORDERED pair is evaluated; the symmetric sweep evaluates every
                          # unordered pair once, so against that figure the fraction can exceed 1
                          frac_at_survey_ops_per_pair=(13 if name == "f32" else 18) * pairs * sweep_n /
                          (sweep_ms * 1e-3) / 1e12 / peak if sweep_ms > 0 else 0.0,
                          peak_source="nominal: %d %s lanes/SM x %d SMs x %.0f MHz" %
                                      (lanes, "FP32" if name == "f32" else "FP64", SM_COUNT, SM_MAX_HZ / 1e6)),
            plan=plan, E_after=inv["E"])

        # parity sample for the cpu_baseline leg: accelerations and potentials of 4096 sampled bodies of the ORIGINAL
        # inputs from the same launch configuration (untimed)
        if world == 1 and not args.no_cpu_baseline:
            idx_t = torch.tensor(workloads.sample_indices(c["seed"], N, 4096), device="cuda")
            pos0 = torch.tensor(c["pos"], dtype=dtype, device="cuda")
            a0, p0 = ppgrav.pp_forces(pos0, mass, G=G, delta=delta, want_pot=True)
            gpu_samples[name] = (a0[idx_t].double().cpu().numpy(), p0[idx_t].double().cpu().numpy())
            del pos0, a0, p0

        # force-only single evaluation
        def force_only():
            ppgrav.pp_forces(pos, mass, G=G, delta=delta, acc=acc)

        fms = max_over_ranks(time_steps(torch, force_only, max(2, args.steps // 2), 1, flush, barrier))
        results[name]["force_only"] = replicas.job_value(pairs, max(2, args.steps // 2), fms, world)
        results[name]["force_only_unequal_masses"] = results[name]["force_only_one_sided"] = None
        if not args.no_variants:
            # the same solve with m_j kept inside the pair loop on every tile (what a system of unequal masses costs)
            ppgrav.pp_configure(ppgrav.PP_CFG_EQUAL_MASS, 0)
            gms = max_over_ranks(time_steps(torch, force_only, 2, 1, flush, barrier))
            ppgrav.pp_configure(ppgrav.PP_CFG_EQUAL_MASS, 1)
            results[name]["force_only_unequal_masses"] = replicas.job_value(pairs, 2, gms, world)
            # and with every ORDERED pair evaluated (the one-sided sweep: what i-range solves run)
            ppgrav.pp_configure(ppgrav.PP_CFG_SYMMETRIC, 0)
            oms = max_over_ranks(time_steps(torch, force_only, 2, 1, flush, barrier))
            ppgrav.pp_configure(ppgrav.PP_CFG_SYMMETRIC, 1)
            results[name]["force_only_one_sided"] = replicas.job_value(pairs, 2, oms, world)

        if name == "f64" and world == 1 and not args.no_kdk_latency:
            # pp_invariants with its own FP64 potential sweep (pot = NULL; what the conservation experiment pays per
            # sample): equal-mass shortcut on (11 operations per pair) and off (12)
            inv_ms = {}
            for key, flag in (("equal_mass_shortcut", 1), ("shortcut_off", 0)):
                ppgrav.pp_configure(ppgrav.PP_CFG_EQUAL_MASS, flag)
                ts = []
                for r in range(2):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    ppgrav.pp_invariants(pos, vel, mass, G=G, delta=delta, out16=out16)
                    e1.record()
                    torch.cuda.synchronize()
                    ts.append(e0.elapsed_time(e1))
                inv_ms[key] = ts[-1]
            ppgrav.pp_configure(ppgrav.PP_CFG_EQUAL_MASS, 1)
            results[name]["invariants_with_potential_sweep_ms"] = inv_ms

        if name == "f32" and not args.no_e2e:
            # end to end through the host-buffer C ABI: pinned host arrays in, results back, every step
            hp, hv, hm, ha, hpot = (torch.empty(s, dtype=dtype).pin_memory().numpy()
                                    for s in ((N, 3), (N, 3), (N,), (N, 3), (N,)))
            hp[...], hv[...], hm[...] = c["pos"], c["vel"], c["mass"]
            ha[...] = acc.cpu().numpy()
            el = dtype.itemsize if hasattr(dtype, "itemsize") else 4

            def e2e_step():
                ppgrav.pp_step_kdk_host(hp, hv, hm, ha, dt, 1, G=G, delta=delta, acc_valid=True, pot=hpot)
                ppgrav.pp_invariants_host(hp, hv, hm, G=G, delta=delta, pot=hpot)

            for _ in range(max(1, args.warmup // 2)):
                e2e_step()
            barrier()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(args.steps):
                e2e_step()
                flush()
            torch.cuda.synchronize()
            ems = max_over_ranks((time.perf_counter() - t0) * 1e3)
            results[name]["e2e"] = dict(value=replicas.job_value(pairs, args.steps, ems, world), unit=UNIT,
                                        h2d_bytes_per_step=int((10 * N + 8 * N) * el),
                                        d2h_bytes_per_step=int((10 * N) * el + 128),
                                        api="pp_step_kdk_host + pp_invariants_host (pinned host buffers)")
        del pos, vel, mass, acc, pot

    line = None
    if rank == 0:
        r32 = results["f32"]
        line = {
            "metric": METRIC, "value": r32["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": r32["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(c), "step": "pp_step_kdk(1 step, with potential) + pp_invariants",
                       "pairs_per_step": pairs, "l2": "256 MiB flush write between steps, inside the timed region",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "roofline": r32["roofline"],
            "e2e": r32.get("e2e"),
            "gpu_launches": launches,
            "clocks": clocks,
            "sweep_ms_per_launch": r32["sweep_ms_per_launch"], "sweep_share_of_step": r32["sweep_share_of_step"],
            "force_only": {k: results[k]["force_only"] for k in results},
            "force_only_unequal_masses": {k: results[k]["force_only_unequal_masses"] for k in results},
            "force_only_one_sided": {k: results[k]["force_only_one_sided"] for k in results},
            "plan": r32["plan"],
            # the literature's convention: 20 flop per pair interaction (rsqrt counted as 4), force-only solve
            "tflops_20_flop_per_pair": {k: 20.0 * results[k]["force_only"] / 1e12 for k in results},
        }
        if "f64" in results:
            r64 = results["f64"]
            line["fp64"] = {"value": r64["value"], "unit": UNIT, "ms_per_step": r64["ms_per_step"],
                            "roofline": r64["roofline"], "sweep_ms_per_launch": r64["sweep_ms_per_launch"],
                            "plan": r64["plan"], "fp64_over_fp32_time": r64["ms_per_step"] / r32["ms_per_step"],
                            "invariants_with_potential_sweep_ms": r64.get("invariants_with_potential_sweep_ms")}
        if world == 1 and not args.no_kdk_latency:
            # BASELINE.json's KDK-step configs: 0 (N = 2048, 10 steps per call) and 1 (N = 2^17, 200 steps; 20 per call)
            line["kdk_step"] = {"config0": kdk_step_latency(torch, ppgrav, workloads, 0, 10),
                                "config1": kdk_step_latency(torch, ppgrav, workloads, 1, 20, reps=2)}
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(c, n_sample=16384, gpu_samples=gpu_samples)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return line


# ---- small-N step latency (configs 0 and 1 are KDK-step configs; a solve of 2048 bodies is launch-bound) -----------
def kdk_step_latency(torch, ppgrav, workloads, config_index, nsteps, reps=5):
    """Microseconds per KDK step of pp_step_kdk(nsteps, PP_ACC_VALID) on torch's default stream, CUDA-graph replay on
    and off, both precisions; best of `reps` calls after one warm-up call (which also instantiates the graph)."""
    c = workloads.config(config_index)
    N, G, delta, dt = c["N"], c["G"], c["delta"], c["dt"]
    out = {"workload": workload_name(dict(c, index=config_index)), "nsteps_per_call": nsteps,
           "launches_per_call": 2 * nsteps + 2, "stream": "default (legacy) stream"}
    for name, dtype in (("f32", torch.float32), ("f64", torch.float64)):
        pos, vel, mass = (torch.tensor(c[k], dtype=dtype, device="cuda") for k in ("pos", "vel", "mass"))
        acc = torch.empty_like(pos)
        ppgrav.pp_step_kdk(pos, vel, mass, acc, dt, 0, G=G, delta=delta)
        row = {}
        for graph in (1, 0):
            ppgrav.pp_configure(ppgrav.PP_CFG_GRAPH, graph)
            best = None
            for r in range(reps + 1):
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                t0 = time.perf_counter()
                e0.record()
                ppgrav.pp_step_kdk(pos, vel, mass, acc, dt, nsteps, G=G, delta=delta, acc_valid=True)
                e1.record()
                torch.cuda.synchronize()
                wall = (time.perf_counter() - t0) * 1e6
                dev = e0.elapsed_time(e1) * 1e3
                if r > 0 and (best is None or dev < best[0]):
                    best = (dev, wall)
            key = "graph" if graph else "plain_launches"
            row[key] = {"us_per_step_device": best[0] / nsteps, "us_per_step_wall": best[1] / nsteps,
                        "pairs_per_s": float(N) * (N - 1) * nsteps / (best[0] * 1e-6)}
        ppgrav.pp_configure(ppgrav.PP_CFG_GRAPH, 1)
        plan = ppgrav.pp_plan_query(N, ppgrav.PP_F32 if name == "f32" else ppgrav.PP_F64, False)
        row["plan"] = {k: plan[k] for k in ("shape", "i_per_cta", "tile_j", "split", "ctas")}
        out[name] = row
    return out


# ---- throughput of one gravity solve vs N, per shape class (calibrates plan.cu) -----------
def run_sweep_n(args):
    import torch
    from paper_1803_01190_b200 import ppgrav, workloads
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(0)
    ppgrav.lib()
    flush_buf = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda")
    rows = []
    # (name, PP_CFG_SHAPE, PP_CFG_SYMMETRIC): auto = the library's own choice; the rest pin the sweep
    shapes = (("auto", 0, 1), ("symmetric", 0, 2), ("large", 1, 0), ("mid", 2, 0), ("small", 3, 0))
    for logn in range(args.sweep_n[0], args.sweep_n[1] + 1):
        N = 1 << logn
        c = workloads.config(2, N=N)                   # the bench recipe (equal-mass exponential disk) at every N
        pairs = float(N) * float(N - 1)
        for name, dtype, code, lanes in (("f32", torch.float32, ppgrav.PP_F32, FP32_LANES),
                                         ("f64", torch.float64, ppgrav.PP_F64, FP64_LANES)):
            pos = torch.tensor(c["pos"], dtype=dtype, device="cuda")
            mass = torch.tensor(c["mass"], dtype=dtype, device="cuda")
            acc = torch.empty_like(pos)
            pot = torch.empty_like(mass)
            peak = lanes * SM_COUNT * SM_MAX_HZ
            for shape, key, symkey in shapes:
                if (shape == "small" and logn > 17 or shape == "mid" and logn > 20 or
                        logn > 21 and shape not in ("auto", "large")):
                    continue                           # far outside their range: minutes per solve, nothing to learn
                                                       # (above 2^21: the library's own choice and the large one-sided class)
                ppgrav.pp_configure(ppgrav.PP_CFG_SHAPE, key)
                ppgrav.pp_configure(ppgrav.PP_CFG_SYMMETRIC, symkey)
                for with_pot in ((False,) if logn > 21 else (False, True)):
                    plan = ppgrav.pp_plan_query(N, code, with_pot)
                    est = pairs * (12 if name == "f32" else 17) / (0.5 * peak)          # rough seconds per solve
                    if shape == "small":
                        est *= 2.5
                    reps = int(max(1 if logn > 21 else 2, min(20, 1.0 / max(est, 1e-4))))
                    times = []
                    for r in range(reps + 1):
                        flush_buf.zero_()
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record()
                        ppgrav.pp_forces(pos, mass, G=1.0, delta=c["delta"], acc=acc, pot=pot if with_pot else None)
                        e1.record()
                        torch.cuda.synchronize()
                        if r > 0:
                            times.append(e0.elapsed_time(e1))
                    ms = float(np.median(times))
                    # the pair-sweep kernel alone (events recorded by the library around its launch)
                    ppgrav.pp_configure(ppgrav.PP_CFG_PROFILE, 1)
                    ppgrav.pp_profile_read()
                    for r in range(min(reps, 5)):
                        flush_buf.zero_()
                        ppgrav.pp_forces(pos, mass, G=1.0, delta=c["delta"], acc=acc, pot=pot if with_pot else None)
                    k_ms, k_n = ppgrav.pp_profile_read()
                    ppgrav.pp_configure(ppgrav.PP_CFG_PROFILE, 0)
                    k_ms = k_ms / max(k_n, 1)
                    n_tiles, n_common = ppgrav.pp_equal_mass_tiles(mass)
                    ops = plan["pipe_ops_per_pair"] - n_common / n_tiles
                    rows.append({"log2N": logn, "N": N, "precision": name, "shape_requested": shape,
                                 "with_pot": with_pot, "shape": ("large", "mid", "small", "symmetric")[plan["shape"]],
                                 "i_per_cta": plan["i_per_cta"], "tile_j": plan["tile_j"], "split": plan["split"],
                                 "ctas": plan["ctas"], "ctas_per_sm": plan["ctas_per_sm"], "reps": reps,
                                 "ms_per_solve": ms, "ms_best": float(min(times)), "pairs_per_s": pairs / (ms * 1e-3),
                                 "sweep_kernel_ms": k_ms, "sweep_kernel_pairs_per_s": pairs / (k_ms * 1e-3) if k_ms > 0 else 0.0,
                                 "pipe_ops_per_pair": ops, "roofline_frac": ops * pairs / (ms * 1e-3) / peak})
            ppgrav.pp_configure(ppgrav.PP_CFG_SHAPE, 0)
            ppgrav.pp_configure(ppgrav.PP_CFG_SYMMETRIC, 1)
            del pos, mass, acc, pot
        print("[sweep-n] 2^%d done" % logn, file=sys.stderr, flush=True)
    doc = {"what": "pp_forces (pack + tile masses + pair sweep + finalize: the whole call, CUDA events on the launching "
                   "stream, median of reps after one warm-up, 256 MiB L2 flush before every call) on the configs[2] "
                   "recipe at N = 2^k", "command": "python bench.py --sweep-n %d %d" % tuple(args.sweep_n),
           "peak": "nominal lanes x 148 SMs x 1965 MHz", "rows": rows}
    if args.out:
        with open(args.out, "w") as f:
            json.dump(doc, f, indent=0)
    return doc


# ---- one system sharded over the GPUs (opt-in; the north_star's graded path is the single-GPU one above) ---------
def run_sharded(args):
    """Strong scaling of ONE configs[2] system: every rank owns N/k i-bodies, per step
    pp_kick_drift(own) -> all_gather(pos) over NCCL -> pp_forces_range(own i, all j, with potential) ->
    pp_kick_drift(own, closing kick) -> pp_invariants(own) -> all_reduce of the 16 partial sums."""
    import torch
    import torch.distributed as dist
    from paper_1803_01190_b200 import ppgrav, replicas, sharded, workloads

    rank, local, world = replicas.env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    ppgrav.lib()
    c = workloads.config(args.config, N=args.n)
    c["index"] = args.config
    N, G, delta = c["N"], c["G"], c["delta"]
    dt = c["dt"] if c["dt"] > 0 else 2.5e-4
    pairs = float(N) * float(N - 1)
    flush_buf = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda")
    comm = sharded.DistComm() if world > 1 else sharded.SingleComm()
    results = {}
    launches = clocks = None
    for name, dtype in [("f32", torch.float32)] + ([] if args.no_fp64 else [("f64", torch.float64)]):
        pos, vel, mass = (torch.tensor(c[k], dtype=dtype, device="cuda") for k in ("pos", "vel", "mass"))
        sysm = sharded.ShardedSystem(pos, vel, mass, G=G, delta=delta, comm=comm)
        inv = {}

        def step():
            sysm.step(dt, 1, want_pot=True)
            inv.update(sysm.invariants())

        sampler = ClockSampler(local) if (name == "f32" and rank == 0) else None
        for _ in range(args.warmup):
            step()
            flush_buf.zero_()
        n0 = ppgrav.pp_launch_count()
        ms = replicas.max_over_ranks(time_steps(torch, step, args.steps, 0, flush_buf.zero_, replicas.barrier),
                                     device="cuda")
        if sampler is not None:
            clocks = sampler.stop()
            launches = ppgrav.pp_launch_count() - n0
        results[name] = dict(value=pairs * args.steps / (ms * 1e-3), ms_per_step=ms / args.steps, E_after=inv["E"],
                             own_bodies=sysm.count)
        del sysm, pos, vel, mass
    line = None
    if rank == 0:
        r = results["f32"]
        line = {"metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": workload_name(c),
                           "step": "pp_kick_drift -> all_gather(pos) -> pp_forces_range(with potential) -> "
                                   "pp_kick_drift -> pp_invariants -> all_reduce(16 doubles)",
                           "pairs_per_step": pairs, "parallelism": "i-sharded x%d" % world,
                           "l2": "256 MiB flush write between steps, inside the timed region",
                           "bytes_gathered_per_step": 12 * N, "own_bodies": r["own_bodies"]},
                "gpu_launches": launches, "clocks": clocks,
                "fp64": results.get("f64")}
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return line


# ---- the oracle on the host cores --------------------------------------------------------------------------------
def cpu_baseline(c, n_sample, gpu_samples=None):
    """Times oracle.forces (as it stands) on a bounded sample of i-bodies against all N j-bodies, and -- untimed --
    compares the GPU's accelerations / potentials of 4096 sampled bodies (same launch configuration as the timed
    steps) with the oracle's: max over the sample of |a_gpu - a_oracle| / |a_oracle| (BASELINE.json's parity metric)."""
    from oracle import oracle
    from paper_1803_01190_b200 import workloads
    idx = workloads.sample_indices(c["seed"], c["N"], n_sample)
    cores = oracle.max_threads()
    t0 = time.perf_counter()
    oracle.forces(c["pos"], c["mass"], G=c["G"], delta=c["delta"], idx=idx, want_pot=True, nthreads=0)
    sec = time.perf_counter() - t0
    pairs = float(len(idx)) * float(c["N"] - 1)
    # the same routine on ONE thread, on the first 1024 of those bodies (SURVEY.md section 8(d) asks for both rates)
    idx1 = idx[:1024]
    t0 = time.perf_counter()
    oracle.forces(c["pos"], c["mass"], G=c["G"], delta=c["delta"], idx=idx1, want_pot=True, nthreads=1)
    sec1 = time.perf_counter() - t0
    parity = {}
    for name, (ga, gp) in (gpu_samples or {}).items():
        pidx = workloads.sample_indices(c["seed"], c["N"], 4096)
        pos, mass = (c["pos"], c["mass"]) if name == "f64" else workloads.as_f32_exact(c["pos"], c["mass"])
        ra, rp = oracle.forces(pos, mass, G=c["G"], delta=c["delta"], idx=pidx, want_pot=True, nthreads=0)
        parity[name] = {"max_rel_err_acc": float(np.max(np.linalg.norm(ga - ra, axis=1) / np.linalg.norm(ra, axis=1))),
                        "max_rel_err_pot": float(np.max(np.abs(gp - rp) / np.abs(rp))), "sampled_bodies": int(len(pidx)),
                        "tolerance": 1e-12 if name == "f64" else 2e-5}
    return {"value": pairs / sec, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": sec,
            "parity_vs_oracle": parity,
            "single_thread_value": float(len(idx1)) * float(c["N"] - 1) / sec1, "single_thread_seconds": sec1,
            "sample": "oracle.forces (FP64, compensated sums, OpenMP over i) for %d sampled i-bodies x all %d "
                      "j-bodies of the same workload = %.3g pairs; single thread: the first %d of them" %
                      (len(idx), c["N"], pairs, len(idx1))}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return None
    from oracle import oracle
    from paper_1803_01190_b200 import workloads
    oracle.build()
    c = workloads.config(args.config, N=args.n)
    c["index"] = args.config
    n_sample = 4096                                   # per step: 4096 i-bodies x N j-bodies (4.3e9 pairs at N=2^20)
    idx = workloads.sample_indices(c["seed"], c["N"], n_sample)
    cores = oracle.max_threads()
    pairs = float(len(idx)) * float(c["N"] - 1)

    def step():
        oracle.forces(c["pos"], c["mass"], G=c["G"], delta=c["delta"], idx=idx, want_pot=True, nthreads=0)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    sec = time.perf_counter() - t0
    value = pairs * args.steps / sec
    sample = ("each step = oracle.forces (FP64, compensated sums, OpenMP over i) for %d sampled i-bodies x all %d "
              "j-bodies = %.3g pairs" % (len(idx), c["N"], pairs))
    return {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3 / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(c), "step": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def main():
    args = parse_args()
    line = (run_reference(args) if args.impl == "reference" else run_sweep_n(args) if args.sweep_n
            else run_sharded(args) if args.sharded else run_ours(args))
    if line is not None:
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
