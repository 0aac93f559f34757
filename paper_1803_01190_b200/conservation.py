"""Long-run conservation experiment: the paper's Table 2 / Figs. 5-6 on the built path.

PAPER.md:146-176: for N = 128k ... 1024k the authors integrate an equilibrium stellar disk for 10^4 steps in single and
in double precision and record max |dP|, max |dL|/L0, max |dE|/E0 (Table 2) and their time series
(Figs. 5-6).  Their initial conditions cannot be regenerated, so this runs the same protocol on
the synthetic Toomre-unstable exponential disk of BASELINE.json configs[2] (same recipe and seed, any N):

    python -m paper_1803_01190_b200.conservation --logn 17 --steps 10000 --sample-every 100 --out gpurun_out/x.json

The drift report of BASELINE.json's own KDK configs (0: 10 steps, 1: 200 steps, 2: 100 steps)
is the same loop on those workloads with their own dt and step counts:

    python -m paper_1803_01190_b200.conservation --drift-report --precision all --out profiles/r2_drift.json

Everything runs through the library: pp_step_kdk advances `sample_every` steps per call, pp_invariants evaluates
E, P, L, COM of the snapshot with its own O(N^2) FP64 potential pass on the (promoted) state, so the diagnostic is
equally accurate for both state precisions (reading R7) and FP32 drift is not masked by an FP32 potential.
Drift definitions: DESIGN.md reading R9.
"""
import argparse
import json
import time

import numpy as np


def run(logn, steps, dt, sample_every, precision, config_index=2, verbose=True, checkpoint=None, stop_after=None,
        n_bodies=None, ic="config"):
    """One run.  checkpoint: path of an .npz that is loaded if it exists (resume) and rewritten when the run stops;
    stop_after: stop (and checkpoint) after that many steps of THIS call, so that a long run can be cut into jobs.
    A resumed run continues bit for bit: pos and vel are stored in their own precision and a(t) is recomputed."""
    import os
    import torch
    from . import ppgrav, workloads

    N = int(n_bodies) if n_bodies is not None else 1 << logn
    logn = int(np.log2(N))
    c = workloads.config(config_index, N=N)
    G, delta = c["G"], c["delta"]
    if ic == "jeans":      # the equilibrium disk of eqs. (3)-(4) (disk_ic.py) instead of the config's recipe
        from . import disk_ic
        c["pos"], c["vel"], c["mass"] = disk_ic.make(N, c["seed"], G=G, delta=delta)
        c["name"] = "jeans_disk"
    dtype = torch.float32 if precision == "f32" else torch.float64
    mixed = precision == "mixed"                       # FP64 state, FP32 sweep (PP_MIXED)
    out16 = torch.empty(16, dtype=torch.float64, device="cuda")
    series, times = [], []
    done = 0
    wall_before = 0.0
    if checkpoint and not checkpoint.endswith(".npz"):
        checkpoint += ".npz"                            # np.savez appends it; resume must look for the same name
    if checkpoint and os.path.exists(checkpoint):
        z = np.load(checkpoint)
        have = (int(z["N"]), str(z["precision"]), float(z["dt"]))
        if have != (N, precision, dt):
            raise ValueError("checkpoint %s holds a run with (N, precision, dt) = %r, not %r: use one checkpoint file "
                             "per run" % (checkpoint, have, (N, precision, dt)))
        pos, vel = (torch.tensor(z[k], dtype=dtype, device="cuda") for k in ("pos", "vel"))
        mass = torch.tensor(c["mass"], dtype=dtype, device="cuda")
        acc = torch.empty_like(pos)       # not stored: the same force-only solve reproduces it bit for bit
        ppgrav.pp_step_kdk(pos, vel, mass, acc, dt, 0, G=G, delta=delta, mixed=mixed)
        series, times = [row for row in z["series"]], [float(t) for t in z["times"]]
        done, wall_before = int(z["done"]), float(z["wall"])
    else:
        pos, vel, mass = (torch.tensor(c[k], dtype=dtype, device="cuda") for k in ("pos", "vel", "mass"))
        acc = torch.empty_like(pos)
        ppgrav.pp_step_kdk(pos, vel, mass, acc, dt, 0, G=G, delta=delta, mixed=mixed)     # a(t0)

    def sample(t):
        ppgrav.pp_invariants(pos, vel, mass, G=G, delta=delta, pot=None, out16=out16)
        series.append(out16.cpu().numpy().copy())
        times.append(t)

    if not series:
        sample(0.0)
    t_wall = time.perf_counter()
    stop_at = steps if stop_after is None else min(steps, done + int(stop_after))
    while done < stop_at:
        n = min(sample_every, stop_at - done)
        ppgrav.pp_step_kdk(pos, vel, mass, acc, dt, n, G=G, delta=delta, acc_valid=True, mixed=mixed)
        done += n
        sample(done * dt)
        if verbose and (done // sample_every) % 10 == 0:
            s = np.array(series)
            print("[%s N=2^%d] step %d  dE/E0 %.3e  |dP| %.3e" % (precision, logn, done,
                  abs(s[-1, 0] - s[0, 0]) / abs(s[0, 0]), np.linalg.norm(s[-1, 3:6] - s[0, 3:6])), flush=True)
    torch.cuda.synchronize()
    wall = wall_before + time.perf_counter() - t_wall
    if checkpoint:
        tmp = checkpoint[:-4] + ".tmp.npz"              # written whole, then renamed: a killed job leaves the old file
        np.savez(tmp, N=N, precision=precision, dt=dt, done=done, wall=wall, pos=pos.cpu().numpy(),
                 vel=vel.cpu().numpy(), series=np.array(series), times=np.array(times))
        os.replace(tmp, checkpoint)
    s = np.array(series)
    E, P, L, C = s[:, 0], s[:, 3:6], s[:, 6:9], s[:, 9:12]
    drift = {
        "dE_over_E0_max": float(np.max(np.abs(E - E[0])) / abs(E[0])),
        "dP_abs_max": float(np.max(np.linalg.norm(P - P[0], axis=1))),
        "dLz_over_Lz0_max": float(np.max(np.abs(L[:, 2] - L[0, 2])) / abs(L[0, 2])),
        "dCOM_abs_max": float(np.max(np.linalg.norm(C - C[0], axis=1))),
        "two_K_over_W_first_last": [float(-2 * s[0, 1] / s[0, 2]), float(-2 * s[-1, 1] / s[-1, 2])],
        "two_K_over_W_min_max": [float(np.min(-2 * s[:, 1] / s[:, 2])), float(np.max(-2 * s[:, 1] / s[:, 2]))],
    }
    return {"N": N, "precision": precision, "config": config_index, "ic": ic, "steps": done, "dt": dt, "t_end": done * dt, "steps_requested": steps,
            "sample_every": sample_every, "workload": "configs[%d] recipe (%s), seed %d, delta %g" %
            (config_index, c["name"], c["seed"], delta), "wall_seconds": wall,
            "pairs_per_second_incl_diagnostics": float(N) * (N - 1) * done / max(wall, 1e-9), "drift": drift,
            "times": times, "E": E.tolist(), "P": P.tolist(), "Lz": L[:, 2].tolist(), "COM": C.tolist()}


# BASELINE.json's KDK configs and the reduced-N twins the oracle also integrates (tests/golden/oracle_drift.json)
DRIFT_REPORT = (
    # name, config, N (None = the config's), steps between samples
    ("config0", 0, None, 1),
    ("config1_N4096", 1, 4096, 50),
    ("config1", 1, None, 50),
    ("config2_N16384", 2, 16384, 25),
    ("config2", 2, None, 25),
)


def drift_report(precisions, verbose=True):
    from . import workloads
    runs = {}
    for name, k, n, every in DRIFT_REPORT:
        cfg = workloads.CONFIGS[k]
        for prec in precisions:
            r = run(0, cfg["nsteps"], cfg["dt"], every, prec, config_index=k, verbose=False,
                    n_bodies=n if n is not None else cfg["N"])
            r["name"] = name
            runs["%s_%s" % (name, prec)] = r
            if verbose:
                print(json.dumps({kk: r[kk] for kk in ("name", "N", "precision", "steps", "dt", "wall_seconds", "drift")}),
                      flush=True)
    return runs


def main():
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--logn", type=int, nargs="+", default=[17])
    ap.add_argument("--steps", type=int, default=10000)
    ap.add_argument("--dt", type=float, default=5e-4)
    ap.add_argument("--sample-every", type=int, default=100)
    ap.add_argument("--precision", default="both", choices=["f32", "f64", "mixed", "both", "all"],
                    help="both = f32 and f64 (the paper's SP and DP); all adds mixed (FP64 state, FP32 sweep)")
    ap.add_argument("--out", default=None)
    ap.add_argument("--checkpoint", default=None, help=".npz to resume from / write to (one --logn, one precision)")
    ap.add_argument("--stop-after", type=int, default=None, help="steps to run in this call before checkpointing")
    ap.add_argument("--ic", default="config", choices=["config", "jeans"],
                    help="initial conditions: the config's recipe, or the equilibrium disk of eqs. (3)-(4) (disk_ic.py)")
    ap.add_argument("--drift-report", action="store_true",
                    help="BASELINE.json configs 0, 1, 2 (and their reduced-N twins) with their own dt and step counts")
    a = ap.parse_args()
    if a.drift_report:
        precs = {"both": ("f32", "f64"), "all": ("f32", "mixed", "f64")}.get(a.precision, (a.precision,))
        runs = drift_report(precs)
        if a.out:
            with open(a.out, "w") as f:
                json.dump(runs, f, indent=0, sort_keys=True)
        return runs
    runs = []
    for logn in a.logn:
        for prec in {"both": ("f32", "f64"), "all": ("f32", "mixed", "f64")}.get(a.precision, (a.precision,)):
            r = run(logn, a.steps, a.dt, a.sample_every, prec, checkpoint=a.checkpoint, stop_after=a.stop_after,
                    ic=a.ic)
            print(json.dumps({k: r[k] for k in ("N", "precision", "steps", "dt", "wall_seconds", "drift")}), flush=True)
            runs.append(r)
            if a.out:                                   # rewritten after every run: a cut-off job keeps what finished
                with open(a.out, "w") as f:
                    json.dump(runs, f)
    return runs


if __name__ == "__main__":
    main()
