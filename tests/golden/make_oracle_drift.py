#!/usr/bin/env python
"""Writes tests/golden/oracle_drift.json: the CPU oracle's own kick-drift-kick runs of BASELINE.json configs 0-2.

    python tests/golden/make_oracle_drift.py [--only NAME ...] [--threads T] [--out FILE]

Calls ONLY oracle/ (kdk_halfkick, invariants: eqs. (5)-(10)) and the seeded input generators
(paper_1803_01190_b200/workloads.py, which holds none of the method's arithmetic).  Nothing here touches the CUDA path.
The stored values are what BASELINE.md's drift table prints in its "oracle" column and what
tests/test_gpu_fullsize.py compares the GPU trajectories with:

    config0        N = 2048 disk,            10 steps, dt = 1e-3     (BASELINE.json configs[0], full size)
    config1        N = 2^16 + 2^16 disk+halo, 200 steps, dt = 5e-4   (configs[1], FULL size: 3.5e12 pair interactions)
    config1_N4096  same recipe and seed at N = 4096                  (the reduced run the GPU tests repeat in full)
    config2_N16384 configs[2] recipe (Toomre-unstable disk) at N = 2^14, 100 steps, dt = 2.5e-4 -- the full-size
                   oracle run would be 1.1e14 pair interactions (6 core-days)

Per run: the invariants series (E, K, W, P, L, COM, M) at the sampled steps, the drifts of DESIGN.md reading R9, and
the final position / velocity of 256 bodies drawn from the config's "sample" stream (workloads.sample_indices), so a
GPU trajectory of the same inputs can be compared body by body without storing the whole state.
"""
import argparse
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
OUT = os.path.join(HERE, "oracle_drift.json")

RUNS = (
    # name, config index, N override, steps between samples, number of chunks
    ("config0", 0, None, 1, 10),
    ("config1_N4096", 1, 4096, 50, 4),
    ("config2_N16384", 2, 16384, 25, 4),
    ("config1", 1, None, 50, 4),
)
N_TRACK = 256


def drifts(series):
    s = np.asarray(series)
    E, P, Lz = s[:, 0], s[:, 3:6], s[:, 8]
    return {"dE_over_E0": float(np.max(np.abs(E - E[0])) / abs(E[0])),
            "dP_abs": float(np.max(np.linalg.norm(P - P[0], axis=1))),
            "dLz_over_Lz0": float(np.max(np.abs(Lz - Lz[0])) / abs(Lz[0]))}


def run_one(name, index, n_override, every, chunks, threads):
    from oracle import oracle
    from paper_1803_01190_b200 import workloads
    c = workloads.config(index, N=n_override)
    G, delta, dt = c["G"], c["delta"], c["dt"]
    pos, vel, mass = c["pos"], c["vel"], c["mass"]
    t0 = time.perf_counter()
    series = [oracle.invariants(pos, vel, mass, G=G, delta=delta, nthreads=threads)["raw"][:13].tolist()]
    steps = [0]
    acc = None
    nforce = 0
    for k in range(chunks):
        pos, vel, acc, nf = oracle.kdk_halfkick(pos, vel, mass, dt, every, G=G, delta=delta, acc=acc, nthreads=threads)
        nforce += nf
        series.append(oracle.invariants(pos, vel, mass, G=G, delta=delta, nthreads=threads)["raw"][:13].tolist())
        steps.append((k + 1) * every)
        print("[%s] step %d  %.0f s" % (name, steps[-1], time.perf_counter() - t0), flush=True)
    track = workloads.sample_indices(c["seed"], c["N"], N_TRACK)
    return {"config": index, "N": c["N"], "delta": delta, "dt": dt, "nsteps": steps[-1], "seed": c["seed"],
            "force_evaluations": nforce, "inputs": "float64 arrays of workloads.config(%d%s)" %
            (index, "" if n_override is None else ", N=%d" % n_override),
            "columns": ["E", "K", "W", "Px", "Py", "Pz", "Lx", "Ly", "Lz", "Cx", "Cy", "Cz", "M"],
            "steps": steps, "series": series, "drift": drifts(series),
            "track_index": track.tolist(), "track_pos": pos[track].tolist(), "track_vel": vel[track].tolist(),
            "max_abs_pos": float(np.abs(pos).max()), "max_abs_vel": float(np.abs(vel).max()),
            "cpu_seconds_wall": time.perf_counter() - t0, "threads": threads}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--only", nargs="*", default=None)
    ap.add_argument("--threads", type=int, default=0, help="OpenMP threads over i (0 = all); results do not depend on it")
    ap.add_argument("--out", default=OUT, help="JSON to update (default: tests/golden/oracle_drift.json); config1 takes "
                    "~30 min on 16 cores, so it may be written elsewhere on a bigger host and merged by re-running with "
                    "--merge")
    ap.add_argument("--merge", default=None, help="copy the runs of this JSON (written by this script) into --out")
    a = ap.parse_args()
    out = json.load(open(a.out)) if os.path.exists(a.out) else {}
    if a.merge:
        out.update(json.load(open(a.merge)))
        with open(a.out, "w") as f:
            json.dump(out, f, indent=0, sort_keys=True)
            f.write("\n")
        print("merged", sorted(out))
        return
    for name, index, n_override, every, chunks in RUNS:
        if a.only and name not in a.only:
            continue
        out[name] = run_one(name, index, n_override, every, chunks, a.threads)
        with open(a.out, "w") as f:
            json.dump(out, f, indent=0, sort_keys=True)
            f.write("\n")
    print("wrote", a.out)


if __name__ == "__main__":
    main()
