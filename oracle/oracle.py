"""ctypes front-end of the CPU oracle (oracle/pp_oracle.cpp) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module.  It imports nothing from the CUDA package and the CUDA package imports nothing from here.

Every function takes and returns float64 numpy arrays (row-major [N,3] positions / velocities / accelerations,
[N] masses) and follows the paper's definitions cited in pp_oracle.cpp:
forces -> eq. (1)-(2) PAPER.md:41-48; kdk_paper -> eqs. (5)-(7) PAPER.md:67-92; invariants -> eqs. (8)-(10)
PAPER.md:148-156; surface_density -> the maps of Fig. 7, PAPER.md:180 (pinned in tests/test_oracle_density.py by a
hand example, mass conservation, numpy.histogram2d and the analytic exponential profile).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pp_oracle.cpp")
_LIB = os.path.join(_HERE, "libpp_oracle.so")

INVARIANT_NAMES = ("E", "K", "W", "Px", "Py", "Pz", "Lx", "Ly", "Lz", "Cx", "Cy", "Cz", "M")


def build(force=False):
    """Compile the oracle with g++ (no fast-math, no FMA contraction).  Returns the path of the .so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int64)
        i64, dbl, cint = ctypes.c_int64, ctypes.c_double, ctypes.c_int
        for name in ("oracle_forces", "oracle_forces_ld"):
            f = getattr(lib, name)
            f.argtypes = [dp, dp, i64, dbl, dbl, ip, i64, dp, dp, cint]
            f.restype = None
        for name in ("oracle_kdk_paper", "oracle_kdk_halfkick"):
            f = getattr(lib, name)
            f.argtypes = [dp, dp, dp, dp, i64, dbl, i64, dbl, dbl, cint, cint]
            f.restype = i64
        lib.oracle_invariants.argtypes = [dp, dp, dp, dp, i64, dbl, dbl, dp, cint]
        lib.oracle_invariants.restype = None
        lib.oracle_max_threads.argtypes = []
        lib.oracle_max_threads.restype = cint
        _lib = lib
    return _lib


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == shape, (a.shape, shape)
    return a


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def max_threads():
    return int(_load().oracle_max_threads())


def forces(pos, mass, G=1.0, delta=0.0, idx=None, want_pot=True, nthreads=1, long_double=False):
    """a_i (and Phi_i) for all particles, or for the particles in `idx`.  Returns (acc[n,3], pot[n] or None)."""
    lib = _load()
    pos = _f64(pos)
    N = pos.shape[0]
    pos = _f64(pos, (N, 3))
    mass = _f64(mass, (N,))
    if idx is None:
        n, ip = N, None
    else:
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        assert idx.ndim == 1 and (idx.size == 0 or (idx.min() >= 0 and idx.max() < N))
        n, ip = idx.size, idx.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))
    acc = np.zeros((n, 3), dtype=np.float64)
    pot = np.zeros((n,), dtype=np.float64) if want_pot else None
    fn = lib.oracle_forces_ld if long_double else lib.oracle_forces
    fn(_dp(pos), _dp(mass), N, float(G), float(delta), ip, n, _dp(acc), _dp(pot) if want_pot else None,
       int(nthreads))
    return acc, pot


def _kdk(fn, pos, vel, mass, acc, dt, nsteps, G, delta, nthreads):
    pos = _f64(pos).copy()
    N = pos.shape[0]
    vel = _f64(vel, (N, 3)).copy()
    mass = _f64(mass, (N,))
    acc_valid = acc is not None
    acc = _f64(acc, (N, 3)).copy() if acc_valid else np.zeros((N, 3), dtype=np.float64)
    nforce = fn(_dp(pos), _dp(vel), _dp(mass), _dp(acc), N, float(dt), int(nsteps), float(G), float(delta),
                int(acc_valid), int(nthreads))
    return pos, vel, acc, int(nforce)


def kdk_paper(pos, vel, mass, dt, nsteps, G=1.0, delta=0.0, acc=None, nthreads=1):
    """nsteps of eqs. (5)-(7) as printed.  Returns (pos, vel, acc, number_of_force_evaluations)."""
    return _kdk(_load().oracle_kdk_paper, pos, vel, mass, acc, dt, nsteps, G, delta, nthreads)


def kdk_halfkick(pos, vel, mass, dt, nsteps, G=1.0, delta=0.0, acc=None, nthreads=1):
    """Same scheme in half-kick / drift / half-kick form (must agree with kdk_paper to round-off)."""
    return _kdk(_load().oracle_kdk_halfkick, pos, vel, mass, acc, dt, nsteps, G, delta, nthreads)


def invariants(pos, vel, mass, G=1.0, delta=0.0, pot=None, nthreads=1):
    """dict of E, K, W, P, L, COM, M per eqs. (8)-(10) (W with the minus sign, j != i)."""
    pos = _f64(pos)
    N = pos.shape[0]
    vel = _f64(vel, (N, 3))
    mass = _f64(mass, (N,))
    out = np.zeros(16, dtype=np.float64)
    pp = None
    if pot is not None:
        pot = _f64(pot, (N,))
        pp = _dp(pot)
    _load().oracle_invariants(_dp(pos), _dp(vel), _dp(mass), pp, N, float(G), float(delta), _dp(out),
                              int(nthreads))
    d = {k: float(out[i]) for i, k in enumerate(INVARIANT_NAMES)}
    d["P"] = out[3:6].copy()
    d["L"] = out[6:9].copy()
    d["COM"] = out[9:12].copy()
    d["raw"] = out
    return d


def surface_density(pos, mass, x0, y0, cell, nx, ny):
    """Face-on surface-density map of Fig. 7: sigma[iy, ix] = (sum of m_i over the bodies with
    x0 + ix*cell <= x_i < x0 + (ix+1)*cell and y0 + iy*cell <= y_i < y0 + (iy+1)*cell) / cell^2, z ignored; bodies
    outside the nx x ny grid are dropped.  Plain loop over the bodies in index order, float64.  The cell index is
    floor((x - x0) * (1/cell)) evaluated in float64 -- the one place where floating point decides an integer."""
    pos = _f64(pos)
    mass = _f64(mass, (pos.shape[0],))
    inv = 1.0 / float(cell)
    sigma = np.zeros((int(ny), int(nx)), dtype=np.float64)
    for i in range(pos.shape[0]):
        ix = int(np.floor((pos[i, 0] - x0) * inv))
        iy = int(np.floor((pos[i, 1] - y0) * inv))
        if 0 <= ix < nx and 0 <= iy < ny:
            sigma[iy, ix] += mass[i]
    return sigma / (float(cell) * float(cell))
