"""Seeded synthetic workloads (numpy only).

These stand in for the paper's equilibrium stellar-disk initial conditions, which are
not reproducible from the paper (its iterative procedure lives in refs [1,15,18]).  Shapes and sizes follow
PAPER.md:127-138 (N = 128k ... 8192k) and BASELINE.json `configs`.  This module is the single source of inputs for
the CUDA path, the oracle, the tests and bench.py; it holds none of the method's arithmetic (no forces, no
integrator, no invariants) and imports neither oracle/ nor the CUDA binding.

Recipe:
* exponential disk: M_d = 1, h = 1, surface density ~ exp(-R/h)  =>  p(R) ~ R exp(-R/h): R = -h ln(u1 u2),
  redrawn while R > 4h; phi = 2 pi u; z = z0 atanh(2u - 1) (density ~ sech^2(z/z0), z0 = 0.1); equal masses.
  Velocities: circular speed v_c = sqrt(G M(<R)/R) with the spherical enclosed-mass estimate
  M(<R) = M_d [1 - (1 + R/h) e^{-R/h}] / [1 - 5 e^{-4}] (+ halo M_h R^3/(R^2+a^2)^{3/2}), tangential and
  counter-clockwise, plus Gaussian dispersion sigma = sigma_f v_c per cylindrical component.
* Plummer sphere (mass M, scale a): r = a (u^{-2/3} - 1)^{-1/2}, isotropic direction; speed
  v = q sqrt(2GM/a) (1 + r^2/a^2)^{-1/4} with q drawn by rejection from g(q) = q^2 (1 - q^2)^{7/2}; isotropic.
* disk + halo: disk particles first, halo second (two mass species); the halo DF ignores the disk potential.
* finally the mass-weighted mean position and velocity are subtracted (COM = 0, P = 0 to round-off).
Random numbers: numpy Philox (counter-based), key = (seed, stream id) -- one stream per quantity, so the output
does not depend on how the rejection loops batch their draws.
"""
import math

import numpy as np

_STREAMS = {"disk_R": 1, "disk_phi": 2, "disk_z": 3, "disk_vel": 4, "plummer_r": 5, "plummer_dir": 6,
            "plummer_q": 7, "plummer_vdir": 8, "sample": 9, "jeans_R": 10, "jeans_phi": 11, "jeans_z": 12,
            "jeans_vel": 13}

DISK_TRUNC = 4.0          # truncation radius in units of h
DISK_Z0 = 0.1


def _rng(seed, stream):
    return np.random.Generator(np.random.Philox(key=np.array([seed, _STREAMS[stream]], dtype=np.uint64)))


def _open01(rng, n):
    """Uniform in the open interval (0, 1)."""
    return (rng.integers(0, 1 << 53, size=n, dtype=np.uint64).astype(np.float64) + 0.5) * (2.0 ** -53)


def disk_enclosed_mass(R, h=1.0, M_d=1.0):
    """Mass of the truncated exponential disk inside cylindrical radius R."""
    norm = 1.0 - (1.0 + DISK_TRUNC) * math.exp(-DISK_TRUNC)
    x = np.minimum(R, DISK_TRUNC * h) / h
    return M_d * (1.0 - (1.0 + x) * np.exp(-x)) / norm


def plummer_enclosed_mass(r, M=1.0, a=1.0):
    return M * r ** 3 / (r * r + a * a) ** 1.5


def _isotropic(rng, n):
    cost = 2.0 * _open01(rng, n) - 1.0
    sint = np.sqrt(np.maximum(0.0, 1.0 - cost * cost))
    phi = 2.0 * math.pi * _open01(rng, n)
    return np.stack([sint * np.cos(phi), sint * np.sin(phi), cost], axis=1)


def exponential_disk(n, seed, G=1.0, h=1.0, M_d=1.0, z0=DISK_Z0, sigma_f=0.1, halo=None):
    """Positions, velocities, masses of an n-particle truncated exponential disk.

    halo = (M_h, a_h) adds a Plummer halo's enclosed mass to the circular speed."""
    rng = _rng(seed, "disk_R")
    R = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        r = -h * np.log(_open01(rng, todo.size) * _open01(rng, todo.size))
        ok = r <= DISK_TRUNC * h
        R[todo[ok]] = r[ok]
        todo = todo[~ok]
    phi = 2.0 * math.pi * _open01(_rng(seed, "disk_phi"), n)
    z = z0 * np.arctanh(2.0 * _open01(_rng(seed, "disk_z"), n) - 1.0)
    cphi, sphi = np.cos(phi), np.sin(phi)
    pos = np.stack([R * cphi, R * sphi, z], axis=1)

    M_enc = disk_enclosed_mass(R, h, M_d)
    if halo is not None:
        M_enc = M_enc + plummer_enclosed_mass(R, halo[0], halo[1])
    vc = np.sqrt(G * M_enc / R)
    g = _rng(seed, "disk_vel").standard_normal((n, 3))
    sigma = sigma_f * vc
    vR = sigma * g[:, 0]
    vphi = vc + sigma * g[:, 1]
    vz = sigma * g[:, 2]
    vel = np.stack([vR * cphi - vphi * sphi, vR * sphi + vphi * cphi, vz], axis=1)
    mass = np.full(n, M_d / n)
    return pos, vel, mass


def plummer_sphere(n, seed, G=1.0, M=1.0, a=1.0):
    """Positions, velocities, masses of an n-particle Plummer sphere drawn from its isotropic DF."""
    u = _open01(_rng(seed, "plummer_r"), n)
    r = a / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
    pos = r[:, None] * _isotropic(_rng(seed, "plummer_dir"), n)
    rng = _rng(seed, "plummer_q")
    q = np.empty(n)
    todo = np.arange(n)
    gmax = 0.1                       # > max of q^2 (1-q^2)^3.5 = 0.09245 at q^2 = 2/9
    while todo.size:
        qq = _open01(rng, todo.size)
        yy = gmax * _open01(rng, todo.size)
        ok = yy < qq * qq * (1.0 - qq * qq) ** 3.5
        q[todo[ok]] = qq[ok]
        todo = todo[~ok]
    speed = q * math.sqrt(2.0 * G * M / a) * (1.0 + (r / a) ** 2) ** -0.25
    vel = speed[:, None] * _isotropic(_rng(seed, "plummer_vdir"), n)
    mass = np.full(n, M / n)
    return pos, vel, mass


def _recentre(pos, vel, mass):
    m = mass.astype(np.longdouble)
    M = m.sum()
    for arr in (pos, vel):
        c = (m[:, None] * arr.astype(np.longdouble)).sum(axis=0) / M
        arr -= c.astype(np.float64)
    return pos, vel, mass


def disk_plus_halo(n_disk, n_halo, seed, G=1.0, halo_mass=4.0, halo_a=2.0, sigma_f=0.1):
    pd, vd, md = exponential_disk(n_disk, seed, G=G, sigma_f=sigma_f, halo=(halo_mass, halo_a))
    ph, vh, mh = plummer_sphere(n_halo, seed, G=G, M=halo_mass, a=halo_a)
    return np.concatenate([pd, ph]), np.concatenate([vd, vh]), np.concatenate([md, mh])


# BASELINE.json `configs`, in order.  `nsteps`/`dt` are the KDK run of the config (0 = forces only).
CONFIGS = (
    dict(name="disk_2048", kind="disk", N=2048, delta=0.02, sigma_f=0.1, dt=1e-3, nsteps=10, seed=0),
    dict(name="disk_halo_2x65536", kind="disk+halo", N=2 ** 17, delta=0.01, sigma_f=0.1, dt=5e-4, nsteps=200,
         seed=1),
    dict(name="disk_2^20", kind="disk", N=2 ** 20, delta=0.005, sigma_f=0.05, dt=2.5e-4, nsteps=100, seed=2),
    dict(name="plummer_2^22", kind="plummer", N=2 ** 22, delta=0.005, dt=0.0, nsteps=0, seed=3),
    dict(name="disk_halo_2x2^22", kind="disk+halo", N=2 ** 23, delta=0.002, sigma_f=0.1, dt=0.0, nsteps=0,
         seed=4),
)


def make(kind, N, seed, sigma_f=0.1, G=1.0):
    """(pos[N,3], vel[N,3], mass[N]) float64, COM frame."""
    if kind == "disk":
        p, v, m = exponential_disk(N, seed, G=G, sigma_f=sigma_f)
    elif kind == "plummer":
        p, v, m = plummer_sphere(N, seed, G=G)
    elif kind == "disk+halo":
        assert N % 2 == 0
        p, v, m = disk_plus_halo(N // 2, N // 2, seed, G=G, sigma_f=sigma_f)
    else:
        raise ValueError(kind)
    return _recentre(p, v, m)


def config(k, N=None):
    """Workload of BASELINE.json configs[k] (optionally at a reduced N, same recipe and seed)."""
    c = dict(CONFIGS[k])
    if N is not None:
        c["N"] = int(N)
    c["G"] = 1.0
    c["pos"], c["vel"], c["mass"] = make(c["kind"], c["N"], c["seed"], c.get("sigma_f", 0.1), c["G"])
    return c


def jeans_disk_draws(n, seed):
    """The random numbers of the equilibrium-disk generator of eqs. (3)-(4): uniforms in (0, 1) for
    radius, azimuth and height, standard normals for the three velocity components.  Both the CUDA-path generator
    (disk_ic.py) and the oracle's (oracle/disk_ic.py) take these as INPUTS, so neither draws anything itself."""
    return {"u_R": _open01(_rng(seed, "jeans_R"), n), "u_phi": _open01(_rng(seed, "jeans_phi"), n),
            "u_z": _open01(_rng(seed, "jeans_z"), n), "g": _rng(seed, "jeans_vel").standard_normal((n, 3))}


def sample_indices(seed, N, n=4096):
    """n distinct particle indices (sorted), from the config's 'sample' stream."""
    n = min(n, N)
    return np.sort(_rng(seed, "sample").choice(N, size=n, replace=False)).astype(np.int64)


def as_f32_exact(*arrays):
    """Round to float32 and convert back to float64: the inputs an FP32 run actually sees."""
    return tuple(np.asarray(a, dtype=np.float32).astype(np.float64) for a in arrays)
