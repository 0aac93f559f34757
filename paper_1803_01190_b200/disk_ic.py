"""Equilibrium stellar-disk initial conditions from the paper's eqs. (3)-(4), with the radial
gravity taken from the library's own gravity solve (pp_forces, eq. (1)-(2)) -- SURVEY.md section 8(f) NEXT-4.

    python -m paper_1803_01190_b200.disk_ic --n 131072 --seed 2 --out disk.npz

The paper builds its disk by an iterative procedure that lives in its refs [1, 15, 18] and is not
reproduced here.  What the paper does print are the two equilibrium conditions; this generator satisfies them for
stated profiles in two fixed passes (readings R13-R16):

  eq. (3)  v_phi^2 / r = g_r + (c_r^2 / r) (1 - c_phi^2/c_r^2 + dln(rho c_r^2)/dln r),   <v_r v_z> = 0
           (left side read as the centripetal acceleration of the MEAN rotation, "-dPsi/dr" as the inward pull g_r)
  eq. (4)  (ln rho)'' = -(4 pi G / c_z^2) (rho - rho_*),   rho_* = (1 / 4 pi G r) dV_c^2/dr,   V_c^2 = r g_r
  R14      Sigma(R) = Sigma_0 e^{-R/h} truncated at 4h;  c_z^2 = pi G Sigma z_0;  c_r = c_z / f_z;
           c_phi^2 = c_r^2 kappa^2 / (4 Omega^2)
  pass 1   z from the rho_* = 0 sheet (sech^2), g_r(R) from pp_forces  ->  V_c^2, rho_*
  pass 2   eq. (4) solved per radial bin (RK4 in z, midplane density by bisection on the column), z re-placed, g_r from
           pp_forces again  ->  V_c^2, Omega, kappa, mean v_phi from eq. (3); Gaussian dispersions c_r, c_phi, c_z.

Only the two O(N^2) force evaluations are heavy and they run in libppgrav's kernels (no CPU fallback); the O(N) profile
arithmetic is host numpy, vectorised over the radial bins.  The random numbers are inputs (workloads.jeans_disk_draws).
This module shares no code with oracle/disk_ic.py, the CPU restatement the tests compare it with.
"""
import math

import numpy as np

from . import ppgrav, workloads

TRUNC = workloads.DISK_TRUNC


def _sigma(R, h, M_d):
    return M_d / (2.0 * math.pi * h * h * (1.0 - (1.0 + TRUNC) * math.exp(-TRUNC))) * np.exp(-R / h)


def _radii(u, h):
    """R with enclosed-mass fraction u: bisection on 1 - (1 + x) e^-x, all bodies at once."""
    target = u * (1.0 - (1.0 + TRUNC) * math.exp(-TRUNC))
    lo, hi = np.zeros_like(u), np.full_like(u, TRUNC)
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        below = 1.0 - (1.0 + mid) * np.exp(-mid) < target
        lo = np.where(below, mid, lo)
        hi = np.where(below, hi, mid)
    return 0.5 * (lo + hi) * h


def _sheets(rho0, k, rho_star, dz, nz):
    """eq. (4) for all bins at once: RK4 in z for y = ln rho, y'' = -k (e^y - rho_*), from the midplane.  A bin's layer
    ends at its density minimum (rho_* > 0: y' returns to 0; located by linear interpolation of y' inside the grid
    step, which keeps the column continuous in rho0), 69 e-folds below the midplane, or at the end of the grid.
    Returns (rho[bins, nz+1] at the grid points inside the layer, 0 beyond; n_in[bins] = index of the last such point;
    z_end[bins], rho_end[bins] = the end point, equal to the last grid point where there is no minimum)."""
    nb = len(rho0)
    y, p = np.log(rho0), np.zeros(nb)
    y0 = y.copy()
    alive = np.ones(nb, dtype=bool)
    rho = np.zeros((nb, nz + 1))
    rho[:, 0] = rho0
    n_in = np.zeros(nb, dtype=np.int64)
    z_end, rho_end = np.zeros(nb), rho0.copy()

    def acc(yy):
        return -k * (np.exp(yy) - rho_star)

    for n in range(nz):
        k1y, k1p = p, acc(y)
        k2y, k2p = p + 0.5 * dz * k1p, acc(y + 0.5 * dz * k1y)
        k3y, k3p = p + 0.5 * dz * k2p, acc(y + 0.5 * dz * k2y)
        k4y, k4p = p + dz * k3p, acc(y + dz * k3y)
        y_new = y + dz * (k1y + 2 * k2y + 2 * k3y + k4y) / 6.0
        p_new = p + dz * (k1p + 2 * k2p + 2 * k3p + k4p) / 6.0
        turn = alive & (p_new >= 0.0)
        if turn.any():
            frac = np.where(turn & (n > 0), p / np.where(turn, p - p_new, 1.0), 0.0)
            z_end = np.where(turn, (n + frac) * dz, z_end)
            rho_end = np.where(turn, np.exp(y + frac * (y_new - y)), rho_end)
        alive &= ~(turn | (y_new < y0 - 69.0))
        if not alive.any():
            break
        y, p = np.where(alive, y_new, y), np.where(alive, p_new, p)
        rho[alive, n + 1] = np.exp(y[alive])
        n_in[alive] = n + 1
        z_end[alive] = (n + 1) * dz
        rho_end[alive] = rho[alive, n + 1]
    return rho, n_in, z_end, rho_end


def _columns(rho, n_in, z_end, rho_end, dz):
    """int_0^z_end rho dz per bin: trapezoid over the grid points inside the layer plus the last partial interval."""
    inside = dz * (rho.sum(axis=1) - 0.5 * (rho[:, 0] + rho[np.arange(len(n_in)), n_in]))
    return inside + 0.5 * (rho[np.arange(len(n_in)), n_in] + rho_end) * (z_end - n_in * dz)


def _solve_columns(Sigma, c_z, rho_star, G, z0, nz=600, span=12.0):
    """Midplane densities (bisection, geometric) such that 2 int rho dz = Sigma in every bin."""
    k = 4.0 * math.pi * G / c_z ** 2
    dz = span * z0 / nz
    # rho_* > 0: the column diverges again as rho0 -> rho_*; the thin-disk branch is rho0 >> rho_* (search from 2 rho_*)
    lo, hi = np.maximum(1e-3 * Sigma / (2.0 * z0), 2.0 * rho_star), 1e3 * Sigma / (2.0 * z0)
    for _ in range(80):
        mid = np.sqrt(lo * hi)
        low = 2.0 * _columns(*_sheets(mid, k, rho_star, dz, nz), dz) < Sigma
        lo = np.where(low, mid, lo)
        hi = np.where(low, hi, mid)
    rho0 = np.sqrt(lo * hi)
    return dz, _sheets(rho0, k, rho_star, dz, nz), rho0


def _profiles(R, g_r, n_bins, h):
    width = TRUNC * h / n_bins
    centres = (np.arange(n_bins) + 0.5) * width
    which = np.minimum((R / (TRUNC * h) * n_bins).astype(np.int64), n_bins - 1)
    count = np.bincount(which, minlength=n_bins)
    g_mean = np.divide(np.bincount(which, weights=g_r, minlength=n_bins), count, out=np.zeros(n_bins), where=count > 0)
    vc2 = np.maximum(centres * g_mean, 1e-12)
    dvc2 = np.gradient(vc2, centres)
    omega2 = vc2 / centres ** 2
    kappa2 = np.maximum(2.0 * omega2 * (1.0 + 0.5 * centres * dvc2 / vc2), 1e-12)
    return centres, which, vc2, dvc2, omega2, kappa2


def _inward_pull(pos, mass, G, delta):
    acc, _ = ppgrav.pp_forces_host(np.ascontiguousarray(pos), np.ascontiguousarray(mass), G=G, delta=delta)
    R = np.hypot(pos[:, 0], pos[:, 1])
    return -(pos[:, 0] * acc[:, 0] + pos[:, 1] * acc[:, 1]) / R


def jeans_disk(draws, G=1.0, delta=0.02, h=1.0, M_d=1.0, z0=0.1, f_z=0.6, n_bins=32):
    """(pos[N,3], vel[N,3], mass[N], info) float64; not recentred (the caller subtracts the centre of mass)."""
    uR, uphi, uz, g = (np.asarray(draws[k], dtype=np.float64) for k in ("u_R", "u_phi", "u_z", "g"))
    N = uR.shape[0]
    mass = np.full(N, M_d / N)
    R = _radii(uR, h)
    phi = 2.0 * math.pi * uphi
    cs, sn = np.cos(phi), np.sin(phi)
    s = 2.0 * uz - 1.0
    pos = np.stack([R * cs, R * sn, z0 * np.arctanh(s)], axis=1)            # pass 1: the rho_* = 0 sheet
    centres, which, vc2, dvc2, omega2, kappa2 = _profiles(R, _inward_pull(pos, mass, G, delta), n_bins, h)
    Sigma = _sigma(centres, h, M_d)
    c_z_b = np.sqrt(math.pi * G * Sigma * z0)
    rho_star = dvc2 / (4.0 * math.pi * G * centres)
    rho_star[0] = vc2[0] / (2.0 * math.pi * G * centres[0] ** 2)
    rho_star = np.minimum(rho_star, 0.1 * Sigma / (2.0 * z0))              # thin-disk guard (R16): acts at R < 0.5 h
    dz, (rho, n_in, z_end, rho_end), rho0 = _solve_columns(Sigma, c_z_b, rho_star, G, z0)   # pass 2: eq. (4) with rho_*
    z = np.empty(N)
    for b in range(n_bins):
        sel = which == b
        if not sel.any():
            continue
        zb, rb = dz * np.arange(n_in[b] + 1), rho[b, :n_in[b] + 1]          # grid points inside the layer ...
        if z_end[b] > zb[-1]:
            zb, rb = np.append(zb, z_end[b]), np.append(rb, rho_end[b])     # ... and its end point (density minimum)
        cum = np.concatenate([[0.0], np.cumsum(0.5 * (rb[1:] + rb[:-1]) * np.diff(zb))])
        z[sel] = np.copysign(np.interp(np.abs(s[sel]), cum / cum[-1], zb), s[sel])
    pos = np.stack([R * cs, R * sn, z], axis=1)
    centres, which, vc2, dvc2, omega2, kappa2 = _profiles(R, _inward_pull(pos, mass, G, delta), n_bins, h)
    c_r_b = c_z_b / f_z
    ratio = np.minimum(kappa2 / (4.0 * omega2), 1.0)                        # c_phi^2 / c_r^2
    slope = centres * np.gradient(np.log(rho0 * c_r_b ** 2), centres)       # dln(rho c_r^2)/dln r at the midplane
    vphi_b = np.sqrt(np.maximum(vc2 + c_r_b ** 2 * (1.0 - ratio + slope), 0.0))      # eq. (3)
    c_r, c_p, c_z = (np.interp(R, centres, a) for a in (c_r_b, c_r_b * np.sqrt(ratio), c_z_b))
    vR, vp, vz = c_r * g[:, 0], np.interp(R, centres, vphi_b) + c_p * g[:, 1], c_z * g[:, 2]
    vel = np.stack([vR * cs - vp * sn, vR * sn + vp * cs, vz], axis=1)
    info = {"R_bin": centres, "Vc2": vc2, "rho_star": rho_star, "rho0": rho0, "c_r": c_r_b, "c_z": c_z_b,
            "c_phi": c_r_b * np.sqrt(ratio), "vphi_mean": vphi_b}
    return pos, vel, mass, info


def make(N, seed, G=1.0, delta=0.02, **kw):
    """Seeded equilibrium disk in its centre-of-mass frame: (pos, vel, mass) float64."""
    pos, vel, mass, _ = jeans_disk(workloads.jeans_disk_draws(N, seed), G=G, delta=delta, **kw)
    pos -= (mass[:, None] * pos).sum(axis=0) / mass.sum()
    vel -= (mass[:, None] * vel).sum(axis=0) / mass.sum()
    return pos, vel, mass


if __name__ == "__main__":
    import argparse
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--n", type=int, default=1 << 17)
    ap.add_argument("--seed", type=int, default=2)
    ap.add_argument("--delta", type=float, default=0.005)
    ap.add_argument("--out", required=True)
    a = ap.parse_args()
    p, v, m = make(a.n, a.seed, delta=a.delta)
    np.savez(a.out, pos=p, vel=v, mass=m)
