"""Equilibrium-disk initial conditions from eqs. (3)-(4) -- ORACLE, TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Plain, slow, step-by-step numpy/python restatement of the two equilibrium conditions the paper prints
(PAPER.md:54-65); the CUDA-path generator (paper_1803_01190_b200/disk_ic.py) shares no code with this file and
neither imports the other.  Only tests/ may import it.  The radial force comes from oracle.forces (eq. (1)-(2)).

What the paper fixes, and the reading taken where it is garbled or silent (readings R13-R16):

  eq. (3), radial balance "between the disk self-gravity, rotation and chaotic (thermal) motions":
      v_phi^2 / r = g_r + (c_r^2 / r) (1 - c_phi^2/c_r^2 + (r / (rho c_r^2)) d(rho c_r^2)/dr + (r/c_r^2) d<v_r v_z>/dz)
    R13: the printed left side "v_phi / r" is the centripetal acceleration v_phi^2 / r, and the printed "-dPsi/dr" is
    the inward gravitational acceleration g_r = -a_r > 0 (with Psi the usual negative potential the sign would make
    v_phi imaginary).  v_phi is the MEAN azimuthal velocity.  <v_r v_z> = 0 (velocity ellipsoid aligned with the
    cylindrical axes), so the last term drops.
  eq. (4), vertical equilibrium of the thin disk, divided by rho^2 and with <v_r v_z> = 0 (rho_alpha = 0):
      d^2 ln(rho) / dz^2 = -(4 pi G / c_z^2) (rho - rho_*),     rho_* = (1 / (4 pi G r)) dV_c^2/dr,   V_c^2 = r g_r(z=0)
    For rho_* = 0 its solution is the isothermal self-gravitating sheet rho = rho_0 sech^2(z/z_0),
    z_0 = c_z^2 / (pi G Sigma), rho_0 = Sigma / (2 z_0)  -- the closed form that pins vertical_profile().
  R14 (paper silent: the dispersion profiles are inputs "described in Ref. [1, 15, 18]"):
      c_z^2(R) = pi G Sigma(R) z_0   (the sheet relation for a constant scale height z_0),  c_r = c_z / f_z,
      c_phi^2 = c_r^2 kappa^2 / (4 Omega^2)  (epicyclic closure),  Omega = V_c / R,  kappa^2 = 2 Omega^2 (1 + dlnV_c/dlnR).
  R15 (iteration): the paper's "iterative procedure" is not in the paper.  This generator does a FIXED two passes:
      pass 1 places z from the rho_* = 0 sheet, measures g_r(R) from the particles, hence V_c^2 and rho_*;
      pass 2 re-solves eq. (4) with that rho_*, re-places z, measures g_r again and sets the velocities from eq. (3).
      It is NOT the relaxation of refs [1, 15, 18]; it satisfies eqs. (3)-(4) for the profiles above up to O(N^-1/2).
  R16 (discretisation): n_bins equal-width radial bins on [0, R_max]; bin means; derivatives by central differences
      on the bin centres (one-sided at the ends; rho_* of the innermost bin from the solid-body form V_c^2 ~ R^2, i.e.
      rho_* = Omega^2 / (2 pi G)); rho_* is capped at 0.1 of the rho_* = 0 sheet's midplane density Sigma / (2 z_0):
      eq. (4) is a thin-disk equation, and for rho_* comparable to rho no layer of the wanted column exists; the cap
      only acts at R < 0.5 h, where the disk is not thin compared with R; profiles are interpolated linearly in R to
      the particles.

Random numbers are INPUTS (`draws`, from paper_1803_01190_b200.workloads.jeans_disk_draws): u_R, u_phi, u_z uniform in
(0, 1), g[N,3] standard normal.
"""
import math

import numpy as np

from . import oracle as _oracle

R_MAX = 4.0     # truncation radius in units of h (the configs' recipe)


def surface_density(R, h=1.0, M_d=1.0):
    """Sigma(R) = Sigma_0 exp(-R/h) of the exponential disk truncated at R_MAX h with total mass M_d."""
    norm = 1.0 - (1.0 + R_MAX) * math.exp(-R_MAX)
    return M_d / (2.0 * math.pi * h * h * norm) * np.exp(-np.asarray(R, dtype=np.float64) / h)


def radius_from_uniform(u, h=1.0):
    """Inverse of the cumulative mass fraction m(x) = [1 - (1 + x) e^-x] / [1 - (1 + X) e^-X], x = R/h, X = R_MAX,
    by bisection (60 halvings: exact to round-off)."""
    norm = 1.0 - (1.0 + R_MAX) * math.exp(-R_MAX)
    out = np.empty(len(u))
    for i, ui in enumerate(u):
        lo, hi = 0.0, R_MAX
        target = ui * norm
        for _ in range(60):
            mid = 0.5 * (lo + hi)
            if 1.0 - (1.0 + mid) * math.exp(-mid) < target:
                lo = mid
            else:
                hi = mid
        out[i] = 0.5 * (lo + hi) * h
    return out


def _integrate_sheet(rho0, k, rho_star, dz, nz):
    """RK4 for y = ln rho:  y'' = -k (e^y - rho_star),  y(0) = ln rho0, y'(0) = 0, on z = 0, dz, ..., nz dz.
    For rho_star > 0 the density has a minimum (y' returns to 0) where the layer ends: its height z_end is located by
    linear interpolation of y' between the two grid points that bracket it, so that the column depends continuously on
    rho0.  The layer also ends 69 e-folds below the midplane or at the end of the grid.
    Returns (z[m+1], rho[m+1]): the grid points inside the layer plus the end point (z_end, rho_end)."""
    def f(y, p):
        return p, -k * (math.exp(y) - rho_star)
    y, p = math.log(rho0), 0.0
    zs, rho = [0.0], [rho0]
    for n in range(nz):
        k1y, k1p = f(y, p)
        k2y, k2p = f(y + 0.5 * dz * k1y, p + 0.5 * dz * k1p)
        k3y, k3p = f(y + 0.5 * dz * k2y, p + 0.5 * dz * k2p)
        k4y, k4p = f(y + dz * k3y, p + dz * k3p)
        y_new = y + dz * (k1y + 2 * k2y + 2 * k3y + k4y) / 6.0
        p_new = p + dz * (k1p + 2 * k2p + 2 * k3p + k4p) / 6.0
        if p_new >= 0.0:                                   # the minimum lies in (z_n, z_n+1]
            frac = p / (p - p_new) if n > 0 else 0.0
            zs.append((n + frac) * dz)
            rho.append(math.exp(y + frac * (y_new - y)))
            break
        if y_new < math.log(rho0) - 69.0:
            break
        y, p = y_new, p_new
        zs.append((n + 1) * dz)
        rho.append(math.exp(y))
    return np.array(zs), np.array(rho)


def _column(z, rho):
    """int_0^z_end rho dz by the trapezoid rule on the (possibly uneven last) intervals."""
    return float(np.sum(0.5 * (rho[1:] + rho[:-1]) * np.diff(z)))


def vertical_profile(Sigma, c_z, rho_star, G=1.0, z0_guess=0.1, nz=600, zmax_over_z0=12.0):
    """Solution of eq. (4) with <v_r v_z> = 0 for one radius: rho(z) from the midplane to the end of the layer, with
    the midplane density chosen (bisection) so that 2 int rho dz = Sigma.  Returns (z[m], rho[m], rho0)."""
    k = 4.0 * math.pi * G / (c_z * c_z)
    dz = zmax_over_z0 * z0_guess / nz
    # For rho_* > 0 the column is not monotonic in rho0 (it diverges again as rho0 -> rho_*, where the layer becomes
    # infinitely wide); the thin-disk solution is the branch rho0 >> rho_*, so the search starts at 2 rho_*.
    lo, hi = max(1e-3 * Sigma / (2.0 * z0_guess), 2.0 * rho_star), 1e3 * Sigma / (2.0 * z0_guess)
    for _ in range(80):
        mid = math.sqrt(lo * hi)
        if 2.0 * _column(*_integrate_sheet(mid, k, rho_star, dz, nz)) < Sigma:
            lo = mid
        else:
            hi = mid
    rho0 = math.sqrt(lo * hi)
    z, rho = _integrate_sheet(rho0, k, rho_star, dz, nz)
    return z, rho, rho0


def cumulative_column(z, rho):
    """Normalised cumulative column int_0^z rho dz' / int_0^z_end rho dz' (trapezoid).  Returns (z, cum)."""
    cum = np.concatenate([[0.0], np.cumsum(0.5 * (rho[1:] + rho[:-1]) * np.diff(z))])
    return z, cum / cum[-1]


def _z_from_uniform(u, z_part, cum_part):
    """z with |z| distributed as rho(z): inverse of the cumulative column by linear interpolation, sign from u."""
    s = 2.0 * u - 1.0
    return math.copysign(float(np.interp(abs(s), cum_part, z_part)), s)


def _bin_profiles(R, g_r, n_bins, h):
    """Bin means of g_r, hence V_c^2 = R g_r, Omega, kappa^2 and dV_c^2/dR on the bin centres (R16)."""
    edges = np.linspace(0.0, R_MAX * h, n_bins + 1)
    centres = 0.5 * (edges[1:] + edges[:-1])
    which = np.minimum((R / (R_MAX * h) * n_bins).astype(np.int64), n_bins - 1)
    g_mean = np.zeros(n_bins)
    for b in range(n_bins):
        sel = which == b
        g_mean[b] = g_r[sel].mean() if sel.any() else 0.0
    vc2 = np.maximum(centres * g_mean, 1e-12)
    dvc2 = np.gradient(vc2, centres)
    omega2 = vc2 / centres ** 2
    dlnv_dlnr = 0.5 * centres * dvc2 / vc2
    kappa2 = np.maximum(2.0 * omega2 * (1.0 + dlnv_dlnr), 1e-12)
    return centres, which, vc2, dvc2, omega2, kappa2


def _radial_gravity(pos, mass, G, delta, nthreads):
    acc, _ = _oracle.forces(pos, mass, G=G, delta=delta, want_pot=False, nthreads=nthreads)
    R = np.hypot(pos[:, 0], pos[:, 1])
    return -(pos[:, 0] * acc[:, 0] + pos[:, 1] * acc[:, 1]) / R


def jeans_disk(draws, G=1.0, delta=0.02, h=1.0, M_d=1.0, z0=0.1, f_z=0.6, n_bins=32, nthreads=0):
    """Positions, velocities, masses of a disk that satisfies eqs. (3)-(4) for the profiles of R14, in two passes (R15).
    Returns (pos[N,3], vel[N,3], mass[N], info) with the binned profiles in `info`.  The frame is NOT recentred."""
    uR, uphi, uz, g = (np.asarray(draws[k], dtype=np.float64) for k in ("u_R", "u_phi", "u_z", "g"))
    N = len(uR)
    mass = np.full(N, M_d / N)
    R = radius_from_uniform(uR, h)
    phi = 2.0 * math.pi * uphi
    cphi, sphi = np.cos(phi), np.sin(phi)
    # pass 1: rho_* = 0 -> the sech^2 sheet, whose inverse cumulative is closed-form
    z = z0 * np.arctanh(2.0 * uz - 1.0)
    pos = np.stack([R * cphi, R * sphi, z], axis=1)
    g_r = _radial_gravity(pos, mass, G, delta, nthreads)
    centres, which, vc2, dvc2, omega2, kappa2 = _bin_profiles(R, g_r, n_bins, h)
    Sigma_b = surface_density(centres, h, M_d)
    cz_b = np.sqrt(math.pi * G * Sigma_b * z0)                      # R14
    rho_star_b = dvc2 / (4.0 * math.pi * G * centres)               # eq. (4)
    rho_star_b[0] = vc2[0] / (2.0 * math.pi * G * centres[0] ** 2)  # innermost bin: solid-body rise V_c^2 ~ R^2 (R16)
    rho_star_b = np.minimum(rho_star_b, 0.1 * Sigma_b / (2.0 * z0))   # thin-disk guard: rho_* <= 0.1 of the sheet's rho_0
    # pass 2: eq. (4) with rho_* per bin; z re-placed from its cumulative column
    profiles = [vertical_profile(Sigma_b[b], cz_b[b], rho_star_b[b], G, z0) for b in range(n_bins)]
    columns = [cumulative_column(p[0], p[1]) for p in profiles]
    for i in range(N):
        z[i] = _z_from_uniform(uz[i], *columns[which[i]])
    pos = np.stack([R * cphi, R * sphi, z], axis=1)
    g_r = _radial_gravity(pos, mass, G, delta, nthreads)
    centres, which, vc2, dvc2, omega2, kappa2 = _bin_profiles(R, g_r, n_bins, h)
    rho0_b = np.array([p[2] for p in profiles])
    cr_b = cz_b / f_z
    cphi2_over_cr2_b = np.minimum(kappa2 / (4.0 * omega2), 1.0)     # R14, epicyclic closure (<= 1)
    dln_rho_cr2 = centres * np.gradient(np.log(rho0_b * cr_b ** 2), centres)
    vphi2_b = vc2 + cr_b ** 2 * (1.0 - cphi2_over_cr2_b + dln_rho_cr2)     # eq. (3) x r
    vphi_b = np.sqrt(np.maximum(vphi2_b, 0.0))
    # to the particles (linear in R between bin centres, constant beyond the outermost centres)
    c_r = np.interp(R, centres, cr_b)
    c_p = np.interp(R, centres, cr_b * np.sqrt(cphi2_over_cr2_b))
    c_z = np.interp(R, centres, cz_b)
    vphi = np.interp(R, centres, vphi_b)
    vR = c_r * g[:, 0]
    vp = vphi + c_p * g[:, 1]
    vz = c_z * g[:, 2]
    vel = np.stack([vR * cphi - vp * sphi, vR * sphi + vp * cphi, vz], axis=1)
    info = {"R_bin": centres, "Vc2": vc2, "rho_star": rho_star_b, "rho0": rho0_b, "c_r": cr_b, "c_z": cz_b,
            "c_phi": cr_b * np.sqrt(cphi2_over_cr2_b), "vphi_mean": vphi_b, "kappa2": kappa2, "omega2": omega2,
            "dln_rho_cr2_dlnR": dln_rho_cr2}
    return pos, vel, mass, info
