"""Pins of the oracle's KDK leapfrog (eqs. (5)-(7)) and invariants (eqs. (8)-(10),
PAPER.md:148-156) to closed forms and structural properties (CPU only).

P5 softened circular binary: omega^2 = 2Gm/(d^2+delta^2)^{3/2}  (fixes the delta convention in the dynamics)
P6 Kepler two-body: period, energy -G m1 m2 / 2a, eccentricity; E error ~ dt^2, no secular drift
P7 time reversibility
P8 exact conservation of P and L by the scheme
R4 eqs. (5)-(7) as printed == half-kick/drift/half-kick to round-off; one force evaluation per step
"""
import math

import numpy as np
import pytest


def _kepler(m1, m2, a, e, G):
    """Two bodies at apocentre in the COM frame; returns pos, vel, mass and the closed-form T, E, L_z."""
    M = m1 + m2
    r_ap = a * (1 + e)
    v_ap = math.sqrt(G * M * (1 - e) / (a * (1 + e)))       # vis-viva at apocentre
    pos = np.array([[m2 / M * r_ap, 0, 0], [-m1 / M * r_ap, 0, 0]], dtype=float)
    vel = np.array([[0, m2 / M * v_ap, 0], [0, -m1 / M * v_ap, 0]], dtype=float)
    T = 2 * math.pi * math.sqrt(a ** 3 / (G * M))
    E = -G * m1 * m2 / (2 * a)
    Lz = m1 * m2 / M * r_ap * v_ap
    return pos, vel, np.array([m1, m2], dtype=float), T, E, Lz


def _ecc_vector(pos, vel, mass, G):
    """Laplace-Runge-Lenz eccentricity vector of the relative orbit."""
    r = pos[0] - pos[1]
    v = vel[0] - vel[1]
    mu = G * mass.sum()
    h = np.cross(r, v)
    return np.cross(v, h) / mu - r / np.linalg.norm(r)


def test_invariants_closed_form_two_body(oracle):
    G, m1, m2, a, e = 2.0, 3.0, 1.0, 1.5, 0.4
    pos, vel, mass, T, E, Lz = _kepler(m1, m2, a, e, G)
    inv = oracle.invariants(pos, vel, mass, G=G, delta=0.0)
    assert inv["E"] == pytest.approx(E, rel=1e-15)                   # needs the MINUS sign in eq. (8) (reading R3)
    assert inv["W"] == pytest.approx(-G * m1 * m2 / (a * (1 + e)), rel=1e-15)
    assert inv["K"] > 0 and inv["W"] < 0
    assert inv["Lz"] == pytest.approx(Lz, rel=1e-15)
    np.testing.assert_allclose(inv["P"], 0.0, atol=1e-15)
    np.testing.assert_allclose(inv["COM"], 0.0, atol=1e-15)
    assert inv["M"] == m1 + m2


def test_invariants_general_definitions(oracle):
    rng = np.random.default_rng(3)
    n = 30
    pos, vel, mass = rng.normal(size=(n, 3)), rng.normal(size=(n, 3)), rng.uniform(0.5, 1.5, n)
    G, delta = 1.7, 0.2
    inv = oracle.invariants(pos, vel, mass, G=G, delta=delta)
    K = sum(0.5 * mass[i] * np.dot(vel[i], vel[i]) for i in range(n))
    W = 0.0
    for i in range(n):
        for j in range(i + 1, n):                                    # each unordered pair once == (1/2) sum_{i != j}
            W -= G * mass[i] * mass[j] / math.sqrt(np.sum((pos[i] - pos[j]) ** 2) + delta ** 2)
    assert inv["K"] == pytest.approx(K, rel=1e-14)
    assert inv["W"] == pytest.approx(W, rel=1e-14)
    assert inv["E"] == pytest.approx(K + W, rel=1e-13)
    np.testing.assert_allclose(inv["P"], (mass[:, None] * vel).sum(0), rtol=1e-13, atol=1e-14)
    np.testing.assert_allclose(inv["L"], (mass[:, None] * np.cross(pos, vel)).sum(0), rtol=1e-13, atol=1e-14)
    np.testing.assert_allclose(inv["COM"], (mass[:, None] * pos).sum(0) / mass.sum(), rtol=1e-13, atol=1e-15)
    # a supplied potential is used as is
    _, pot = oracle.forces(pos, mass, G=G, delta=delta)
    inv2 = oracle.invariants(pos, vel, mass, G=G, delta=delta, pot=pot)
    assert inv2["W"] == inv["W"] and inv2["E"] == inv["E"]


def test_P5_softened_circular_binary_stays_circular(oracle):
    G, m, d, delta = 1.0, 0.5, 1.0, 0.75
    omega = math.sqrt(2 * G * m / (d * d + delta * delta) ** 1.5)    # Plummer-softened pair, eq. (2) + PAPER.md:48
    pos = np.array([[d / 2, 0, 0], [-d / 2, 0, 0]], dtype=float)
    vel = np.array([[0, omega * d / 2, 0], [0, -omega * d / 2, 0]], dtype=float)
    mass = np.array([m, m])
    T = 2 * math.pi / omega
    nsteps = 4000
    sep = []
    p, v, a = pos, vel, None
    for _ in range(8):                                               # 2 periods in 8 chunks
        p, v, a, _ = oracle.kdk_paper(p, v, mass, T / 2000, nsteps // 8, G=G, delta=delta, acc=a)
        sep.append(np.linalg.norm(p[0] - p[1]))
    assert max(abs(s - d) for s in sep) < 5e-6 * d                   # O(dt^2) wobble only
    # after exactly two periods the bodies are back (phase error O(dt^2))
    np.testing.assert_allclose(p, pos, atol=2e-5)
    # the literal (|r|+delta)^3 reading would need omega'^2 = 2Gm/(d (d+delta)^2) -- a 40 % different speed, i.e.
    # a strongly eccentric orbit with these initial conditions:
    omega_lit = math.sqrt(2 * G * m / (d * (d + delta) ** 2))
    assert abs(omega_lit - omega) / omega > 0.1


def test_P6_kepler_period_energy_eccentricity(oracle):
    G, m1, m2, a, e = 1.0, 1.0, 0.5, 1.0, 0.5
    pos, vel, mass, T, E, Lz = _kepler(m1, m2, a, e, G)
    steps_per_orbit = 2000
    dt = T / steps_per_orbit
    p, v, acc = pos, vel, None
    Es, Ls, es = [], [], []
    for orbit in range(100):
        p, v, acc, nf = oracle.kdk_paper(p, v, mass, dt, steps_per_orbit, G=G, acc=acc)
        inv = oracle.invariants(p, v, mass, G=G)
        Es.append(inv["E"]); Ls.append(inv["Lz"]); es.append(_ecc_vector(p, v, mass, G))
    Es, Ls, es = np.array(Es), np.array(Ls), np.array(es)
    # energy: bounded O(dt^2) error, no secular drift over 100 orbits
    assert np.max(np.abs(Es - E)) < 2e-5 * abs(E)
    assert abs(Es[-1] - Es[0]) < 1e-9 * abs(E)
    # angular momentum: conserved to round-off by the scheme
    assert np.max(np.abs(Ls - Lz)) < 1e-12 * Lz
    # eccentricity magnitude stays put; the apsidal line precesses slowly and linearly (a known leapfrog error)
    assert np.max(np.abs(np.linalg.norm(es, axis=1) - e)) < 1e-4
    # period: after 100 nominal periods the body is back at apocentre up to the O(dt^2) phase/precession error
    sep = np.linalg.norm(p[0] - p[1])
    assert sep == pytest.approx(a * (1 + e), rel=2e-3)
    # semi-major axis from the conserved energy gives the closed-form period
    a_num = -G * m1 * m2 / (2 * np.mean(Es))
    assert 2 * math.pi * math.sqrt(a_num ** 3 / (G * (m1 + m2))) == pytest.approx(T, rel=1e-5)


def test_P6_second_order_convergence(oracle):
    G, m1, m2, a, e = 1.0, 1.0, 1.0, 1.0, 0.3
    pos, vel, mass, T, E, _ = _kepler(m1, m2, a, e, G)
    # exact state after a quarter period is not needed: compare errors against a much finer run
    ref_p, ref_v, _, _ = oracle.kdk_paper(pos, vel, mass, T / 4 / 6400, 6400, G=G)
    errs = []
    for n in (100, 200, 400):
        p, v, _, _ = oracle.kdk_paper(pos, vel, mass, T / 4 / n, n, G=G)
        errs.append(np.linalg.norm(p - ref_p))
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.05)
    assert errs[1] / errs[2] == pytest.approx(4.0, rel=0.05)
    # energy error amplitude also ~ dt^2
    dE = []
    for n in (200, 400):
        p, v, _, _ = oracle.kdk_paper(pos, vel, mass, T / 4 / n, n, G=G)
        dE.append(abs(oracle.invariants(p, v, mass, G=G)["E"] - E))
    assert dE[0] / dE[1] == pytest.approx(4.0, rel=0.1)


def _small_cluster(n=64, seed=4):
    from paper_1803_01190_b200 import workloads
    p, v, m = workloads.make("plummer", n, seed)
    return p, v, m


def test_P7_time_reversibility(oracle):
    pos, vel, mass = _small_cluster()
    dt, n, delta = 1e-3, 1000, 0.05
    p, v, a, _ = oracle.kdk_paper(pos, vel, mass, dt, n, delta=delta)
    p2, v2, _, _ = oracle.kdk_paper(p, -v, mass, dt, n, delta=delta, acc=a)
    assert np.max(np.abs(p2 - pos)) < 1e-11
    assert np.max(np.abs(-v2 - vel)) < 1e-11
    assert np.max(np.abs(p - pos)) > 1e-2                             # it did move


def test_P8_momentum_and_angular_momentum_conserved_to_roundoff(oracle):
    pos, vel, mass = _small_cluster(96, 7)
    delta = 0.05
    inv0 = oracle.invariants(pos, vel, mass, delta=delta)
    p, v, _, _ = oracle.kdk_paper(pos, vel, mass, 2e-3, 500, delta=delta)
    inv1 = oracle.invariants(p, v, mass, delta=delta)
    pscale = np.sum(mass * np.linalg.norm(vel, axis=1))
    lscale = np.sum(mass * np.linalg.norm(np.cross(pos, vel), axis=1))
    assert np.linalg.norm(inv1["P"] - inv0["P"]) < 1e-14 * pscale     # cf. Table 2 DP column ~1e-15
    assert np.linalg.norm(inv1["L"] - inv0["L"]) < 1e-13 * lscale     # cf. Table 2 DP column ~1e-14..1e-13
    assert abs(inv1["E"] - inv0["E"]) < 1e-4 * abs(inv0["E"])         # O(dt^2), cf. Table 2 DP ~5e-5
    assert abs(inv1["E"] - inv0["E"]) > 0
    # COM moves with P/M (here ~0)
    np.testing.assert_allclose(inv1["COM"], inv0["COM"] + 1.0 * inv0["P"] / inv0["M"], atol=1e-14)


def test_R4_paper_form_equals_halfkick_form_and_one_force_per_step(oracle):
    pos, vel, mass = _small_cluster(8, 2)
    p1, v1, a1, nf1 = oracle.kdk_paper(pos, vel, mass, 1e-3, 100, delta=0.05)
    p2, v2, a2, nf2 = oracle.kdk_halfkick(pos, vel, mass, 1e-3, 100, delta=0.05)
    assert nf1 == nf2 == 101                                          # initial + one per step
    assert np.max(np.abs(p1 - p2)) < 1e-14 and np.max(np.abs(v1 - v2)) < 1e-13
    # continuing with the carried acceleration costs exactly nsteps evaluations and gives the same trajectory
    p3, v3, a3, nf3 = oracle.kdk_paper(pos, vel, mass, 1e-3, 50, delta=0.05)
    p4, v4, a4, nf4 = oracle.kdk_paper(p3, v3, mass, 1e-3, 50, delta=0.05, acc=a3)
    assert nf3 == 51 and nf4 == 50
    assert np.array_equal(p4, p1) and np.array_equal(v4, v1) and np.array_equal(a4, a1)


def test_single_step_by_hand(oracle):
    # one step of (5)-(7) for a two-body problem, evaluated by hand from the printed equations
    G, dt = 1.0, 0.1
    pos = np.array([[1.0, 0, 0], [-1.0, 0, 0]])
    vel = np.array([[0, 0.5, 0], [0, -0.5, 0]])
    mass = np.array([1.0, 1.0])
    a0 = np.array([[-0.25, 0, 0], [0.25, 0, 0]])                      # G m / 2^2 towards the other body
    vt = vel + dt * a0                                                # (5)
    r1 = pos + dt / 2 * (vt + vel)                                    # (6)
    d = r1[0] - r1[1]
    a1 = np.array([-d / np.linalg.norm(d) ** 3, d / np.linalg.norm(d) ** 3])
    v1 = (vel + vt) / 2 + dt / 2 * a1                                 # (7)
    p, v, a, nf = oracle.kdk_paper(pos, vel, mass, dt, 1, G=G)
    np.testing.assert_allclose(p, r1, rtol=1e-15, atol=1e-16)
    np.testing.assert_allclose(v, v1, rtol=1e-15, atol=1e-16)
    np.testing.assert_allclose(a, a1, rtol=1e-15, atol=1e-16)
    assert nf == 2
