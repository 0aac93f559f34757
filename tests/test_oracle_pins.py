"""Pins of the CPU oracle's force / potential routine to things other than itself (CPU only).

P1 Pythagorean two-body values (tests/golden/two_body_pythagorean.txt; eq. (2) + PAPER.md:48)
P2 regular polygons, closed forms
P3 pairwise antisymmetry: sum m a = 0, sum m r x a = 0
P4 a = -grad Phi (central differences of W)
P9 brute force N <= 8 in 50-digit arithmetic with an independent loop
plus: long-double variant vs compensated double, sampled-index call vs all-particle call, thread invariance,
G and delta scaling laws.
"""
import math
import os

import mpmath
import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "two_body_pythagorean.txt")


def _golden_rows():
    rows = []
    with open(GOLDEN) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                rows.append([float(t) for t in line.split()])
    return rows


@pytest.mark.parametrize("row", _golden_rows())
def test_P1_pythagorean_two_body(oracle, row):
    dx, dy, dz, delta, n = row
    assert dx * dx + dy * dy + dz * dz + delta * delta == n * n      # the fixture itself is consistent
    pos = np.array([[dx, dy, dz], [0.0, 0.0, 0.0]])
    mass = np.array([1.0, 1.0])
    acc, pot = oracle.forces(pos, mass, G=1.0, delta=delta)
    want = -np.array([dx, dy, dz]) / n ** 3
    np.testing.assert_allclose(acc[0], want, rtol=4e-16, atol=0)
    np.testing.assert_allclose(acc[1], -want, rtol=4e-16, atol=0)     # f_21 = -f_12 for equal masses
    np.testing.assert_allclose(pot, [-1.0 / n, -1.0 / n], rtol=4e-16)
    # the literal "(|r| + delta)^3" reading of eq. (2) would give a different number whenever delta > 0
    if delta > 0:
        r = math.sqrt(dx * dx + dy * dy + dz * dz)
        assert abs(np.linalg.norm(acc[0]) - r / (r + delta) ** 3) > 1e-3 * np.linalg.norm(acc[0])


def test_P1_mass_and_G_enter_linearly_and_use_m_j(oracle):
    # a_1 depends on m_2 (the OTHER particle's mass), a_2 on m_1; G multiplies everything.
    pos = np.array([[3.0, 4.0, 0.0], [0.0, 0.0, 0.0]])
    acc, pot = oracle.forces(pos, np.array([2.0, 7.0]), G=3.0, delta=0.0)
    np.testing.assert_allclose(acc[0], -3.0 * 7.0 * np.array([3.0, 4.0, 0.0]) / 125.0, rtol=4e-16)
    np.testing.assert_allclose(acc[1], +3.0 * 2.0 * np.array([3.0, 4.0, 0.0]) / 125.0, rtol=4e-16)
    np.testing.assert_allclose(pot, [-3.0 * 7.0 / 5.0, -3.0 * 2.0 / 5.0], rtol=4e-16)


def test_P2_equilateral_triangle(oracle):
    s, m, G = 2.0, 0.5, 1.5
    pos = np.array([[0.0, 0.0, 0.0], [s, 0.0, 0.0], [s / 2, s * math.sqrt(3) / 2, 0.0]])
    acc, pot = oracle.forces(pos, np.full(3, m), G=G, delta=0.0)
    centroid = pos.mean(axis=0)
    for i in range(3):
        mag = np.linalg.norm(acc[i])
        assert mag == pytest.approx(math.sqrt(3) * G * m / s ** 2, rel=1e-15)
        to_c = centroid - pos[i]
        np.testing.assert_allclose(acc[i] / mag, to_c / np.linalg.norm(to_c), atol=1e-15)
        assert pot[i] == pytest.approx(-2 * G * m / s, rel=1e-15)


def test_P2_square_with_centre_body(oracle):
    s, m, G = 1.0, 1.0, 1.0
    pos = np.array([[0, 0, 0], [s, 0, 0], [s, s, 0], [0, s, 0], [s / 2, s / 2, 0]], dtype=float)
    mass = np.array([m, m, m, m, 0.0])                # massless test body at the centre
    acc, _ = oracle.forces(pos, mass, G=G, delta=0.0)
    want = (math.sqrt(2) + 0.5) * G * m / s ** 2
    for i in range(4):
        assert np.linalg.norm(acc[i]) == pytest.approx(want, rel=1e-15)
        d = (pos[(i + 2) % 4] - pos[i]) / (s * math.sqrt(2))          # along the diagonal, inwards
        np.testing.assert_allclose(acc[i] / want, d, atol=2e-15)
    np.testing.assert_allclose(acc[4], 0.0, atol=1e-15)              # centre of symmetry


def test_P2_cube_corners_point_to_centre(oracle):
    pos = np.array([[x, y, z] for x in (0.0, 1.0) for y in (0.0, 1.0) for z in (0.0, 1.0)])
    acc, pot = oracle.forces(pos, np.ones(8), G=1.0, delta=0.0)
    # 3 neighbours at 1, 3 at sqrt2, 1 at sqrt3; by symmetry the pull is along the body diagonal
    want = (3 * (1 / math.sqrt(3)) + 3 * (2 / math.sqrt(6)) / 2 + 1 / 3.0)
    for i in range(8):
        d = (np.array([0.5, 0.5, 0.5]) - pos[i]) / (math.sqrt(3) / 2)
        assert np.dot(acc[i], d) == pytest.approx(want, rel=1e-15)
        np.testing.assert_allclose(np.cross(acc[i], d), 0.0, atol=1e-15)
        assert pot[i] == pytest.approx(-(3 + 3 / math.sqrt(2) + 1 / math.sqrt(3)), rel=1e-15)


def _random_system(n, seed, spread=1.0):
    rng = np.random.default_rng(seed)
    pos = rng.normal(size=(n, 3)) * spread
    vel = rng.normal(size=(n, 3))
    mass = rng.uniform(0.1, 2.0, size=n)
    return pos, vel, mass


@pytest.mark.parametrize("delta", [0.0, 0.05])
def test_P3_antisymmetry(oracle, delta):
    pos, _, mass = _random_system(300, 11)
    acc, _ = oracle.forces(pos, mass, G=1.3, delta=delta)
    scale = np.sum(mass * np.linalg.norm(acc, axis=1))
    net_force = np.sum(mass[:, None] * acc, axis=0)
    net_torque = np.sum(mass[:, None] * np.cross(pos, acc), axis=0)
    assert np.linalg.norm(net_force) < 1e-14 * scale
    assert np.linalg.norm(net_torque) < 1e-14 * scale * np.abs(pos).max()


def test_P4_acceleration_is_minus_gradient_of_potential(oracle):
    pos, _, mass = _random_system(40, 5)
    G, delta = 0.7, 0.1
    acc, _ = oracle.forces(pos, mass, G=G, delta=delta)

    def W(p):
        _, pot = oracle.forces(p, mass, G=G, delta=delta, long_double=True)
        return 0.5 * np.sum(mass * pot)

    h = 1e-5
    for i, k in [(0, 0), (7, 1), (23, 2), (39, 0)]:
        pp, pm = pos.copy(), pos.copy()
        pp[i, k] += h
        pm[i, k] -= h
        dW = (W(pp) - W(pm)) / (2 * h)
        assert -dW == pytest.approx(mass[i] * acc[i, k], rel=1e-6, abs=1e-9)


def _brute_mp(pos, mass, G, delta):
    """Independent 50-digit loop, written straight from eq. (1)-(2) and PAPER.md:48."""
    mpmath.mp.dps = 50
    n = len(mass)
    acc = [[mpmath.mpf(0)] * 3 for _ in range(n)]
    pot = [mpmath.mpf(0) for _ in range(n)]
    for i in range(n):
        for j in range(n):
            if i == j:
                continue
            d = [mpmath.mpf(float(pos[i][k])) - mpmath.mpf(float(pos[j][k])) for k in range(3)]
            norm = mpmath.sqrt(d[0] ** 2 + d[1] ** 2 + d[2] ** 2 + mpmath.mpf(delta) ** 2)
            for k in range(3):
                acc[i][k] = acc[i][k] - mpmath.mpf(G) * mpmath.mpf(float(mass[j])) * d[k] / norm ** 3
            pot[i] = pot[i] - mpmath.mpf(G) * mpmath.mpf(float(mass[j])) / norm
    return (np.array([[float(c) for c in a] for a in acc]), np.array([float(p) for p in pot]))


@pytest.mark.parametrize("n,delta,seed", [(2, 0.0, 1), (3, 0.3, 2), (4, 0.0, 3), (5, 0.01, 4), (8, 0.1, 5), (8, 0.0, 6)])
def test_P9_brute_force_tiny(oracle, n, delta, seed):
    pos, _, mass = _random_system(n, seed)
    G = 1.0 + 0.25 * seed
    acc, pot = oracle.forces(pos, mass, G=G, delta=delta)
    acc_mp, pot_mp = _brute_mp(pos, mass, G, delta)
    scale = np.linalg.norm(acc_mp, axis=1)[:, None]
    assert np.max(np.abs(acc - acc_mp) / scale) < 1e-15 * n * 4
    np.testing.assert_allclose(pot, pot_mp, rtol=1e-15 * n)


def test_compensated_double_matches_long_double_on_a_disk(oracle):
    from paper_1803_01190_b200 import workloads
    c = workloads.config(0)
    idx = workloads.sample_indices(0, c["N"], 64)
    a, p = oracle.forces(c["pos"], c["mass"], delta=c["delta"], idx=idx)
    al, pl = oracle.forces(c["pos"], c["mass"], delta=c["delta"], idx=idx, long_double=True)
    rel = np.linalg.norm(a - al, axis=1) / np.linalg.norm(al, axis=1)
    assert rel.max() < 2e-15
    np.testing.assert_allclose(p, pl, rtol=1e-15)


def test_sampled_call_equals_full_call_and_threads_do_not_matter(oracle):
    pos, _, mass = _random_system(500, 21)
    a_all, p_all = oracle.forces(pos, mass, G=1.0, delta=0.02, nthreads=1)
    idx = np.array([0, 3, 17, 250, 499])
    a_s, p_s = oracle.forces(pos, mass, G=1.0, delta=0.02, idx=idx, nthreads=1)
    assert np.array_equal(a_all[idx], a_s) and np.array_equal(p_all[idx], p_s)
    a_mt, p_mt = oracle.forces(pos, mass, G=1.0, delta=0.02, nthreads=0)
    assert np.array_equal(a_all, a_mt) and np.array_equal(p_all, p_mt)     # bit-identical


def test_scaling_laws(oracle):
    # positions x lambda, delta x lambda  =>  a / lambda^2, Phi / lambda (exact for lambda a power of two)
    pos, _, mass = _random_system(50, 8)
    a1, p1 = oracle.forces(pos, mass, G=1.0, delta=0.125)
    a2, p2 = oracle.forces(pos * 4.0, mass, G=1.0, delta=0.5)
    assert np.array_equal(a1 / 16.0, a2) and np.array_equal(p1 / 4.0, p2)


def test_far_field_monopole(oracle):
    # a compact cluster seen from far away pulls like a point mass at its centre of mass (error ~ (size/D)^2)
    pos, _, mass = _random_system(200, 9, spread=0.01)
    com = np.sum(mass[:, None] * pos, axis=0) / mass.sum()
    probe = com + np.array([30.0, -40.0, 0.0])
    allpos = np.vstack([pos, probe])
    allmass = np.concatenate([mass, [0.0]])
    acc, pot = oracle.forces(allpos, allmass, G=2.0, delta=0.0, idx=np.array([200]))
    want = -2.0 * mass.sum() * (probe - com) / 50.0 ** 3
    np.testing.assert_allclose(acc[0], want, rtol=0, atol=1e-6 * np.linalg.norm(want))
    assert pot[0] == pytest.approx(-2.0 * mass.sum() / 50.0, rel=1e-6)
