"""Seeded input generators (P10 of DESIGN.md): determinism, structure, and large-N sanity against closed forms,
the latter also exercising the oracle's force routine on a realistic mass distribution (CPU only)."""
import math

import numpy as np
import pytest

from paper_1803_01190_b200 import workloads as w


def test_deterministic_and_seed_dependent():
    a = w.config(0)
    b = w.config(0)
    assert np.array_equal(a["pos"], b["pos"]) and np.array_equal(a["vel"], b["vel"])
    c = w.make("disk", 2048, seed=1)
    assert not np.array_equal(a["pos"], c[0])
    assert np.array_equal(w.sample_indices(3, 10 ** 6, 100), w.sample_indices(3, 10 ** 6, 100))
    idx = w.sample_indices(3, 10 ** 6, 4096)
    assert len(np.unique(idx)) == 4096 and idx.min() >= 0 and idx.max() < 10 ** 6


def test_config_table_matches_baseline_json():
    import json, os
    base = json.load(open(os.path.join(os.path.dirname(__file__), "..", "BASELINE.json")))
    assert len(base["configs"]) == len(w.CONFIGS) == 5
    assert [c["N"] for c in w.CONFIGS] == [2048, 2 ** 17, 2 ** 20, 2 ** 22, 2 ** 23]
    assert [c["seed"] for c in w.CONFIGS] == [0, 1, 2, 3, 4]
    assert [c["delta"] for c in w.CONFIGS] == [0.02, 0.01, 0.005, 0.005, 0.002]


def test_com_frame_and_masses():
    for kind, n in (("disk", 4096), ("plummer", 4096), ("disk+halo", 8192)):
        p, v, m = w.make(kind, n, seed=5)
        assert p.shape == (n, 3) and v.shape == (n, 3) and m.shape == (n,)
        assert np.all(np.isfinite(p)) and np.all(np.isfinite(v)) and np.all(m > 0)
        np.testing.assert_allclose((m[:, None] * p).sum(0) / m.sum(), 0.0, atol=1e-14)
        np.testing.assert_allclose((m[:, None] * v).sum(0), 0.0, atol=1e-14)
    p, v, m = w.make("disk+halo", 8192, seed=5)
    assert m[:4096].sum() == pytest.approx(1.0) and m[4096:].sum() == pytest.approx(4.0)   # two mass species
    assert m[0] != m[-1]


def test_disk_structure():
    n = 200000
    p, v, m = w.make("disk", n, seed=6)
    R = np.hypot(p[:, 0], p[:, 1])
    assert R.max() <= 4.0 + 0.05
    mean_R = (2 - 26 * math.exp(-4)) / (1 - 5 * math.exp(-4))        # <R> of R e^{-R} truncated at 4
    assert R.mean() == pytest.approx(mean_R, rel=0.01)
    assert np.mean(p[:, 2] ** 2) == pytest.approx(math.pi ** 2 * 0.1 ** 2 / 12, rel=0.03)   # sech^2 law
    Lz = np.sum(m * (p[:, 0] * v[:, 1] - p[:, 1] * v[:, 0]))
    assert Lz > 0                                                    # counter-clockwise rotation
    vphi = (p[:, 0] * v[:, 1] - p[:, 1] * v[:, 0]) / R
    sel = (R > 1.9) & (R < 2.1)
    vc = math.sqrt(float(w.disk_enclosed_mass(np.array([2.0]))[0]) / 2.0)
    assert vphi[sel].mean() == pytest.approx(vc, rel=0.02)
    assert vphi[sel].std() == pytest.approx(0.1 * vc, rel=0.1)


def test_plummer_structure_and_oracle_forces(oracle):
    n = 20000
    p, v, m = w.make("plummer", n, seed=7)
    r = np.linalg.norm(p, axis=1)
    assert np.median(r) == pytest.approx(1.0 / math.sqrt(2 ** (2 / 3) - 1), rel=0.03)       # half-mass radius
    delta = 0.01
    idx = w.sample_indices(7, n, 2000)
    acc, pot = oracle.forces(p, m, G=1.0, delta=delta, nthreads=0)
    inv = oracle.invariants(p, v, m, G=1.0, delta=delta, pot=pot)
    assert inv["W"] == pytest.approx(-3 * math.pi / 32, rel=0.03)     # Plummer: W = -(3 pi/32) G M^2 / a
    assert 2 * inv["K"] / abs(inv["W"]) == pytest.approx(1.0, abs=0.05)                       # virial equilibrium
    # mean radial acceleration in shells follows -G M r / (r^2 + a^2)^{3/2}
    rhat = p / r[:, None]
    a_r = np.sum(acc * rhat, axis=1)
    for lo, hi in ((0.3, 0.5), (0.9, 1.1), (1.8, 2.2)):
        sel = (r > lo) & (r < hi)
        want = np.mean(-r[sel] / (r[sel] ** 2 + 1.0) ** 1.5)
        assert a_r[sel].mean() == pytest.approx(want, rel=0.05)
    # mean potential follows -G M / sqrt(r^2 + a^2)
    sel = (r > 0.9) & (r < 1.1)
    assert pot[sel].mean() == pytest.approx(np.mean(-1.0 / np.sqrt(r[sel] ** 2 + 1.0)), rel=0.03)


def test_as_f32_exact_roundtrip():
    c = w.config(0)
    (p32,) = w.as_f32_exact(c["pos"])
    assert p32.dtype == np.float64
    assert np.array_equal(p32.astype(np.float32).astype(np.float64), p32)
    assert np.max(np.abs(p32 - c["pos"])) < 4.0 * 2 ** -24
