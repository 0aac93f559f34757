"""Pins of oracle.surface_density (the surface-density maps of Fig. 7) against things other than
itself: a hand-worked example, mass conservation, numpy.histogram2d (an independent library binning) and the analytic
exponential profile of the disk workload."""
import numpy as np

from paper_1803_01190_b200 import workloads


def test_hand_example_edges_and_outside(oracle):
    # 2 x 2 grid of unit... cell 0.5 starting at (-0.5, -0.5): cells [-0.5,0) and [0,0.5) in each direction
    pos = np.array([[-0.25, -0.25, 9.0],     # cell (iy=0, ix=0)
                    [0.25, -0.25, 0.0],      # (0, 1)
                    [0.0, 0.0, 0.0],         # exactly on the inner edges -> upper cell (1, 1)
                    [0.49, 0.1, 0.0],        # (1, 1)
                    [-0.5, 0.25, 0.0],       # on the lower boundary -> inside, (1, 0)
                    [0.5, 0.0, 0.0],         # on the upper boundary -> outside
                    [-0.6, 0.0, 0.0],        # outside
                    [0.1, 7.0, 0.0]])        # outside
    mass = np.array([1.0, 2.0, 4.0, 8.0, 16.0, 32.0, 64.0, 128.0])
    s = oracle.surface_density(pos, mass, -0.5, -0.5, 0.5, 2, 2)
    assert s.shape == (2, 2)
    assert np.array_equal(s * 0.25, np.array([[1.0, 2.0], [16.0, 12.0]]))


def test_mass_conservation_and_histogram2d(oracle):
    pos, _, mass = workloads.make("disk", 20000, 7)
    x0 = y0 = -4.5
    cell, n = 0.125, 72
    s = oracle.surface_density(pos, mass, x0, y0, cell, n, n)
    inside = (np.abs(pos[:, 0]) < 4.5) & (np.abs(pos[:, 1]) < 4.5)
    assert inside.all()                                   # the disk is truncated at R = 4
    assert abs(s.sum() * cell * cell - mass.sum()) <= 1e-13
    edges = x0 + cell * np.arange(n + 1)
    h, _, _ = np.histogram2d(pos[:, 1], pos[:, 0], bins=(edges, edges), weights=mass)
    assert np.abs(h / cell ** 2 - s).max() <= 1e-12 * s.max()


def test_exponential_profile(oracle):
    """Azimuthal average of the map follows exp(-R/h)/(2 pi h^2 [1 - 5 e^-4]) (workload recipe)."""
    n_body = 200000
    pos, _, mass = workloads.make("disk", n_body, 3)
    cell, n = 0.1, 90
    s = oracle.surface_density(pos, mass, -4.5, -4.5, cell, n, n)
    c = -4.5 + cell * (np.arange(n) + 0.5)
    R = np.hypot(c[None, :], c[:, None])
    norm = 2 * np.pi * (1 - 5 * np.exp(-4.0))
    for lo, hi in ((0.5, 1.0), (1.0, 2.0), (2.0, 3.0)):
        ring = (R >= lo) & (R < hi)
        got = s[ring].mean()
        want = (np.exp(-R[ring]) / norm).mean()
        n_in = got * ring.sum() * cell * cell * n_body           # bodies in the ring
        assert abs(got - want) <= 5.0 / np.sqrt(n_in) * want + 0.01 * want
