"""GPU parity of pp_surface_density (Fig. 7) against oracle.surface_density on the same seeded bodies:
identical cell decisions (both sides take floor((x - x0)/cell) in FP64 on what the run actually sees), cell sums equal
up to summation order (1e-12 of the fullest cell)."""
import numpy as np
import pytest

from paper_1803_01190_b200 import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("a -m gpu test was started without a CUDA device")
    from paper_1803_01190_b200 import ppgrav
    ppgrav.lib()
    return ppgrav


def _run(gpu, oracle, prec, pos, mass, x0, y0, cell, nx, ny):
    import torch
    dt = torch.float64 if prec == "f64" else torch.float32
    dpos = torch.tensor(pos, dtype=dt, device="cuda")
    dmass = torch.tensor(mass, dtype=dt, device="cuda")
    got = gpu.pp_surface_density(dpos, dmass, x0, y0, cell, nx, ny).cpu().numpy()
    seen_p, seen_m = dpos.cpu().numpy().astype(np.float64), dmass.cpu().numpy().astype(np.float64)
    ref = oracle.surface_density(seen_p, seen_m, x0, y0, cell, nx, ny)
    assert got.shape == ref.shape == (ny, nx)
    assert np.array_equal(got == 0.0, ref == 0.0), "a body landed in a different cell"
    # a cell holds up to n bodies; two summation orders of n positive terms differ by <= n eps (typically sqrt(n) eps),
    # and the kernel scales each mass by 1/cell^2 before adding where the oracle divides the sum: 30000 eps = 7e-12
    assert np.abs(got - ref).max() <= 1e-12 * max(ref.max(), 1e-300)
    return got, ref


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("nx,ny,cell", [(64, 64, 0.140625), (37, 11, 0.25), (512, 300, 0.017578125), (1, 1, 9.0)])
def test_density_map_matches_oracle(gpu, oracle, prec, nx, ny, cell):
    pos, _, mass = workloads.make("disk+halo", 30000, 9)       # two mass species, halo bodies partly off the grid
    x0, y0 = -0.5 * nx * cell, -0.5 * ny * cell
    got, ref = _run(gpu, oracle, prec, pos, mass, x0, y0, cell, nx, ny)
    assert got.sum() > 0.0


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_density_edges_outside_and_single_body(gpu, oracle, prec):
    pos = np.array([[-0.25, -0.25, 9.0], [0.25, -0.25, 0.0], [0.0, 0.0, 0.0], [0.49, 0.1, 0.0], [-0.5, 0.25, 0.0],
                    [0.5, 0.0, 0.0], [-0.6, 0.0, 0.0], [0.1, 7.0, 0.0]])
    mass = np.array([1.0, 2.0, 4.0, 8.0, 16.0, 32.0, 64.0, 128.0])
    got, _ = _run(gpu, oracle, prec, pos, mass, -0.5, -0.5, 0.5, 2, 2)
    assert np.array_equal(got * 0.25, np.array([[1.0, 2.0], [16.0, 12.0]]))     # the oracle pin's hand values
    got, _ = _run(gpu, oracle, prec, pos[:1], mass[:1], 5.0, 5.0, 1.0, 4, 4)    # nothing on the grid
    assert not got.any()


def test_density_rejects_bad_arguments(gpu):
    import ctypes
    import torch
    pos = torch.zeros((4, 3), device="cuda", dtype=torch.float64)
    mass = torch.ones(4, device="cuda", dtype=torch.float64)
    sigma = torch.zeros(16, device="cuda", dtype=torch.float64)
    lib, st = gpu.lib(), ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    for cell, nx, ny in ((0.0, 4, 4), (-1.0, 4, 4), (float("nan"), 4, 4), (1.0, 0, 4), (1.0, 1 << 14, 1 << 14)):
        rc = lib.pp_surface_density(pos.data_ptr(), mass.data_ptr(), 4, 0.0, 0.0, cell, nx, ny, gpu.PP_F64,
                                    sigma.data_ptr(), st)
        assert rc == -1 and b"pp_surface_density" in lib.pp_last_error()
    assert lib.pp_surface_density(pos.data_ptr(), mass.data_ptr(), 4, -1.0, -1.0, 0.5, 4, 4, gpu.PP_F64,
                                  sigma.data_ptr(), st) == 0
    torch.cuda.synchronize()
    assert float(sigma.sum()) == 4.0 / 0.25
