"""pp_invariants_noalloc -- the allocation-free entry point (include/ppgrav.h): the kernels of pp_invariants with their
scratch in a static device array inside the library -- against the existing path, pp_invariants with the same supplied
potential, on two calls in a row that share that array (the second with fewer blocks than the first, so the array still
holds the first call's partial sums beyond the blocks the second call launches).

The file name sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide other tests.
It passes alone in a fresh process and after the rest of the suite (nothing here depends on library state: it sets no
pp_configure key and uses the default stream).
"""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("a -m gpu test was started without a CUDA device")
    from paper_1803_01190_b200 import ppgrav
    ppgrav.lib()
    return ppgrav


def _cloud(n, seed):
    rng = np.random.Generator(np.random.Philox(key=seed))
    pos = rng.standard_normal((n, 3)) + 0.3
    vel = 0.1 * rng.standard_normal((n, 3))
    mass = rng.uniform(0.5, 1.5, size=n) / n
    mass[n // 2:] *= 4.0
    return pos, vel, mass


def _check(got, ref, mass, vel):
    """Tolerances of tests/test_gpu_parity.py::_check_invariants (the two paths run the same kernels, so they in fact
    agree bit for bit, which is asserted separately)."""
    for k in (0, 1, 2):
        assert abs(got[k] - ref[k]) <= 1e-12 * abs(ref[k])
    p_scale = float(np.sum(np.abs(mass)[:, None] * np.abs(vel)))
    assert np.abs(got[3:6] - ref[3:6]).max() <= 1e-14 * p_scale
    assert np.abs(got[6:9] - ref[6:9]).max() <= 1e-12 * np.abs(ref[6:9]).max()
    assert np.abs(got[9:12] - ref[9:12]).max() <= 1e-13
    assert abs(got[12] - ref[12]) <= 1e-14 * ref[12]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_noalloc_invariants_match_the_existing_path_on_two_calls_in_a_row(gpu, oracle, prec):
    import torch
    dtype = torch.float64 if prec == "f64" else torch.float32
    out_a = torch.empty(16, dtype=torch.float64, device="cuda")
    out_b = torch.empty(16, dtype=torch.float64, device="cuda")
    # first 120011 bodies (296 blocks: the whole scratch array), then 1000 (4 blocks), then the first again
    cases = []
    for n, seed in ((120011, 41), (1000, 42)):
        pos, vel, mass = _cloud(n, seed)
        dpos, dvel, dmass = (torch.tensor(a, dtype=dtype, device="cuda") for a in (pos, vel, mass))
        _, dpot = gpu.pp_forces(dpos, dmass, G=1.3, delta=0.05, want_pot=True)
        ref = gpu.pp_invariants(dpos, dvel, dmass, G=1.3, delta=0.05, pot=dpot).clone()     # the existing path
        cases.append((dpos, dvel, dmass, dpot, ref))
    torch.cuda.synchronize()
    launches0 = gpu.pp_launch_count()
    for out, k in ((out_a, 0), (out_b, 1), (out_a, 0)):                  # back to back, no synchronisation in between
        dpos, dvel, dmass, dpot, ref = cases[k]
        got = gpu.pp_invariants_noalloc(dpos, dvel, dmass, dpot, out)
        assert got is out
        seen = dpos.double().cpu().numpy(), dvel.double().cpu().numpy(), dmass.double().cpu().numpy()
        _check(out.cpu().numpy(), ref.cpu().numpy(), seen[2], seen[1])
        assert torch.equal(out, ref), "same kernels, same inputs: the two paths must agree bit for bit"
    assert gpu.pp_launch_count() - launches0 == 3 * 2                    # partial + final kernel per call, nothing else
    # and against the oracle once (the oracle is handed the same potential values)
    dpos, dvel, dmass, dpot, _ = cases[1]
    p, v, m, phi = (t.double().cpu().numpy() for t in (dpos, dvel, dmass, dpot))
    o = oracle.invariants(p, v, m, G=1.3, delta=0.05, pot=phi)
    _check(out_b.cpu().numpy(), o["raw"], m, v)


def test_noalloc_rejects_what_it_cannot_serve(gpu):
    import torch
    n = 64
    pos, vel, mass = _cloud(n, 7)
    dpos, dvel, dmass = (torch.tensor(a, dtype=torch.float64, device="cuda") for a in (pos, vel, mass))
    dpot = torch.zeros(n, dtype=torch.float64, device="cuda")
    out = torch.empty(16, dtype=torch.float64, device="cuda")
    L = gpu.lib()
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    args = (dpos.data_ptr(), dvel.data_ptr(), dmass.data_ptr())
    # beyond the stated maximum: rejected before any memory is touched, with the limit in the message
    assert L.pp_invariants_noalloc(*args, dpot.data_ptr(), gpu.PP_NOALLOC_MAX_N + 1, gpu.PP_F64, out.data_ptr(), st) == -1
    assert b"PP_NOALLOC_MAX_N" in L.pp_last_error()
    assert L.pp_invariants_noalloc(*args, dpot.data_ptr(), 0, gpu.PP_F64, out.data_ptr(), st) == -1
    # no potential: that would need the allocating O(N^2) pass
    assert L.pp_invariants_noalloc(*args, None, n, gpu.PP_F64, out.data_ptr(), st) == -1
    assert b"pot is NULL" in L.pp_last_error()
    assert L.pp_invariants_noalloc(*args, dpot.data_ptr(), n, 9, out.data_ptr(), st) == -1
    assert L.pp_invariants_noalloc(*args, dpot.data_ptr(), n, gpu.PP_F64, None, st) == -1
    assert L.pp_invariants_noalloc(*args, dpot.data_ptr(), n, gpu.PP_F64, out.data_ptr(), st) == 0
    torch.cuda.synchronize()
    assert abs(float(out[12]) - float(dmass.sum())) <= 1e-14
