"""GPU tests of PP_MIXED (an extension the paper's conclusion motivates): FP64
state and time integration around the FP32 pair sweep.  Forces are compared with the oracle evaluated on what the
sweep actually sees (positions and masses rounded to FP32, promoted exactly), at the FP32 tolerance of BASELINE.json;
trajectories with the oracle's FP64 trajectory."""
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


def _dev64(*arrays):
    import torch
    return tuple(torch.tensor(np.asarray(a), dtype=torch.float64, device="cuda").contiguous() for a in arrays)


def _rel_rows(got, ref):
    got, ref = np.asarray(got, dtype=np.float64), np.asarray(ref, dtype=np.float64)
    return np.linalg.norm(got - ref, axis=1) / np.linalg.norm(ref, axis=1)


@pytest.mark.parametrize("n", [1, 2, 129, 1537, 6000])
def test_mixed_forces_match_oracle_on_rounded_inputs(gpu, oracle, n):
    import torch
    rng = np.random.Generator(np.random.Philox(key=17))
    pos = rng.standard_normal((n, 3))
    mass = rng.uniform(0.5, 1.5, size=n) / n
    G, delta = 0.7, 0.04
    dpos, dmass = _dev64(pos, mass)
    acc, pot = gpu.pp_forces(dpos, dmass, G=G, delta=delta, want_pot=True, mixed=True)
    assert acc.dtype == torch.float64 and pot.dtype == torch.float64
    seen_p, seen_m = workloads.as_f32_exact(pos, mass)
    a_ref, p_ref = oracle.forces(seen_p, seen_m, G=G, delta=delta, nthreads=0)
    if n > 1:
        assert _rel_rows(acc.cpu().numpy(), a_ref).max() <= 2e-5
        assert (np.abs(pot.cpu().numpy() - p_ref) / np.abs(p_ref)).max() <= 2e-5
        # the sweep is the PP_F32 one: same sums, scaled by G in FP64 instead of FP32
        a32, p32 = gpu.pp_forces(dpos.float(), dmass.float(), G=G, delta=delta, want_pot=True)
        assert _rel_rows(acc.cpu().numpy(), a32.double().cpu().numpy()).max() <= 3e-7
    else:
        assert not acc.cpu().numpy().any() and not pot.cpu().numpy().any()
    # an i-range of the same solve
    if n >= 129:
        a_r, _ = gpu.pp_forces_range(dpos, dmass, 100, 29, G=G, delta=delta, mixed=True)
        assert _rel_rows(a_r.cpu().numpy(), a_ref[100:129]).max() <= 2e-5


def test_mixed_trajectory_config0(gpu, oracle):
    """10 KDK steps of config 0: the FP64 state integrates exactly like PP_F64; only the force carries FP32 error."""
    import torch
    c = workloads.config(0)
    pos, vel, mass = c["pos"], c["vel"], c["mass"]
    p_ref, v_ref, _, _ = oracle.kdk_halfkick(pos, vel, mass, c["dt"], 10, G=c["G"], delta=c["delta"], nthreads=0)
    out = {}
    for name, mixed, dt in (("mixed", True, torch.float64), ("f32", False, torch.float32)):
        dpos, dvel, dmass = (torch.tensor(a, dtype=dt, device="cuda") for a in (pos, vel, mass))
        acc = torch.empty_like(dpos)
        pot = torch.empty_like(dmass)
        gpu.pp_step_kdk(dpos, dvel, dmass, acc, c["dt"], 10, G=c["G"], delta=c["delta"], pot=pot, mixed=mixed)
        out[name] = (np.abs(dpos.double().cpu().numpy() - p_ref).max() / np.abs(p_ref).max(),
                     np.abs(dvel.double().cpu().numpy() - v_ref).max() / np.abs(v_ref).max())
        if mixed:
            inv = gpu.invariants_dict(gpu.pp_invariants(dpos, dvel, dmass, G=c["G"], delta=c["delta"], pot=pot))
            ref = oracle.invariants(dpos.cpu().numpy(), dvel.cpu().numpy(), mass, G=c["G"], delta=c["delta"],
                                    nthreads=0)
            assert abs(inv["K"] - ref["K"]) <= 1e-12 * ref["K"]
            assert abs(inv["W"] - ref["W"]) <= 2e-6 * abs(ref["W"])        # FP32-sweep potential
    assert out["mixed"][0] <= 1e-8 and out["mixed"][1] <= 1e-6, out
    assert out["mixed"][0] < out["f32"][0], out          # the state no longer rounds r += dt v to FP32


def test_mixed_host_entry_and_argument_checks(gpu):
    import ctypes
    import torch
    c = workloads.config(0)
    pos, mass = np.ascontiguousarray(c["pos"]), np.ascontiguousarray(c["mass"])
    acc = np.empty_like(pos)
    lib = gpu.lib()
    rc = lib.pp_forces_host(pos.ctypes.data, mass.ctypes.data, acc.ctypes.data, None, len(mass), 1.0, 0.02,
                            gpu.PP_MIXED, None)
    assert rc == 0
    dacc, _ = gpu.pp_forces(*_dev64(pos, mass), delta=0.02, mixed=True)
    assert np.array_equal(acc, dacc.cpu().numpy())
    with pytest.raises(TypeError):
        gpu.pp_forces(torch.zeros((4, 3), device="cuda"), torch.ones(4, device="cuda"), delta=0.1, mixed=True)
    buf = torch.zeros(64, device="cuda", dtype=torch.float32)
    rc = lib.pp_forces(buf.data_ptr() + 4, buf.data_ptr() + 128, buf.data_ptr() + 160, None, 2, 1.0, 0.1, gpu.PP_MIXED,
                       ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == -1 and b"aligned" in lib.pp_last_error()
    assert lib.pp_forces(buf.data_ptr(), buf.data_ptr() + 128, buf.data_ptr() + 160, None, 2, 1.0, 0.1, 3,
                         ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)) == -1
