"""GPU parity tests: libppgrav (through its C ABI, via the ctypes binding) against the CPU oracle, element by element
on the same seeded inputs.  Tolerances are BASELINE.json's: accelerations within 1e-12 (FP64) / 2e-5 (FP32) of the
oracle, relative to |a_i| (max over all checked i).  FP32 runs are compared with the oracle evaluated on the
FP32-rounded inputs promoted exactly to double.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_ACC = {"f64": 1e-12, "f32": 2e-5}
TOL_POT = {"f64": 1e-12, "f32": 2e-5}


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("a -m gpu test was started without a CUDA device")
    from paper_1803_01190_b200 import ppgrav
    ppgrav.lib()           # raises if the extension has not been built: no fallback
    return ppgrav


def _torch_dtype(prec):
    import torch
    return torch.float64 if prec == "f64" else torch.float32


def _to_dev(prec, *arrays):
    import torch
    return tuple(torch.tensor(np.asarray(a), dtype=_torch_dtype(prec), device="cuda").contiguous() for a in arrays)


def _inputs_seen(prec, *arrays):
    """float64 copies of what the GPU run of this precision actually receives."""
    if prec == "f64":
        return tuple(np.asarray(a, dtype=np.float64) for a in arrays)
    return tuple(np.asarray(a, dtype=np.float32).astype(np.float64) for a in arrays)


def rel_err_rows(got, ref):
    """max_i |got_i - ref_i| / |ref_i| with the Euclidean norm over the row."""
    got = np.asarray(got, dtype=np.float64).reshape(len(ref), -1)
    ref = np.asarray(ref, dtype=np.float64).reshape(len(ref), -1)
    num = np.linalg.norm(got - ref, axis=1)
    den = np.linalg.norm(ref, axis=1)
    return float(np.max(num / den)) if len(ref) else 0.0


def _random_cloud(n, seed, two_species=True):
    rng = np.random.Generator(np.random.Philox(key=seed))
    pos = rng.standard_normal((n, 3))
    vel = 0.1 * rng.standard_normal((n, 3))
    mass = rng.uniform(0.5, 1.5, size=n) / n
    if two_species:
        mass[n // 2:] *= 4.0
    return pos, vel, mass


# ---- pp_forces ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_forces_config0_all_bodies(gpu, oracle, prec):
    from paper_1803_01190_b200 import workloads
    c = workloads.config(0)
    pos, mass = _inputs_seen(prec, c["pos"], c["mass"])
    a_ref, p_ref = oracle.forces(pos, mass, G=c["G"], delta=c["delta"], nthreads=0)
    dpos, dmass = _to_dev(prec, pos, mass)
    acc, pot = gpu.pp_forces(dpos, dmass, G=c["G"], delta=c["delta"], want_pot=True)
    assert rel_err_rows(acc.cpu().numpy(), a_ref) <= TOL_ACC[prec]
    assert rel_err_rows(pot.cpu().numpy(), p_ref) <= TOL_POT[prec]
    acc2, none = gpu.pp_forces(dpos, dmass, G=c["G"], delta=c["delta"], want_pot=False)   # force-only kernel
    assert none is None
    assert rel_err_rows(acc2.cpu().numpy(), a_ref) <= TOL_ACC[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [1, 2, 3, 127, 128, 129, 255, 257, 511, 513, 1000, 1535, 1537, 3001, 5000])
@pytest.mark.parametrize("split", [0, 1, 3])
def test_forces_ragged_sizes_and_splits(gpu, oracle, prec, n, split):
    """Sizes around the tile and i-block edge of the SMALL shape class (128 bodies; the plan picks it for every N here),
    automatic and forced split-j, two mass species, G != 1.  The same edges of the mid and large classes (256/512-body
    tiles, 512/1536/1792-body i-blocks) are covered in tests/test_gpu_shapes.py with the class pinned."""
    pos, _, mass = _random_cloud(n, 100 + n)
    pos, mass = _inputs_seen(prec, pos, mass)
    a_ref, p_ref = oracle.forces(pos, mass, G=2.5, delta=0.05, nthreads=0)
    dpos, dmass = _to_dev(prec, pos, mass)
    gpu.pp_configure(gpu.PP_CFG_SPLIT_J, split)
    try:
        acc, pot = gpu.pp_forces(dpos, dmass, G=2.5, delta=0.05, want_pot=True)
        acc2, _ = gpu.pp_forces(dpos, dmass, G=2.5, delta=0.05, want_pot=False)
    finally:
        gpu.pp_configure(gpu.PP_CFG_SPLIT_J, 0)
    if n == 1:
        assert np.all(acc.cpu().numpy() == 0.0) and np.all(pot.cpu().numpy() == 0.0)
        assert np.all(acc2.cpu().numpy() == 0.0)
        return
    assert rel_err_rows(acc.cpu().numpy(), a_ref) <= TOL_ACC[prec]
    assert rel_err_rows(acc2.cpu().numpy(), a_ref) <= TOL_ACC[prec]
    assert rel_err_rows(pot.cpu().numpy(), p_ref) <= TOL_POT[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_forces_delta_zero_guarded(gpu, oracle, prec):
    """delta = 0 (guarded kernels): distinct bodies match the oracle; a coincident pair contributes nothing to each
    other (reading R2) and everything stays finite."""
    pos, _, mass = _random_cloud(700, 7)
    pos, mass = _inputs_seen(prec, pos, mass)
    a_ref, p_ref = oracle.forces(pos, mass, G=1.0, delta=0.0, nthreads=0)
    dpos, dmass = _to_dev(prec, pos, mass)
    acc, pot = gpu.pp_forces(dpos, dmass, delta=0.0, want_pot=True)
    assert rel_err_rows(acc.cpu().numpy(), a_ref) <= TOL_ACC[prec]
    assert rel_err_rows(pot.cpu().numpy(), p_ref) <= TOL_POT[prec]
    # coincident bodies 0 and 1: the oracle is asked for body 0 with body 1 made massless, and vice versa
    pos[1] = pos[0]
    dpos, dmass = _to_dev(prec, pos, mass)
    acc, pot = gpu.pp_forces(dpos, dmass, delta=0.0, want_pot=True)
    acc, pot = acc.cpu().numpy(), pot.cpu().numpy()
    assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot))
    for me, other in ((0, 1), (1, 0)):
        m2 = mass.copy()
        m2[other] = 0.0
        p2 = pos.copy()
        p2[other] += 1.0           # anywhere else: it is massless
        a1, p1 = oracle.forces(p2, m2, delta=0.0, idx=np.array([me]))
        assert rel_err_rows(acc[me:me + 1], a1) <= TOL_ACC[prec]
        assert rel_err_rows(pot[me:me + 1], p1) <= TOL_POT[prec]


def test_forces_bit_reproducible_and_host_variant(gpu):
    import torch
    pos, _, mass = _random_cloud(4099, 11)
    for prec in ("f64", "f32"):
        dpos, dmass = _to_dev(prec, pos, mass)
        a1, p1 = gpu.pp_forces(dpos, dmass, delta=0.01, want_pot=True)
        a2, p2 = gpu.pp_forces(dpos, dmass, delta=0.01, want_pot=True)
        assert torch.equal(a1, a2) and torch.equal(p1, p2)
        ah, ph = gpu.pp_forces_host(dpos.cpu().numpy(), dmass.cpu().numpy(), delta=0.01, want_pot=True)
        assert np.array_equal(ah, a1.cpu().numpy()) and np.array_equal(ph, p1.cpu().numpy())


def test_forces_rejects_bad_arguments(gpu):
    import torch
    pos, _, mass = _random_cloud(16, 3)
    dpos, dmass = _to_dev("f64", pos, mass)
    with pytest.raises(gpu.PPGravError):
        gpu.pp_forces(dpos, dmass, delta=-1.0)
    with pytest.raises(gpu.PPGravError):
        gpu.pp_forces(dpos, dmass, G=float("nan"))
    L = gpu.lib()
    assert L.pp_forces(None, dmass.data_ptr(), dpos.data_ptr(), None, 16, 1.0, 0.0, gpu.PP_F64, None) == -1
    assert L.pp_forces(dpos.data_ptr(), dmass.data_ptr(), dpos.data_ptr() + 4, None, 16, 1.0, 0.0, gpu.PP_F64,
                       None) == -1
    assert L.pp_forces(dpos.data_ptr(), dmass.data_ptr(), dpos.data_ptr(), None, 0, 1.0, 0.0, gpu.PP_F64, None) == -1
    assert L.pp_forces(dpos.data_ptr(), dmass.data_ptr(), dpos.data_ptr(), None, 16, 1.0, 0.0, 7, None) == -1
    assert b"precision" in L.pp_last_error()
    torch.cuda.synchronize()


# ---- equal-mass j-tiles (m_j taken out of the pair loop) -----------------------------------------------------------
def _species_cloud(n, seed, bounds, masses):
    """n bodies in mass species: bodies [bounds[k], bounds[k+1]) all have mass masses[k] (exactly)."""
    pos, vel, _ = _random_cloud(n, seed)
    mass = np.empty(n)
    edges = list(bounds) + [n]
    for k, m in enumerate(masses):
        mass[edges[k]:edges[k + 1]] = m
    return pos, vel, mass


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n,bounds", [(3001, (0, 1300)), (40003, (0, 700, 21000)), (1537, (0,))])
def test_equal_mass_tiles_against_oracle_and_general_path(gpu, oracle, prec, n, bounds):
    """Species boundaries off the tile grid and a ragged tail: tiles inside one species run without the per-pair
    m_j, the straddling tiles and the padded last tile with it.  Both settings of PP_CFG_EQUAL_MASS must meet the
    oracle; they differ from each other by summation round-off only."""
    masses = [1.0 / n, 4.0 / n, 0.25 / n][:len(bounds)]
    pos, vel, mass = _species_cloud(n, 77 + n, bounds, masses)
    pos, mass = _inputs_seen(prec, pos, mass)
    a_ref, p_ref = oracle.forces(pos, mass, G=1.5, delta=0.03, nthreads=0)
    dpos, dmass = _to_dev(prec, pos, mass)
    tile_j = gpu.pp_plan_query(n, gpu.PP_F64 if prec == "f64" else gpu.PP_F32)["tile_j"]
    edges = list(bounds) + [n]
    expect = sum(1 for t in range((n + tile_j - 1) // tile_j)
                 if (t + 1) * tile_j <= n and any(edges[k] <= t * tile_j and (t + 1) * tile_j <= edges[k + 1]
                                                  for k in range(len(bounds))))
    assert gpu.pp_equal_mass_tiles(dmass) == ((n + tile_j - 1) // tile_j, expect) and expect > 0
    res = {}
    try:
        for flag in (1, 0):
            gpu.pp_configure(gpu.PP_CFG_EQUAL_MASS, flag)
            acc, pot = gpu.pp_forces(dpos, dmass, G=1.5, delta=0.03, want_pot=True)
            acc2, _ = gpu.pp_forces(dpos, dmass, G=1.5, delta=0.03, want_pot=False)
            assert rel_err_rows(acc.cpu().numpy(), a_ref) <= TOL_ACC[prec]
            assert rel_err_rows(acc2.cpu().numpy(), a_ref) <= TOL_ACC[prec]
            assert rel_err_rows(pot.cpu().numpy(), p_ref) <= TOL_POT[prec]
            res[flag] = (acc.cpu().numpy(), pot.cpu().numpy())
    finally:
        gpu.pp_configure(gpu.PP_CFG_EQUAL_MASS, 1)
    assert not np.array_equal(res[0][0], res[1][0])          # the two paths really are different instruction streams
    assert rel_err_rows(res[1][0], res[0][0]) <= {"f64": 1e-13, "f32": 1e-5}[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_mixed_mass_tiles_do_not_depend_on_the_switch(gpu, prec):
    """No tile of a random-mass cloud has a common mass: PP_CFG_EQUAL_MASS on/off are then bit-identical."""
    pos, vel, mass = _random_cloud(3001, 13)
    dpos, dmass = _to_dev(prec, pos, mass)
    assert gpu.pp_equal_mass_tiles(dmass)[1] == 0
    outs = []
    try:
        for flag in (1, 0):
            gpu.pp_configure(gpu.PP_CFG_EQUAL_MASS, flag)
            outs.append(gpu.pp_forces(dpos, dmass, delta=0.05, want_pot=True))
    finally:
        gpu.pp_configure(gpu.PP_CFG_EQUAL_MASS, 1)
    import torch
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])


def test_equal_mass_tiles_delta_zero_and_massless(gpu, oracle):
    """Guarded (delta = 0) kernels and an all-massless species go through the equal-mass path too."""
    n = 2048
    pos, vel, mass = _species_cloud(n, 5, (0, 1024), [1.0 / n, 0.0])
    a_ref, p_ref = oracle.forces(pos, mass, delta=0.0, nthreads=0)
    for prec in ("f64", "f32"):
        p, m = _inputs_seen(prec, pos, mass)
        ar, pr = (a_ref, p_ref) if prec == "f64" else oracle.forces(p, m, delta=0.0, nthreads=0)
        dpos, dmass = _to_dev(prec, p, m)
        assert gpu.pp_equal_mass_tiles(dmass)[1] == gpu.pp_equal_mass_tiles(dmass)[0]
        acc, pot = gpu.pp_forces(dpos, dmass, delta=0.0, want_pot=True)
        assert rel_err_rows(acc.cpu().numpy(), ar) <= TOL_ACC[prec]
        assert rel_err_rows(pot.cpu().numpy(), pr) <= TOL_POT[prec]


# ---- pp_step_kdk -------------------------------------------------------------------------------------------------
TOL_TRAJ = {"f64": 1e-11, "f32": 5e-6}


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_kdk_config0_trajectory(gpu, oracle, prec):
    """Config 0: 10 KDK steps, dt = 1e-3; final pos/vel/acc against the oracle started from the same state."""
    import torch
    from paper_1803_01190_b200 import workloads
    c = workloads.config(0)
    pos, vel, mass = _inputs_seen(prec, c["pos"], c["vel"], c["mass"])
    p_ref, v_ref, a_ref, nforce = oracle.kdk_halfkick(pos, vel, mass, c["dt"], c["nsteps"], G=c["G"],
                                                      delta=c["delta"], nthreads=0)
    assert nforce == c["nsteps"] + 1
    dpos, dvel, dmass = _to_dev(prec, pos, vel, mass)
    dacc = torch.zeros_like(dpos)
    dpot = torch.empty_like(dmass)
    n0 = gpu.pp_launch_count()
    gpu.pp_step_kdk(dpos, dvel, dmass, dacc, c["dt"], c["nsteps"], G=c["G"], delta=c["delta"], pot=dpot)
    torch.cuda.synchronize()
    # one gravity solve per step + the cold-start solve: tile masses once per call, (pack, sweep,
    # finalize) for the cold start, kick+drift+pack, (sweep, fused update) per interior step, (sweep, finalize+kick)
    assert gpu.pp_launch_count() - n0 == 5 + 2 * c["nsteps"]
    scale_r, scale_v = np.abs(p_ref).max(), np.abs(v_ref).max()
    assert np.abs(dpos.cpu().numpy() - p_ref).max() / scale_r <= TOL_TRAJ[prec]
    assert np.abs(dvel.cpu().numpy() - v_ref).max() / scale_v <= TOL_TRAJ[prec]
    assert rel_err_rows(dacc.cpu().numpy(), a_ref) <= 10 * TOL_ACC[prec]     # a(t_end) of slightly different states
    _, pot_ref = oracle.forces(p_ref, mass, G=c["G"], delta=c["delta"], nthreads=0)
    assert rel_err_rows(dpot.cpu().numpy(), pot_ref) <= 10 * TOL_POT[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("graph", [0, 1])
def test_kdk_restart_and_graph_are_bitwise_identical(gpu, prec, graph):
    """10 steps in one call == 4 + 6 steps with PP_ACC_VALID, with and without CUDA-graph replay, on a side stream."""
    import torch
    pos, vel, mass = _random_cloud(1500, 21)
    st = torch.cuda.Stream()
    outs = []
    gpu.pp_configure(gpu.PP_CFG_GRAPH, graph)
    try:
        for chunks in ((10,), (4, 6)):
            dpos, dvel, dmass = _to_dev(prec, pos, vel, mass)
            dacc = torch.zeros_like(dpos)
            torch.cuda.synchronize()
            with torch.cuda.stream(st):
                for k, n in enumerate(chunks):
                    gpu.pp_step_kdk(dpos, dvel, dmass, dacc, 1e-3, n, delta=0.05, acc_valid=(k > 0))
            st.synchronize()
            outs.append((dpos.clone(), dvel.clone(), dacc.clone()))
    finally:
        gpu.pp_configure(gpu.PP_CFG_GRAPH, 1)
    for a, b in zip(outs[0], outs[1]):
        assert torch.equal(a, b)
    key = "ref_%s" % prec
    if not hasattr(test_kdk_restart_and_graph_are_bitwise_identical, key):
        setattr(test_kdk_restart_and_graph_are_bitwise_identical, key, outs[0])
    else:
        for a, b in zip(outs[0], getattr(test_kdk_restart_and_graph_are_bitwise_identical, key)):
            assert torch.equal(a, b)


def test_kdk_nsteps_zero_and_host_variant(gpu, oracle):
    import torch
    pos, vel, mass = _random_cloud(600, 5)
    dpos, dvel, dmass = _to_dev("f64", pos, vel, mass)
    dacc = torch.zeros_like(dpos)
    gpu.pp_step_kdk(dpos, dvel, dmass, dacc, 1e-3, 0, delta=0.05)       # only computes acc
    a_ref, _ = oracle.forces(pos, mass, delta=0.05)
    assert rel_err_rows(dacc.cpu().numpy(), a_ref) <= 1e-12
    assert np.array_equal(dpos.cpu().numpy(), pos) and np.array_equal(dvel.cpu().numpy(), vel)
    dpot = torch.empty_like(dmass)
    gpu.pp_step_kdk(dpos, dvel, dmass, dacc, 1e-3, 7, delta=0.05, acc_valid=True, pot=dpot)
    hp, hv, ha = pos.copy(), vel.copy(), np.zeros_like(pos)
    hpot = np.zeros_like(mass)
    gpu.pp_step_kdk_host(hp, hv, mass, ha, 1e-3, 7, delta=0.05, pot=hpot)
    assert np.array_equal(hp, dpos.cpu().numpy()) and np.array_equal(hv, dvel.cpu().numpy())
    assert np.array_equal(ha, dacc.cpu().numpy()) and np.array_equal(hpot, dpot.cpu().numpy())
    _, p_ref = oracle.forces(hp, mass, delta=0.05)
    assert rel_err_rows(hpot, p_ref) <= 1e-12


# ---- pp_invariants -----------------------------------------------------------------------------------------------
def _check_invariants(gpu_out, ref, mass, vel):
    g = np.asarray(gpu_out, dtype=np.float64)
    r = ref["raw"]
    for k in (0, 1, 2):                                  # E, K, W
        assert abs(g[k] - r[k]) <= 1e-12 * abs(r[k])
    p_scale = float(np.sum(np.abs(mass)[:, None] * np.abs(vel)))
    assert np.abs(g[3:6] - r[3:6]).max() <= 1e-14 * p_scale       # P is ~0 by construction: absolute
    l_scale = np.abs(r[6:9]).max()
    assert np.abs(g[6:9] - r[6:9]).max() <= 1e-12 * l_scale
    assert np.abs(g[9:12] - r[9:12]).max() <= 1e-13
    assert abs(g[12] - r[12]) <= 1e-14 * r[12]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_invariants_config0_against_oracle(gpu, oracle, prec):
    from paper_1803_01190_b200 import workloads
    c = workloads.config(0)
    pos, vel, mass = _inputs_seen(prec, c["pos"], c["vel"], c["mass"])
    ref = oracle.invariants(pos, vel, mass, G=c["G"], delta=c["delta"], nthreads=0)
    dpos, dvel, dmass = _to_dev(prec, pos, vel, mass)
    out = gpu.pp_invariants(dpos, dvel, dmass, G=c["G"], delta=c["delta"])          # FP64 O(N^2) potential pass
    _check_invariants(out.cpu().numpy(), ref, mass, vel)
    host = gpu.pp_invariants_host(dpos.cpu().numpy(), dvel.cpu().numpy(), dmass.cpu().numpy(), G=c["G"],
                                  delta=c["delta"])
    assert np.array_equal(host, out.cpu().numpy())
    # supplied potential (state precision): the oracle is given the same potential values
    _, dpot = gpu.pp_forces(dpos, dmass, G=c["G"], delta=c["delta"], want_pot=True)
    out2 = gpu.pp_invariants(dpos, dvel, dmass, G=c["G"], delta=c["delta"], pot=dpot)
    ref2 = oracle.invariants(pos, vel, mass, G=c["G"], delta=c["delta"], pot=dpot.cpu().numpy().astype(np.float64))
    _check_invariants(out2.cpu().numpy(), ref2, mass, vel)


@pytest.mark.parametrize("n", [1, 2, 255, 300, 30011])
def test_invariants_ragged_sizes(gpu, oracle, n):
    pos, vel, mass = _random_cloud(n, 900 + n)
    pos += 0.3                                            # COM != 0
    if n == 1:
        ref = oracle.invariants(pos, vel, mass, delta=0.1, pot=np.zeros(1))
    else:
        ref = oracle.invariants(pos, vel, mass, delta=0.1, nthreads=0)
    dpos, dvel, dmass = _to_dev("f64", pos, vel, mass)
    out = gpu.pp_invariants(dpos, dvel, dmass, delta=0.1).cpu().numpy()
    if n == 1:
        assert out[2] == 0.0
    _check_invariants(out, ref, mass, vel)
