"""GPU tests of the i-sharded path ("each GPU calculates the dynamics of N/k
particles"): pp_forces_range and pp_kick_drift through the C ABI against the oracle and against the unsharded
entry points, and the ShardedSystem step logic on ONE GPU -- world_size 1, and several in-process shards driven
phase by phase (no rank ever waits on another: the exchange is a plain copy between the instances).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-5}


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("a -m gpu test was started without a CUDA device")
    from paper_1803_01190_b200 import ppgrav
    ppgrav.lib()
    return ppgrav


def _dt(prec):
    import torch
    return torch.float64 if prec == "f64" else torch.float32


def _cloud(n, seed):
    rng = np.random.Generator(np.random.Philox(key=seed))
    pos = rng.standard_normal((n, 3))
    vel = 0.1 * rng.standard_normal((n, 3))
    mass = rng.uniform(0.5, 1.5, size=n) / n
    mass[n // 2:] *= 4.0
    return pos, vel, mass


def _dev(prec, *arrays):
    import torch
    return tuple(torch.tensor(np.asarray(a), dtype=_dt(prec), device="cuda").contiguous() for a in arrays)


def _seen(prec, a):
    a = np.asarray(a)
    return a.astype(np.float64) if prec == "f64" else a.astype(np.float32).astype(np.float64)


def _rel_rows(got, ref):
    got = np.asarray(got, dtype=np.float64).reshape(len(ref), -1)
    ref = np.asarray(ref, dtype=np.float64).reshape(len(ref), -1)
    return float(np.max(np.linalg.norm(got - ref, axis=1) / np.linalg.norm(ref, axis=1)))


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n,ranges", [(5000, [(0, 1667), (1667, 1667), (3334, 1666)]),
                                      (4097, [(0, 1), (1, 2047), (2048, 2049)]),
                                      (700, [(699, 1), (0, 699)])])
def test_forces_range_matches_oracle_and_full_solve(gpu, oracle, prec, n, ranges):
    pos, _, mass = _cloud(n, 31)
    dpos, dmass = _dev(prec, pos, mass)
    G, delta = 1.7, 0.03
    a_ref, p_ref = oracle.forces(_seen(prec, pos), _seen(prec, mass), G=G, delta=delta, nthreads=0)
    # same j-tile size (shape class) and same j-split in every call => same summation order per body (include/ppgrav.h)
    gpu.pp_configure(gpu.PP_CFG_SPLIT_J, 2)
    gpu.pp_configure(gpu.PP_CFG_SHAPE, gpu.SHAPE_SMALL)
    try:
        a_full, p_full = gpu.pp_forces(dpos, dmass, G=G, delta=delta, want_pot=True)
        for b, c in ranges:
            a, p = gpu.pp_forces_range(dpos, dmass, b, c, G=G, delta=delta, want_pot=True)
            assert a.shape == (c, 3) and p.shape == (c,)
            assert _rel_rows(a.cpu().numpy(), a_ref[b:b + c]) <= TOL[prec]
            assert np.max(np.abs(p.cpu().numpy() - p_ref[b:b + c]) / np.abs(p_ref[b:b + c])) <= TOL[prec]
            assert np.array_equal(a.cpu().numpy(), a_full[b:b + c].cpu().numpy()), "range rows differ bitwise"
            assert np.array_equal(p.cpu().numpy(), p_full[b:b + c].cpu().numpy())
    finally:
        gpu.pp_configure(gpu.PP_CFG_SPLIT_J, 0)
        gpu.pp_configure(gpu.PP_CFG_SHAPE, 0)
    # automatic plan (shape class and split may differ from the full solve's): still within tolerance, force only
    b, c = ranges[-1]
    a, p = gpu.pp_forces_range(dpos, dmass, b, c, G=G, delta=delta)
    assert p is None and _rel_rows(a.cpu().numpy(), a_ref[b:b + c]) <= TOL[prec]


def test_forces_range_rejects_bad_ranges(gpu):
    import ctypes
    import torch
    pos = torch.zeros((10, 3), device="cuda", dtype=torch.float64)
    mass = torch.ones(10, device="cuda", dtype=torch.float64)
    acc = torch.empty((16, 3), device="cuda", dtype=torch.float64)
    lib = gpu.lib()
    for b, c in ((0, 0), (-1, 3), (8, 3), (10, 1), (0, 11)):
        rc = lib.pp_forces_range(pos.data_ptr(), mass.data_ptr(), acc.data_ptr(), None, 10, b, c, 1.0, 0.1,
                                 gpu.PP_F64, ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
        assert rc == -1 and b"range" in lib.pp_last_error()
    assert lib.pp_forces_range(pos.data_ptr(), mass.data_ptr(), acc.data_ptr(), None, 10, 7, 3, 1.0, 0.1,
                               gpu.PP_F64, ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)) == 0


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_kick_drift_is_the_fused_multiply_add_pair(gpu, prec):
    import torch
    n = 1000
    pos, vel, _ = _cloud(n, 7)
    acc = np.random.Generator(np.random.Philox(key=8)).standard_normal((n, 3))
    dpos, dvel, dacc = _dev(prec, pos, vel, acc)
    kick, dt = 0.5 * 1e-3, 1e-3
    # v' = fma(kick, a, v); r' = fma(dt, v', r) evaluated exactly in float64 and rounded once each
    npd = np.float64 if prec == "f64" else np.float32
    p0, v0, a0 = (x.cpu().numpy().astype(npd) for x in (dpos, dvel, dacc))
    gpu.pp_kick_drift(dpos, dvel, dacc, kick, dt)
    if prec == "f32":     # the double product/sum of floats is exact enough to reproduce a single rounding
        v1 = (npd(kick).astype(np.float64) * a0.astype(np.float64) + v0.astype(np.float64)).astype(npd)
        r1 = (npd(dt).astype(np.float64) * v1.astype(np.float64) + p0.astype(np.float64)).astype(npd)
        assert np.array_equal(dvel.cpu().numpy(), v1) and np.array_equal(dpos.cpu().numpy(), r1)
    else:
        v1 = kick * a0 + v0
        r1 = dt * v1 + p0
        assert np.abs(dvel.cpu().numpy() - v1).max() <= 2e-16 * np.abs(v1).max()
        assert np.abs(dpos.cpu().numpy() - r1).max() <= 2e-16 * np.abs(r1).max()
    # dt == 0: kick only, positions untouched
    before = dpos.clone()
    gpu.pp_kick_drift(dpos, dvel, dacc, kick, 0.0)
    assert torch.equal(dpos, before)


class _Loopback:
    """Stands in for a rank's communicator when several shards live in one process: the test copies the rows."""

    def __init__(self, world, rank):
        self.world, self.rank = world, rank

    def all_reduce_sum(self, t):
        return t


def _run_shards(gpu, prec, pos, vel, mass, world, dt, nsteps, G, delta):
    from paper_1803_01190_b200 import sharded
    dpos, dvel, dmass = _dev(prec, pos, vel, mass)
    shards = [sharded.ShardedSystem(dpos, dvel, dmass, G=G, delta=delta, comm=_Loopback(world, r), initial_pot=False)
              for r in range(world)]
    for s in range(nsteps):
        for sh in shards:
            sh.predict(dt)
        for sh in shards:                       # the all-gather, as plain copies between the instances
            for other in shards:
                if other is not sh:
                    sh.pos_all[other.row0:other.row0 + other.count].copy_(other.pos)
        for sh in shards:
            sh.solve(want_pot=(s == nsteps - 1))
            sh.correct(dt)
    return shards


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("world,n", [(1, 3001), (3, 3000), (3, 3001)])
def test_sharded_step_equals_single_gpu_step(gpu, oracle, prec, world, n):
    """world | N: the padded layout is the original one and the sharded run is bit-identical to pp_step_kdk; otherwise
    (3001 bodies on 3 ranks: one massless padding row in two of the blocks) equal to summation-order round-off."""
    import torch
    dt, nsteps, G, delta = 1e-3, 4, 1.0, 0.05
    pos, vel, mass = _cloud(n, 11)
    gpu.pp_configure(gpu.PP_CFG_SPLIT_J, 2)
    gpu.pp_configure(gpu.PP_CFG_SHAPE, gpu.SHAPE_MID)       # shards and the whole system on one shape class
    try:
        shards = _run_shards(gpu, prec, pos, vel, mass, world, dt, nsteps, G, delta)
        dpos, dvel, dmass = _dev(prec, pos, vel, mass)
        acc = torch.empty_like(dpos)
        pot = torch.empty_like(dmass)
        gpu.pp_step_kdk(dpos, dvel, dmass, acc, dt, nsteps, G=G, delta=delta, pot=pot)
    finally:
        gpu.pp_configure(gpu.PP_CFG_SPLIT_J, 0)
        gpu.pp_configure(gpu.PP_CFG_SHAPE, 0)
    for sh in shards:
        b, e = sh.begin, sh.begin + sh.count
        assert sh.force_evaluations == nsteps + 1                       # one solve per step
        assert torch.equal(sh.pos_all, shards[0].pos_all), "replicated positions diverged between the ranks"
        if n % world == 0:
            assert torch.equal(sh.positions(), dpos)
            assert torch.equal(sh.vel, dvel[b:e]) and torch.equal(sh.acc, acc[b:e]) and torch.equal(sh.pot, pot[b:e])
        else:
            rt = {"f64": 1e-13, "f32": 1e-5}[prec]
            assert (sh.positions() - dpos).abs().max() <= rt * dpos.abs().max()
            assert (sh.vel - dvel[b:e]).abs().max() <= rt * dvel.abs().max()
            assert _rel_rows(sh.acc.cpu().numpy(), acc[b:e].cpu().numpy()) <= 10 * rt
    # and against the oracle's trajectory
    p_ref, v_ref, _, _ = oracle.kdk_halfkick(_seen(prec, pos), _seen(prec, vel), _seen(prec, mass), dt, nsteps, G=G,
                                             delta=delta, nthreads=0)
    tol = 1e-11 if prec == "f64" else 5e-6
    assert np.abs(dpos.cpu().numpy() - p_ref).max() <= tol * np.abs(p_ref).max()
    # whole-system invariants from the shards' partial sums
    whole = gpu.invariants_dict(gpu.pp_invariants(dpos, dvel, dmass, G=G, delta=delta, pot=pot))
    parts = [sh.ops.invariants(sh.pos.contiguous(), sh.vel, sh.mass.contiguous(), sh.pot, G, delta).cpu().numpy()
             for sh in shards]
    E = sum(p[0] for p in parts)
    P = sum(p[3:6] for p in parts)
    M = sum(p[12] for p in parts)
    com = sum(p[9:12] * p[12] for p in parts) / M
    # (world does not divide N: the shards' potentials differ from the whole-system ones by summation-order round-off)
    loose = 1.0 if n % world == 0 or prec == "f64" else 1e6       # FP32 states that differ by FP32 round-off
    assert abs(E - whole["E"]) <= 1e-12 * loose * abs(whole["E"])
    assert np.abs(P - whole["P"]).max() <= 1e-14 * loose * float(np.sum(mass[:, None] * np.abs(vel)))
    assert abs(M - whole["M"]) <= 1e-14 * M and np.abs(com - whole["COM"]).max() <= 1e-13 * loose


def test_sharded_system_world1_invariants(gpu):
    import torch
    from paper_1803_01190_b200 import sharded
    pos, vel, mass = _cloud(2048, 5)
    dpos, dvel, dmass = _dev("f64", pos, vel, mass)
    sysm = sharded.ShardedSystem(dpos, dvel, dmass, G=1.0, delta=0.02)
    inv0 = sysm.invariants()
    torch.cuda.synchronize()
    n0 = gpu.pp_launch_count()
    sysm.step(1e-3, 5, want_pot=True)
    # per step: kick+drift, (tile masses, pack, sweep, finalize), closing kick -- and nothing for the exchange
    assert gpu.pp_launch_count() - n0 == 6 * 5
    inv1 = sysm.invariants()
    assert abs(inv1["E"] - inv0["E"]) <= 1e-6 * abs(inv0["E"])
    assert np.abs(inv1["P"] - inv0["P"]).max() <= 1e-15
    with pytest.raises(RuntimeError):
        sysm.step(1e-3, 1)
        sysm.invariants()
