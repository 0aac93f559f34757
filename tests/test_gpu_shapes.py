"""GPU parity on EVERY kernel shape class, above all the large one that bench.py times (force_f32_kernel<256,7,512,...>,
force_f64_kernel<256,6|7,256,...>): the launch plan picks the large class only from N ~ 2^16 up, so the edge cases
(ragged sizes around the tile and i-block edges, forced split-j, delta = 0, tiny delta, off-block i-ranges, PP_MIXED,
equal-mass tiles) are run with PP_CFG_SHAPE pinning the class at sizes the oracle sweeps in full, and again at sizes
where the plan chooses the class by itself.  Every test asserts through pp_plan_query which shape it is running.

Tolerances: BASELINE.json's 1e-12 (FP64) / 2e-5 (FP32) of |a_i|, the same for Phi_i; trajectories: DESIGN.md section 6.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-5}
TOL_TRAJ = {"f64": 1e-11, "f32": 5e-6}
I_PER_CTA_MIN = {"large": 1536, "mid": 512}


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("a -m gpu test was started without a CUDA device")
    from paper_1803_01190_b200 import ppgrav
    ppgrav.lib()
    yield ppgrav
    ppgrav.pp_configure(ppgrav.PP_CFG_SHAPE, 0)
    ppgrav.pp_configure(ppgrav.PP_CFG_SPLIT_J, 0)
    ppgrav.pp_configure(ppgrav.PP_CFG_SYMMETRIC, 1)


def _dtype(prec):
    import torch
    return torch.float64 if prec == "f64" else torch.float32


def _dev(prec, *arrays):
    import torch
    return tuple(torch.tensor(np.asarray(a), dtype=_dtype(prec), device="cuda").contiguous() for a in arrays)


def _seen(prec, *arrays):
    if prec == "f64":
        return tuple(np.asarray(a, dtype=np.float64) for a in arrays)
    return tuple(np.asarray(a, dtype=np.float32).astype(np.float64) for a in arrays)


def _rel(got, ref):
    got = np.asarray(got, dtype=np.float64).reshape(len(ref), -1)
    ref = np.asarray(ref, dtype=np.float64).reshape(len(ref), -1)
    return float(np.max(np.linalg.norm(got - ref, axis=1) / np.linalg.norm(ref, axis=1))) if len(ref) else 0.0


def _cloud(n, seed, masses="random"):
    """masses: "random" = all different, two species by a factor 4 (no j-tile has a common mass);
    "species" = three exact mass values with boundaries off every tile grid (most tiles take the equal-mass path)."""
    rng = np.random.Generator(np.random.Philox(key=seed))
    pos = rng.standard_normal((n, 3))
    vel = 0.1 * rng.standard_normal((n, 3))
    if masses == "random":
        mass = rng.uniform(0.5, 1.5, size=n) / n
        mass[n // 2:] *= 4.0
    else:
        mass = np.full(n, 1.0 / n)
        mass[n // 3 + 5:] = 4.0 / n
        mass[(3 * n) // 4 + 1:] = 0.25 / n
    return pos, vel, mass


class _Pinned:
    """Pins the shape class (and optionally split-j) for the duration of a with-block and checks the plan."""

    def __init__(self, gpu, shape, split=0):
        self.gpu, self.shape, self.split = gpu, shape, split

    def __enter__(self):
        g = self.gpu
        g.pp_configure(g.PP_CFG_SHAPE, {"auto": 0, "large": 1, "mid": 2, "small": 3}[self.shape])
        g.pp_configure(g.PP_CFG_SPLIT_J, self.split)
        return self

    def __exit__(self, *exc):
        self.gpu.pp_configure(self.gpu.PP_CFG_SHAPE, 0)
        self.gpu.pp_configure(self.gpu.PP_CFG_SPLIT_J, 0)

    def check(self, n, prec, with_pot):
        p = self.gpu.pp_plan_query(n, self.gpu.PP_F64 if prec == "f64" else self.gpu.PP_F32, with_pot)
        if self.shape in I_PER_CTA_MIN:
            assert p["i_per_cta"] >= I_PER_CTA_MIN[self.shape], p
            assert p["shape"] == {"large": 0, "mid": 1}[self.shape]
        return p


_oracle_cache = {}


def _oracle_forces(oracle, key, pos, mass, G, delta):
    if key not in _oracle_cache:
        _oracle_cache[key] = oracle.forces(pos, mass, G=G, delta=delta, nthreads=0)
    return _oracle_cache[key]


# sizes around the j-tile (256 / 512) and i-block (512 / 1536 / 1792) edges of the large and mid shapes, one i-block and
# several, with a ragged last tile and a ragged last i-block
EDGE_N = [1, 2, 255, 257, 511, 513, 1535, 1537, 1791, 1793, 3071, 3073, 3583, 3585, 5377]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("shape", ["large", "mid"])
@pytest.mark.parametrize("n", EDGE_N)
def test_edge_sizes_forced_splits_on_pinned_shape(gpu, oracle, prec, shape, n):
    """Ragged N x split-j {auto, 1, 3, 7} x {random masses, mass species} x {with, without potential}, G != 1."""
    for masses in ("random", "species"):
        pos, _, mass = _cloud(n, 4000 + n, masses)
        pos, mass = _seen(prec, pos, mass)
        a_ref, p_ref = _oracle_forces(oracle, (n, prec, masses), pos, mass, 2.5, 0.05)
        dpos, dmass = _dev(prec, pos, mass)
        for split in (0, 1, 3, 7):
            with _Pinned(gpu, shape, split) as pin:
                plan = pin.check(n, prec, True)
                if split:
                    assert plan["split"] == min(split, -(-n // plan["tile_j"]))
                acc, pot = gpu.pp_forces(dpos, dmass, G=2.5, delta=0.05, want_pot=True)
                acc2, _ = gpu.pp_forces(dpos, dmass, G=2.5, delta=0.05, want_pot=False)
            if n == 1:
                assert np.all(acc.cpu().numpy() == 0.0) and np.all(pot.cpu().numpy() == 0.0)
                assert np.all(acc2.cpu().numpy() == 0.0)
                continue
            assert _rel(acc.cpu().numpy(), a_ref) <= TOL[prec], (masses, split)
            assert _rel(acc2.cpu().numpy(), a_ref) <= TOL[prec], (masses, split)
            assert _rel(pot.cpu().numpy(), p_ref) <= TOL[prec], (masses, split)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [2 ** 17 + 1, 125439])
def test_ragged_sizes_where_the_plan_picks_the_bench_kernels(gpu, oracle, prec, n):
    """No pinning: at N = 2^17 + 1 and 70 x 1792 - 1 the plan itself chooses the symmetric sweep and, with
    PP_CFG_SYMMETRIC off, the large one-sided class -- the two kernels bench.py times.  8192 sampled bodies against
    the oracle (1e9 pairs), with and without the potential."""
    pos, _, mass = _cloud(n, 17 + n, "species")
    pos, mass = _seen(prec, pos, mass)
    idx = np.sort(np.random.Generator(np.random.Philox(key=n)).choice(n, size=8192, replace=False))
    a_ref, p_ref = oracle.forces(pos, mass, G=1.0, delta=0.01, idx=idx, nthreads=0)
    dpos, dmass = _dev(prec, pos, mass)
    try:
        for symmetric, shape in ((1, 3), (0, 0)):
            gpu.pp_configure(gpu.PP_CFG_SYMMETRIC, symmetric)
            for with_pot in (True, False):
                p = gpu.pp_plan_query(n, gpu.PP_F64 if prec == "f64" else gpu.PP_F32, with_pot)
                assert p["shape"] == shape and p["i_per_cta"] >= 1536, p
                acc, pot = gpu.pp_forces(dpos, dmass, delta=0.01, want_pot=with_pot)
                assert _rel(acc[idx].cpu().numpy(), a_ref) <= TOL[prec]
                if with_pot:
                    assert _rel(pot[idx].cpu().numpy(), p_ref) <= TOL[prec]
    finally:
        gpu.pp_configure(gpu.PP_CFG_SYMMETRIC, 1)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("shape", ["large", "mid", "small"])
@pytest.mark.parametrize("masses", ["random", "species"])
def test_delta_zero_guarded_kernels_on_every_shape(gpu, oracle, prec, shape, masses):
    """delta = 0 selects the GUARD instantiations (with and without potential, mixed-mass and equal-mass tiles):
    distinct bodies match the oracle; a coincident pair contributes nothing to each other and all stays finite."""
    n = 4001
    pos, _, mass = _cloud(n, 91, masses)
    pos, mass = _seen(prec, pos, mass)
    a_ref, p_ref = oracle.forces(pos, mass, G=1.0, delta=0.0, nthreads=0)
    dpos, dmass = _dev(prec, pos, mass)
    with _Pinned(gpu, shape) as pin:
        pin.check(n, prec, True)
        acc, pot = gpu.pp_forces(dpos, dmass, delta=0.0, want_pot=True)
        acc2, _ = gpu.pp_forces(dpos, dmass, delta=0.0, want_pot=False)
        assert _rel(acc.cpu().numpy(), a_ref) <= TOL[prec]
        assert _rel(acc2.cpu().numpy(), a_ref) <= TOL[prec]
        assert _rel(pot.cpu().numpy(), p_ref) <= TOL[prec]
        # coincident bodies 7 and 2900 (different i-blocks and j-tiles of every shape)
        a, b = 7, 2900
        pos2 = pos.copy()
        pos2[b] = pos2[a]
        dpos2, = _dev(prec, pos2)
        acc, pot = gpu.pp_forces(dpos2, dmass, delta=0.0, want_pot=True)
        acc2, _ = gpu.pp_forces(dpos2, dmass, delta=0.0, want_pot=False)
    acc, pot, acc2 = acc.cpu().numpy(), pot.cpu().numpy(), acc2.cpu().numpy()
    assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot)) and np.all(np.isfinite(acc2))
    for me, other in ((a, b), (b, a)):
        m2 = mass.copy()
        m2[other] = 0.0                      # the oracle is asked for `me` with its twin made massless and moved away
        p2 = pos2.copy()
        p2[other] += 1.0
        a1, p1 = oracle.forces(p2, m2, delta=0.0, idx=np.array([me]))
        assert _rel(acc[me:me + 1], a1) <= TOL[prec] and _rel(acc2[me:me + 1], a1) <= TOL[prec]
        assert _rel(pot[me:me + 1], p1) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("delta", [1e-15, 1e-12, 3e-9])
def test_tiny_nonzero_delta_is_finite_and_matches_the_oracle(gpu, oracle, prec, delta):
    """0 < delta below ~1e-13 made the FP32 self term overflow (w^3 = inf, inf x 0 = NaN).  The guarded
    kernels now take every delta^2 below 1e-20 (FP32) / 1e-200 (FP64); distinct bodies are unaffected."""
    n = 3000
    pos, _, mass = _cloud(n, 23)
    pos, mass = _seen(prec, pos, mass)
    a_ref, p_ref = oracle.forces(pos, mass, delta=delta, nthreads=0)
    dpos, dmass = _dev(prec, pos, mass)
    for shape in ("large", "small"):
        with _Pinned(gpu, shape):
            acc, pot = gpu.pp_forces(dpos, dmass, delta=delta, want_pot=True)
        assert np.all(np.isfinite(acc.cpu().numpy())) and np.all(np.isfinite(pot.cpu().numpy()))
        assert _rel(acc.cpu().numpy(), a_ref) <= TOL[prec]
        assert _rel(pot.cpu().numpy(), p_ref) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_forces_range_eighths_of_2p17_on_the_large_shape(gpu, oracle, prec):
    """What `bench.py --sharded` launches on 8 GPUs at N = 2^17: the eight ranges [k N/8, (k+1) N/8), whose starts are
    not multiples of the 1792 / 1536-body i-block.  Each range must run the large class; 64 sampled bodies per range
    against the oracle, and every row bit-identical to the full solve with the same j-tile size and split."""
    import torch
    from paper_1803_01190_b200 import workloads
    c = workloads.config(1)
    n = c["N"]
    pos, mass = _seen(prec, c["pos"], c["mass"])
    dpos, dmass = _dev(prec, pos, mass)
    rng = np.random.Generator(np.random.Philox(key=5))
    with _Pinned(gpu, "large", 2) as pin:
        full_plan = pin.check(n, prec, True)
        assert sum(1 for k in range(8) if (k * (n // 8)) % full_plan["i_per_cta"]) >= 5   # starts off the block grid
        a_full, p_full = gpu.pp_forces(dpos, dmass, delta=c["delta"], want_pot=True)
        for k in range(8):
            b, cnt = k * (n // 8), n // 8
            a, p = gpu.pp_forces_range(dpos, dmass, b, cnt, delta=c["delta"], want_pot=True)
            assert torch.equal(a, a_full[b:b + cnt]) and torch.equal(p, p_full[b:b + cnt]), "range rows differ bitwise"
            idx = np.sort(rng.choice(cnt, size=64, replace=False)) + b
            a_ref, p_ref = oracle.forces(pos, mass, delta=c["delta"], idx=idx, nthreads=0)
            assert _rel(a[idx - b].cpu().numpy(), a_ref) <= TOL[prec]
            assert _rel(p[idx - b].cpu().numpy(), p_ref) <= TOL[prec]


@pytest.mark.parametrize("shape", ["large", "mid"])
def test_mixed_precision_on_pinned_shapes(gpu, oracle, shape):
    """PP_MIXED (FP64 state, FP32 sweep) on the large and mid classes: forces against the oracle on the FP32-rounded
    inputs, ragged N, species boundaries inside tiles."""
    n = 40003
    pos, _, mass = _cloud(n, 61, "species")
    p32, m32 = _seen("f32", pos, mass)
    a_ref, p_ref = oracle.forces(p32, m32, G=1.5, delta=0.03, nthreads=0)
    dpos, dmass = _dev("f64", pos, mass)
    with _Pinned(gpu, shape) as pin:
        pin.check(n, "f32", True)
        acc, pot = gpu.pp_forces(dpos, dmass, G=1.5, delta=0.03, want_pot=True, mixed=True)
        acc2, _ = gpu.pp_forces(dpos, dmass, G=1.5, delta=0.03, mixed=True)
    assert _rel(acc.cpu().numpy(), a_ref) <= TOL["f32"] and _rel(acc2.cpu().numpy(), a_ref) <= TOL["f32"]
    assert _rel(pot.cpu().numpy(), p_ref) <= TOL["f32"]


@pytest.mark.parametrize("prec", ["f64", "f32", "mixed"])
def test_five_step_trajectory_at_2p15_on_the_large_shape(gpu, oracle, prec):
    """pp_step_kdk against oracle.kdk_halfkick step for step on the kernels the bench times: config 1's recipe (disk +
    halo, two mass species) at N = 2^15, 5 steps, large class pinned.
    Final r, v of ALL bodies within DESIGN.md section 6's trajectory tolerances; a(t_end) and Phi(t_end) too."""
    import torch
    from paper_1803_01190_b200 import workloads
    c = workloads.config(1, N=2 ** 15)
    n, dt, nsteps = c["N"], c["dt"], 5
    seen = "f64" if prec != "f32" else "f32"
    pos, vel, mass = _seen(seen, c["pos"], c["vel"], c["mass"])
    p_ref, v_ref, a_ref, nforce = oracle.kdk_halfkick(pos, vel, mass, dt, nsteps, G=c["G"], delta=c["delta"], nthreads=0)
    assert nforce == nsteps + 1
    _, pot_ref = oracle.forces(p_ref, mass, G=c["G"], delta=c["delta"], nthreads=0)
    dpos, dvel, dmass = _dev(seen, pos, vel, mass)
    dacc = torch.zeros_like(dpos)
    dpot = torch.empty_like(dmass)
    with _Pinned(gpu, "large") as pin:
        pin.check(n, "f32" if prec != "f64" else "f64", True)
        n0 = gpu.pp_launch_count()
        gpu.pp_step_kdk(dpos, dvel, dmass, dacc, dt, nsteps, G=c["G"], delta=c["delta"], pot=dpot,
                        mixed=(prec == "mixed"))
        torch.cuda.synchronize()
        # tile masses + cold start (pack, sweep, finalize) + kick_drift_pack + 2 per interior step + (sweep, finalize)
        assert gpu.pp_launch_count() - n0 == 2 * nsteps + 5
    if prec == "mixed":      # FP64 state, FP32 forces (~1e-7): dr ~ dt^2 |a| 1e-7, dv ~ dt |a| 1e-7 per step
        tol_r, tol_v, tol_a = 1e-9, 1e-7, TOL["f32"]
    else:
        tol_r = tol_v = TOL_TRAJ[prec]
        tol_a = 10 * TOL[prec]
    assert np.abs(dpos.cpu().numpy() - p_ref).max() / np.abs(p_ref).max() <= tol_r
    assert np.abs(dvel.cpu().numpy() - v_ref).max() / np.abs(v_ref).max() <= tol_v
    if prec == "mixed":      # the FP32 sweep sees the FP32-rounded final positions: the oracle is given the same
        p32, m32 = _seen("f32", dpos.cpu().numpy(), mass)
        a_ref, pot_ref = oracle.forces(p32, m32, G=c["G"], delta=c["delta"], nthreads=0)
    assert _rel(dacc.cpu().numpy(), a_ref) <= tol_a
    assert _rel(dpot.cpu().numpy(), pot_ref) <= tol_a


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_invariants_potential_sweep_equal_mass_shortcut(gpu, oracle, prec):
    """pp_invariants(pot=NULL) runs the FP64 potential-only sweep (MODE_POT); on tiles with a common mass it now leaves
    m_j out of the pair loop.  Shortcut on and off both meet the oracle's E, W at 1e-12, on the large and mid classes."""
    n = 20011
    pos, vel, mass = _cloud(n, 77, "species")
    pos, vel, mass = _seen(prec, pos, vel, mass)
    ref = oracle.invariants(pos, vel, mass, G=1.0, delta=0.02, nthreads=0)
    dpos, dvel, dmass = _dev(prec, pos, vel, mass)
    outs = {}
    try:
        for shape in ("large", "mid"):
            for flag in (1, 0):
                gpu.pp_configure(gpu.PP_CFG_EQUAL_MASS, flag)
                with _Pinned(gpu, shape):
                    out = gpu.pp_invariants(dpos, dvel, dmass, G=1.0, delta=0.02).cpu().numpy()
                for k in (0, 1, 2):
                    assert abs(out[k] - ref["raw"][k]) <= 1e-12 * abs(ref["raw"][k]), (shape, flag, k)
                outs[(shape, flag)] = out
    finally:
        gpu.pp_configure(gpu.PP_CFG_EQUAL_MASS, 1)
    # (the double-double tile folding makes W of the two paths agree to the last bits; that the shortcut path exists
    # on these masses is what pp_equal_mass_tiles reports)
    n_tiles, n_common = gpu.pp_equal_mass_tiles(dmass)
    assert n_common >= n_tiles - 4 and abs(outs[("large", 1)][2] - outs[("large", 0)][2]) <= 1e-14 * abs(ref["raw"][2])


def test_default_stream_replays_the_step_graph(gpu):
    """pp_step_kdk on torch's default (legacy) stream: the interior steps are replayed from the cached CUDA graph through
    the library's internal stream, bit-identical to plain launches and with the same launch count; a second call with
    the same buffers reuses the instantiated graph."""
    import torch
    pos, vel, mass = _cloud(1500, 21)
    outs = []
    for graph in (0, 1, 1):
        gpu.pp_configure(gpu.PP_CFG_GRAPH, graph)
        try:
            dpos, dvel, dmass = _dev("f32", pos, vel, mass)
            dacc = torch.zeros_like(dpos)
            assert torch.cuda.current_stream().cuda_stream == 0
            n0 = gpu.pp_launch_count()
            gpu.pp_step_kdk(dpos, dvel, dmass, dacc, 1e-3, 12, delta=0.05)
            gpu.pp_step_kdk(dpos, dvel, dmass, dacc, 1e-3, 3, delta=0.05, acc_valid=True)   # cache hit: 2 interior steps
            torch.cuda.synchronize()
            assert gpu.pp_launch_count() - n0 == (2 * 12 + 5) + (2 * 3 + 2)
            outs.append((dpos.clone(), dvel.clone(), dacc.clone()))
        finally:
            gpu.pp_configure(gpu.PP_CFG_GRAPH, 1)
    for other in outs[1:]:
        for a, b in zip(outs[0], other):
            assert torch.equal(a, b)


def test_two_streams_share_the_workspace_safely(gpu):
    """Calls issued alternately on two streams without host synchronisation: the second stream's call waits on the
    device for the first one's use of the shared workspace, so every result equals the single-stream result bit for bit."""
    import torch
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    clouds = [_cloud(6000 + 37 * k, 300 + k) for k in range(6)]
    devs = [_dev("f32", c[0], c[2]) for c in clouds]
    ref = [gpu.pp_forces(p, m, delta=0.02, want_pot=True) for p, m in devs]
    torch.cuda.synchronize()
    got = []
    for k, (p, m) in enumerate(devs):
        with torch.cuda.stream(sa if k % 2 == 0 else sb):
            got.append(gpu.pp_forces(p, m, delta=0.02, want_pot=True))
    torch.cuda.synchronize()
    for (a, p), (a0, p0) in zip(got, ref):
        assert torch.equal(a, a0) and torch.equal(p, p0)


# ---- the symmetric sweep (every unordered pair once, force_sym_f32.cu) ---------------------------------------------
class _Symmetric:
    """PP_CFG_SYMMETRIC = 2 (always) for the duration of a with-block, optionally with a pinned split-j and a pinned
    j-tile variant (256: what N >= 98304 runs, i.e. the bench; 128: what smaller systems run; 0: by size)."""

    def __init__(self, gpu, split=0, tile=0):
        self.gpu, self.split, self.tile = gpu, split, tile

    def __enter__(self):
        self.gpu.pp_configure(self.gpu.PP_CFG_SYMMETRIC, 2)
        self.gpu.pp_configure(self.gpu.PP_CFG_SPLIT_J, self.split)
        self.gpu.pp_configure(self.gpu.PP_CFG_SHAPE, {0: 0, 256: 1, 128: 2}[self.tile])
        return self

    def __exit__(self, *exc):
        self.gpu.pp_configure(self.gpu.PP_CFG_SYMMETRIC, 1)
        self.gpu.pp_configure(self.gpu.PP_CFG_SPLIT_J, 0)
        self.gpu.pp_configure(self.gpu.PP_CFG_SHAPE, 0)


# one block; two blocks (even: no symmetric partner, the opposite block one-sided); three (odd, H = 1); four (H = 1 and
# the opposite block); five, six, seven, eight, ten blocks; ragged tails just around the block and 256-body tile edges
# (block = 2048 bodies)
SYM_N = [1, 2, 255, 2047, 2049, 4097, 6145, 8193, 10241, 12289, 15000, 18433]


@pytest.mark.parametrize("prec", ["f64", "f32", "mixed"])
@pytest.mark.parametrize("tile", [256, 128])
@pytest.mark.parametrize("n", SYM_N)
def test_symmetric_sweep_edge_sizes(gpu, oracle, prec, tile, n):
    """All bodies against the oracle, split-j {auto, 1, 3}, random masses and mass species, with and without potential."""
    seen = "f64" if prec == "f64" else "f32"
    for masses in ("random", "species"):
        pos, _, mass = _cloud(n, 7000 + n, masses)
        ps, ms = _seen(seen, pos, mass)
        a_ref, p_ref = _oracle_forces(oracle, (n, "sym" + seen, masses), ps, ms, 2.5, 0.05)
        dpos, dmass = _dev("f32" if prec == "f32" else "f64", ps if prec != "mixed" else pos, ms if prec != "mixed" else mass)
        for split in (0, 1, 3):
            with _Symmetric(gpu, split, tile):
                plan = gpu.pp_plan_query(n, gpu.PP_F64 if prec == "f64" else gpu.PP_F32, True)
                assert plan["shape"] == 3 and plan["i_per_cta"] == 2048 and plan["tile_j"] == tile
                acc, pot = gpu.pp_forces(dpos, dmass, G=2.5, delta=0.05, want_pot=True, mixed=(prec == "mixed"))
                acc2, _ = gpu.pp_forces(dpos, dmass, G=2.5, delta=0.05, want_pot=False, mixed=(prec == "mixed"))
            if n == 1:
                assert np.all(acc.cpu().numpy() == 0.0) and np.all(pot.cpu().numpy() == 0.0)
                continue
            assert _rel(acc.cpu().numpy(), a_ref) <= TOL[seen], (masses, split)
            assert _rel(acc2.cpu().numpy(), a_ref) <= TOL[seen], (masses, split)
            assert _rel(pot.cpu().numpy(), p_ref) <= TOL[seen], (masses, split)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("tile", [256, 128])
@pytest.mark.parametrize("masses", ["random", "species"])
def test_symmetric_sweep_delta_zero_and_bitwise_reproducible(gpu, oracle, prec, tile, masses):
    import torch
    n = 9001
    pos, _, mass = _cloud(n, 93, masses)
    pos, mass = _seen(prec, pos, mass)
    a, b = 7, 6000                       # a coincident pair in two different 2048-body blocks: met in a symmetric tile
    pos[b] = pos[a]
    dpos, dmass = _dev(prec, pos, mass)
    with _Symmetric(gpu, 0, tile):
        acc, pot = gpu.pp_forces(dpos, dmass, delta=0.0, want_pot=True)
        acc_b, pot_b = gpu.pp_forces(dpos, dmass, delta=0.0, want_pot=True)
    assert torch.equal(acc, acc_b) and torch.equal(pot, pot_b)
    acc, pot = acc.cpu().numpy(), pot.cpu().numpy()
    assert np.all(np.isfinite(acc)) and np.all(np.isfinite(pot))
    m2, p2 = mass.copy(), pos.copy()
    m2[b] = 0.0
    p2[b] += 1.0
    keep = np.array([i for i in range(n) if i != b])
    a_ref, p_ref = oracle.forces(p2, m2, delta=0.0, idx=keep, nthreads=0)       # everyone but b, with b made massless
    # b is NOT massless for the others: add its pull back for all bodies but its twin a
    others = keep[keep != a]
    d = pos[b] - pos[others]
    r2 = (d * d).sum(axis=1)
    a_ref[keep != a] += mass[b] * d / r2[:, None] ** 1.5
    p_ref[keep != a] -= mass[b] / np.sqrt(r2)
    assert _rel(acc[keep], a_ref) <= TOL[prec] and _rel(pot[keep], p_ref) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32", "mixed"])
@pytest.mark.parametrize("band_rows", [1, 2])
def test_symmetric_sweep_in_bands(gpu, oracle, prec, band_rows):
    """Beyond N = 2^21 the j-side rows no longer fit the workspace at once and the partner offsets are worked through
    in bands (rows reused, folded into running sums in between).  PP_CFG_SYM_BAND_ROWS pins 1 or 2 offsets per band at
    N = 15000 (8 blocks, H = 3: 3 bands of one offset, or 2 bands the second of which is ragged); all bodies against
    the oracle, forced split-j 1 and 3, a 3-step trajectory, and bit-identical run to run."""
    import torch
    n = 15000
    seen = "f64" if prec == "f64" else "f32"
    pos, vel, mass = _cloud(n, 7000 + n, "species")
    ps, vs, ms = _seen(seen, pos, vel, mass)
    a_ref, p_ref = _oracle_forces(oracle, (n, "sym" + seen, "species"), ps, ms, 2.5, 0.05)
    st = "f32" if prec == "f32" else "f64"
    dpos, dvel, dmass = _dev(st, *((ps, vs, ms) if prec != "mixed" else (pos, vel, mass)))
    mixed = prec == "mixed"
    gpu.pp_configure(gpu.PP_CFG_SYM_BAND_ROWS, band_rows)
    try:
        for split in (1, 3):
            with _Symmetric(gpu, split, 256 if split == 1 else 128):
                plan = gpu.pp_plan_query(n, gpu.PP_F64 if prec == "f64" else gpu.PP_F32, True)
                assert plan["shape"] == 3 and plan["sym_bands"] == -(-plan["sym_partner_blocks"] // band_rows) >= 2
                acc, pot = gpu.pp_forces(dpos, dmass, G=2.5, delta=0.05, want_pot=True, mixed=mixed)
                acc2, _ = gpu.pp_forces(dpos, dmass, G=2.5, delta=0.05, mixed=mixed)
                acc3, pot3 = gpu.pp_forces(dpos, dmass, G=2.5, delta=0.05, want_pot=True, mixed=mixed)
            assert torch.equal(acc, acc3) and torch.equal(pot, pot3)
            assert _rel(acc.cpu().numpy(), a_ref) <= TOL[seen] and _rel(acc2.cpu().numpy(), a_ref) <= TOL[seen]
            assert _rel(pot.cpu().numpy(), p_ref) <= TOL[seen]
        if prec != "mixed":
            p3, v3, _, _ = oracle.kdk_halfkick(ps, vs, ms, 1e-3, 3, G=2.5, delta=0.05, nthreads=0)
            dacc = torch.zeros_like(dpos)
            with _Symmetric(gpu):
                gpu.pp_step_kdk(dpos, dvel, dmass, dacc, 1e-3, 3, G=2.5, delta=0.05)
            assert np.abs(dpos.cpu().numpy() - p3).max() / np.abs(p3).max() <= TOL_TRAJ[seen]
            assert np.abs(dvel.cpu().numpy() - v3).max() / np.abs(v3).max() <= TOL_TRAJ[seen]
    finally:
        gpu.pp_configure(gpu.PP_CFG_SYM_BAND_ROWS, 0)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_symmetric_sweep_where_the_plan_picks_it(gpu, oracle, prec):
    """No forcing: at N = 2^17 (config 1, two mass species) the default plan is the symmetric sweep.  4096 sampled
    bodies against the oracle, the whole solve against the one-sided sweep, and a 3-step trajectory of all bodies."""
    import torch
    from paper_1803_01190_b200 import workloads
    c = workloads.config(1)
    n = c["N"]
    code = gpu.PP_F64 if prec == "f64" else gpu.PP_F32
    assert gpu.pp_plan_query(n, code, True)["shape"] == 3
    pos, vel, mass = _seen(prec, c["pos"], c["vel"], c["mass"])
    dpos, dvel, dmass = _dev(prec, pos, vel, mass)
    acc, pot = gpu.pp_forces(dpos, dmass, delta=c["delta"], want_pot=True)
    idx = workloads.sample_indices(c["seed"], n, 4096)
    a_ref, p_ref = oracle.forces(pos, mass, delta=c["delta"], idx=idx, nthreads=0)
    assert _rel(acc[idx].cpu().numpy(), a_ref) <= TOL[prec] and _rel(pot[idx].cpu().numpy(), p_ref) <= TOL[prec]
    gpu.pp_configure(gpu.PP_CFG_SYMMETRIC, 0)
    try:
        assert gpu.pp_plan_query(n, code, True)["shape"] == 0
        acc1, pot1 = gpu.pp_forces(dpos, dmass, delta=c["delta"], want_pot=True)
    finally:
        gpu.pp_configure(gpu.PP_CFG_SYMMETRIC, 1)
    assert not torch.equal(acc, acc1)
    assert _rel(acc.cpu().numpy(), acc1.cpu().numpy().astype(np.float64)) <= {"f64": 1e-13, "f32": 1e-5}[prec]
    assert _rel(pot.cpu().numpy(), pot1.cpu().numpy().astype(np.float64)) <= {"f64": 1e-13, "f32": 1e-5}[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_symmetric_sweep_trajectory_at_2p15(gpu, oracle, prec):
    """5 KDK steps at N = 2^15 (config 1's recipe) on the symmetric sweep against oracle.kdk_halfkick, all bodies."""
    import torch
    from paper_1803_01190_b200 import workloads
    c = workloads.config(1, N=2 ** 15)
    pos, vel, mass = _seen(prec, c["pos"], c["vel"], c["mass"])
    p_ref, v_ref, a_ref, _ = oracle.kdk_halfkick(pos, vel, mass, c["dt"], 5, G=c["G"], delta=c["delta"], nthreads=0)
    dpos, dvel, dmass = _dev(prec, pos, vel, mass)
    dacc = torch.zeros_like(dpos)
    dpot = torch.empty_like(dmass)
    with _Symmetric(gpu, 0, 256):      # the tile variant of the bench kernels (the plan would take 128-body tiles here)
        gpu.pp_step_kdk(dpos, dvel, dmass, dacc, c["dt"], 5, G=c["G"], delta=c["delta"], pot=dpot)
    assert np.abs(dpos.cpu().numpy() - p_ref).max() / np.abs(p_ref).max() <= TOL_TRAJ[prec]
    assert np.abs(dvel.cpu().numpy() - v_ref).max() / np.abs(v_ref).max() <= TOL_TRAJ[prec]
    assert _rel(dacc.cpu().numpy(), a_ref) <= 10 * TOL[prec]
