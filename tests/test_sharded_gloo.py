"""world_size-2 gloo test (CPU) of the i-sharded step's host logic (paper_1803_01190_b200/sharded.py): partition,
all-gather of drifted positions, per-rank i-range solve, reduction of the invariants.  The CUDA kernels cannot run
here, so the test injects stand-in `ops` built on the CPU oracle (tests may use the oracle; the product's default
`CudaOps` calls libppgrav and has no fallback) and checks the two-rank run against the oracle's whole-system
trajectory.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1803_01190_b200 import sharded


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


class OracleOps:
    """Test stand-ins with the interface of sharded.CudaOps, evaluated by the CPU oracle in float64."""

    def __init__(self):
        from oracle import oracle
        oracle.build()
        self.o = oracle

    def forces_range(self, pos_all, mass_all, begin, count, G, delta, want_pot, acc, pot):
        a, p = self.o.forces(pos_all.numpy(), mass_all.numpy(), G=G, delta=delta,
                             idx=np.arange(begin, begin + count), nthreads=1)
        acc.copy_(torch.from_numpy(a))
        if want_pot:
            pot.copy_(torch.from_numpy(p))
        return acc, pot

    def kick_drift(self, pos, vel, acc, kick, dt):
        vel.add_(acc, alpha=kick)
        if dt != 0.0:
            pos.add_(vel, alpha=dt)

    def invariants(self, pos, vel, mass, pot, G, delta):
        d = self.o.invariants(pos.numpy(), vel.numpy(), mass.numpy(), G=G, delta=delta, pot=pot.numpy())
        out = np.zeros(16)
        out[0:3] = d["E"], d["K"], d["W"]
        out[3:6], out[6:9], out[9:12], out[12] = d["P"], d["L"], d["COM"], d["M"]
        return torch.from_numpy(out)


def _system(n=301, seed=3):
    rng = np.random.Generator(np.random.Philox(key=seed))
    pos = rng.standard_normal((n, 3))
    vel = 0.2 * rng.standard_normal((n, 3))
    mass = rng.uniform(0.5, 1.5, size=n) / n
    return pos, vel, mass


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        pos, vel, mass = (torch.from_numpy(a) for a in _system())
        sysm = sharded.ShardedSystem(pos, vel, mass, G=1.3, delta=0.05, comm=sharded.DistComm(), ops=OracleOps())
        inv0 = sysm.invariants()
        sysm.step(2e-3, 3, want_pot=True)
        inv1 = sysm.invariants()
        p, v = sysm.gather_state()
        out[rank] = dict(begin=sysm.begin, count=sysm.count, evals=sysm.force_evaluations, pos=p.numpy(),
                         vel=v.numpy(), E0=inv0["E"], E1=inv1["E"], P1=inv1["P"], L1=inv1["L"], COM1=inv1["COM"],
                         M=inv1["M"])
    finally:
        dist.destroy_process_group()


def test_two_rank_sharded_step_matches_whole_system_oracle(oracle):
    world = 2
    mgr = mp.get_context("spawn").Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    r0, r1 = out[0], out[1]
    assert (r0["begin"], r0["count"], r1["begin"], r1["count"]) == (0, 151, 151, 150)     # uneven split of 301
    assert r0["evals"] == r1["evals"] == 4                                              # a(t0) + one per step
    pos, vel, mass = _system()
    p_ref, v_ref, a_ref, pot_ref = oracle.kdk_halfkick(pos, vel, mass, 2e-3, 3, G=1.3, delta=0.05)
    for r in (r0, r1):                      # both ranks hold the same, correct, whole-system state
        assert np.abs(r["pos"] - p_ref).max() <= 1e-14 * np.abs(p_ref).max()
        assert np.abs(r["vel"] - v_ref).max() <= 1e-14 * np.abs(v_ref).max()
    ref0 = oracle.invariants(pos, vel, mass, G=1.3, delta=0.05)
    ref1 = oracle.invariants(p_ref, v_ref, mass, G=1.3, delta=0.05)
    for r in (r0, r1):
        assert abs(r["E0"] - ref0["E"]) <= 1e-13 * abs(ref0["E"])
        assert abs(r["E1"] - ref1["E"]) <= 1e-13 * abs(ref1["E"])
        assert np.abs(r["P1"] - ref1["P"]).max() <= 1e-15
        assert np.abs(r["L1"] - ref1["L"]).max() <= 1e-14 * np.abs(ref1["L"]).max()
        assert np.abs(r["COM1"] - ref1["COM"]).max() <= 1e-14
        assert abs(r["M"] - mass.sum()) <= 1e-15


def test_partition_covers_range_evenly():
    for n, w in ((10, 3), (301, 2), (8, 8), (2 ** 20, 8), (5, 1)):
        parts = sharded.partition(n, w)
        assert parts[0][0] == 0 and sum(c for _, c in parts) == n
        assert all(parts[i][0] + parts[i][1] == parts[i + 1][0] for i in range(w - 1))
        assert max(c for _, c in parts) - min(c for _, c in parts) <= 1
    with pytest.raises(ValueError):
        pos = torch.zeros((1, 3), dtype=torch.float64)

        class TwoRanks(sharded.SingleComm):
            world = 2
        sharded.ShardedSystem(pos, pos.clone(), torch.ones(1, dtype=torch.float64), comm=TwoRanks(), ops=object())
