"""The conservation experiment (paper_1803_01190_b200/conservation.py; protocol of Table 2) at a
size the oracle can follow: its invariants series must agree with the oracle's on the oracle's own trajectory, and
leapfrog must conserve P and L_z to round-off in FP64 (pin P8)."""
import numpy as np
import pytest

from paper_1803_01190_b200 import workloads

pytestmark = pytest.mark.gpu


def test_conservation_series_against_oracle(oracle):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("a -m gpu test was started without a CUDA device")
    from paper_1803_01190_b200 import conservation
    logn, steps, dt, every = 10, 40, 5e-4, 20
    runs = {p: conservation.run(logn, steps, dt, every, p, verbose=False) for p in ("f32", "mixed", "f64")}
    c = workloads.config(2, N=1 << logn)
    pos, vel, mass = c["pos"], c["vel"], c["mass"]
    E_ref = [oracle.invariants(pos, vel, mass, G=c["G"], delta=c["delta"], nthreads=0)["E"]]
    acc = None
    for _ in range(steps // every):
        pos, vel, acc, _ = oracle.kdk_halfkick(pos, vel, mass, dt, every, G=c["G"], delta=c["delta"], acc=acc,
                                               nthreads=0)
        E_ref.append(oracle.invariants(pos, vel, mass, G=c["G"], delta=c["delta"], nthreads=0)["E"])
    E_ref = np.array(E_ref)
    for p, tol in (("f64", 1e-12), ("mixed", 1e-7), ("f32", 1e-6)):
        r = runs[p]
        assert r["times"] == [0.0, every * dt, 2 * every * dt] and len(r["E"]) == 3
        assert np.abs(np.array(r["E"]) - E_ref).max() <= tol * abs(E_ref[0]), p
    d = runs["f64"]["drift"]
    assert d["dP_abs_max"] <= 1e-16 and d["dLz_over_Lz0_max"] <= 1e-14
    assert runs["mixed"]["drift"]["dP_abs_max"] <= 1e-8 and runs["f32"]["drift"]["dP_abs_max"] <= 1e-6


def test_checkpointed_run_continues_bit_for_bit(tmp_path):
    from paper_1803_01190_b200 import conservation
    whole = conservation.run(10, 40, 5e-4, 10, "f32", verbose=False)
    ck = str(tmp_path / "state.npz")
    first = conservation.run(10, 40, 5e-4, 10, "f32", verbose=False, checkpoint=ck, stop_after=20)
    assert first["steps"] == 20 and len(first["E"]) == 3
    second = conservation.run(10, 40, 5e-4, 10, "f32", verbose=False, checkpoint=ck)
    assert second["steps"] == 40 and second["times"] == whole["times"]
    assert second["E"] == whole["E"] and second["P"] == whole["P"] and second["Lz"] == whole["Lz"]


def test_checkpoint_path_without_suffix_and_mismatch(tmp_path):
    """a --checkpoint path without the .npz suffix used to restart from t = 0 on resume (np.savez appends the
    suffix, the resume check looked for the bare name); a checkpoint of another run is now a clear error."""
    import os
    from paper_1803_01190_b200 import conservation
    whole = conservation.run(10, 20, 5e-4, 10, "f64", verbose=False)
    ck = str(tmp_path / "state")                         # no suffix
    first = conservation.run(10, 20, 5e-4, 10, "f64", verbose=False, checkpoint=ck, stop_after=10)
    assert first["steps"] == 10 and os.path.exists(ck + ".npz") and not os.path.exists(ck + ".tmp.npz")
    second = conservation.run(10, 20, 5e-4, 10, "f64", verbose=False, checkpoint=ck)
    assert second["steps"] == 20 and second["E"] == whole["E"] and second["times"] == whole["times"]
    with pytest.raises(ValueError, match="one checkpoint file per run"):
        conservation.run(10, 20, 5e-4, 10, "f32", verbose=False, checkpoint=ck)
