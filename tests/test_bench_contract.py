"""CPU checks of the bench.py contract the driver depends on: the reference arm prints ONE JSON line with the agreed
keys (it times the oracle on the host cores, no GPU), and the binding's configuration constants are the header's."""
import json
import os
import re
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    run = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "1", "--steps", "2",
                          "--warmup", "1", "--n", "8192"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert run.returncode == 0, run.stderr
    lines = [l for l in run.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "pair-interactions/s" and d["unit"] == "pair-interactions/s"
    assert d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] == 1 and d["higher_is_better"] is True
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["vs_baseline"] is None and d["data"] == "synthetic"
    assert d["dtype"] == "f64" and "workload" in d["config"] and "model" not in d["config"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and cb["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    # 4096 sampled i-bodies x (N - 1) j-bodies per step
    assert abs(d["value"] * d["ms_per_step"] * 1e-3 - 4096 * 8191) <= 1e-6 * 4096 * 8191


def test_other_ranks_of_the_reference_arm_do_no_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    run = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, timeout=120, cwd=ROOT, env=env)
    assert run.returncode == 0 and run.stdout.strip() == ""


def test_binding_constants_are_the_headers():
    from paper_1803_01190_b200 import ppgrav
    hdr = open(os.path.join(ROOT, "include", "ppgrav.h")).read()
    defs = dict(re.findall(r"#define\s+(PP[A-Z0-9_]+)\s+\(?(-?\d+)u?\)?", hdr))
    for name in ("PP_F32", "PP_F64", "PP_MIXED", "PP_ACC_VALID", "PP_CFG_SPLIT_J", "PP_CFG_GRAPH", "PP_CFG_PROFILE",
                 "PP_CFG_EQUAL_MASS", "PP_CFG_SHAPE", "PP_CFG_SYMMETRIC", "PP_CFG_SYM_BAND_ROWS"):
        assert int(defs[name]) == getattr(ppgrav, name), name
    assert "#define PP_NOALLOC_MAX_N (1ll << 28)" in hdr and ppgrav.PP_NOALLOC_MAX_N == 1 << 28
    assert int(defs["PPGRAV_VERSION"]) == 200
