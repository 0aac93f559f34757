"""CPU-side checks of the product: the C-ABI library loads and exports every symbol include/ppgrav.h declares, the
launch plan (pure host logic) is sane, and compute calls fail loudly without a CUDA device (no fallback)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def ppgrav():
    from paper_1803_01190_b200 import build, ppgrav
    build.build()
    return ppgrav


def test_header_symbols_are_exported_and_bound(ppgrav):
    hdr = open(os.path.join(ROOT, "include", "ppgrav.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pp_[a-z0-9_]+)\s*\(", hdr))
    assert len(declared) >= 14
    lib = ppgrav.lib()
    for name in declared:
        assert hasattr(lib, name), name
    assert declared == set(ppgrav.SIGNATURES), declared ^ set(ppgrav.SIGNATURES)
    assert lib.pp_version() == 100


def test_no_oracle_import_in_product():
    """The product path must not touch oracle/ (it is test infrastructure)."""
    pkg = os.path.join(ROOT, "paper_1803_01190_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "pp_oracle" not in text, f


@pytest.mark.parametrize("prec", [0, 1])
def test_plan_is_sane(ppgrav, prec):
    for n in (1, 2, 100, 2048, 2 ** 14, 2 ** 17, 2 ** 20, 2 ** 22, 2 ** 23):
        p = ppgrav.pp_plan_query(n, prec)
        assert p["i_per_cta"] in (128, 1536, 1792) and p["tile_j"] in (128, 256, 512)
        n_ib = -(-n // p["i_per_cta"])
        n_tiles = -(-n // p["tile_j"])
        assert 1 <= p["split"] <= max(1, n_tiles)
        assert p["ctas"] == n_ib * p["split"]
        elem = 32 if prec else 16
        n_pad = -(-n // p["i_per_cta"]) * p["i_per_cta"]
        assert p["split"] * n_pad * elem <= (1 << 30) or p["split"] == 1
        assert p["pipe_ops_per_pair"] == (16 if prec else 12)
    # calibrated choices: the throughput shape from N = 2^16 up, the small one below 2^14
    for n in (2 ** 16, 2 ** 17, 2 ** 20, 2 ** 23):
        assert ppgrav.pp_plan_query(n, prec)["i_per_cta"] >= 1536
    for n in (100, 2048, 2 ** 13):
        assert ppgrav.pp_plan_query(n, prec)["i_per_cta"] == 128
    big = ppgrav.pp_plan_query(2 ** 20, prec)
    resident = big["sm_count"] * big["ctas_per_sm"]
    waves = big["ctas"] / resident
    assert waves / -(-big["ctas"] // resident) > 0.95, "last wave of the N=2^20 plan should be nearly full"
    assert ppgrav.pp_plan_query(2 ** 20, prec, True)["pipe_ops_per_pair"] == (18 if prec else 13)


def test_forced_split_is_honoured(ppgrav):
    ppgrav.pp_configure(ppgrav.PP_CFG_SPLIT_J, 5)
    try:
        assert ppgrav.pp_plan_query(2 ** 17, 0)["split"] == 5
        assert ppgrav.pp_plan_query(100, 0)["split"] == 1       # capped by the number of j-tiles
    finally:
        ppgrav.pp_configure(ppgrav.PP_CFG_SPLIT_J, 0)


def test_bad_arguments_and_no_device(ppgrav):
    import ctypes
    import torch
    lib = ppgrav.lib()
    out = (ctypes.c_int64 * 8)()
    assert lib.pp_plan_query(0, 0, 0, out) == -1
    assert lib.pp_plan_query(10, 2, 0, out) == 0          # PP_MIXED plans like PP_F32
    assert lib.pp_plan_query(10, 3, 0, out) == -1
    assert b"precision" in lib.pp_last_error()
    with pytest.raises(ppgrav.PPGravError):
        ppgrav.pp_configure(99, 0)
    if not torch.cuda.is_available():
        # no CPU fallback: a compute call without a device reports PP_ECUDA
        buf = (ctypes.c_double * 64)()
        p = ctypes.addressof(buf)
        assert lib.pp_forces(p, p, p, None, 4, 1.0, 0.1, 1, None) == -2
        assert b"CUDA" in lib.pp_last_error()
        assert lib.pp_forces_host(p, p, p, None, 4, 1.0, 0.1, 1, None) in (-2, -3)
