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
    assert lib.pp_version() == 200


def test_no_oracle_import_in_product():
    """The product path must not touch oracle/ (it is test infrastructure)."""
    pkg = os.path.join(ROOT, "paper_1803_01190_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")) and "__pycache__" not in dirpath:
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "pp_oracle" not in text, f


SHAPES = {0: {"large": (1792, 512), "mid": (512, 256), "small": (128, 128)},
          1: {"large": (1536, 256), "mid": (512, 128), "small": (128, 128)}}     # (i-bodies per CTA, tile_j) with Phi


@pytest.mark.parametrize("prec", [0, 1])
def test_plan_is_sane(ppgrav, prec):
    allowed_i = {v[0] for v in SHAPES[prec].values()} | {1792, 2048}   # FP64 force-only: 7 per thread; symmetric: 8
    allowed_t = {v[1] for v in SHAPES[prec].values()} | {256}                          # symmetric sweeps: 256
    for n in (1, 2, 100, 2048, 2 ** 14, 2 ** 17, 2 ** 20, 2 ** 22, 2 ** 23):
        for with_pot in (False, True):
            p = ppgrav.pp_plan_query(n, prec, with_pot)
            assert p["i_per_cta"] in allowed_i and p["tile_j"] in allowed_t
            assert p["i_per_cta"] == p["threads"] * p["ipt"]
            n_ib = -(-n // p["i_per_cta"])
            n_tiles = -(-n // p["tile_j"])
            assert p["i_blocks"] == n_ib
            assert 1 <= p["split"] <= max(1, n_tiles)
            assert p["ctas"] == n_ib * p["split"]
            elem = 32 if prec else 16
            assert p["split"] * n_ib * p["i_per_cta"] * elem <= (1 << 30) or p["split"] == 1
            if p["shape"] == 3:                    # symmetric sweep: one evaluation serves two ordered pairs
                assert (p["i_per_cta"], p["tile_j"]) == (2048, 128 if n < 98304 else 256)
                assert p["pairs_per_evaluation"] == 2 and p["sym_partner_blocks"] == (n_ib - 1) // 2
                assert p["pipe_ops_per_pair"] == ((11.5 if with_pot else 10) if prec else (9 if with_pot else 8))
            else:
                assert p["pipe_ops_per_pair"] == ((18 if with_pot else 16) if prec else (13 if with_pot else 12))
    # calibrated choices: one body per thread for small systems, the symmetric sweep from
    # 2^14; with it switched off the mid class at 2^14 (FP32) and the large one-sided class from 2^15
    for n in (2 ** 17, 2 ** 20, 2 ** 23):
        p = ppgrav.pp_plan_query(n, prec)
        # full solves take the symmetric sweep; beyond 2^21 its j-side rows (> 48 GB) are worked through in bands
        assert p["shape"] == 3 and p["i_per_cta"] >= 1536 and (p["sym_bands"] == 1) == (n <= 2 ** 21)
        elem = 32 if prec else 16
        rows = -(-p["sym_partner_blocks"] // p["sym_bands"])
        assert rows * p["i_blocks"] * p["i_per_cta"] * elem <= (16 if p["sym_bands"] > 1 else 48) << 30
    for n in (100, 1024, 2 ** 13):
        assert ppgrav.pp_plan_query(n, prec)["shape"] == 2
    for n in (2 ** 14, 2 ** 15, 2 ** 17):
        assert ppgrav.pp_plan_query(n, prec)["shape"] == 3
    ppgrav.pp_configure(ppgrav.PP_CFG_SYMMETRIC, 0)
    try:
        assert ppgrav.pp_plan_query(2 ** 14, prec)["shape"] == (2 if prec else 1)
        assert ppgrav.pp_plan_query(2 ** 15, prec)["shape"] == 0 and ppgrav.pp_plan_query(2 ** 16, prec)["shape"] == 0
    finally:
        ppgrav.pp_configure(ppgrav.PP_CFG_SYMMETRIC, 1)
    # FP64 per-mode shapes of the large class share the tile size (so they share tile masses and padding rules)
    ppgrav.pp_configure(ppgrav.PP_CFG_SYMMETRIC, 0)
    try:
        big = ppgrav.pp_plan_query(2 ** 20, prec, True)
        assert big["shape"] == 0
        if prec:
            f, fp = ppgrav.pp_plan_query(2 ** 20, 1, False), big
            assert (f["ipt"], fp["ipt"]) == (7, 6) and f["tile_j"] == fp["tile_j"]
    finally:
        ppgrav.pp_configure(ppgrav.PP_CFG_SYMMETRIC, 1)
    resident = big["sm_count"] * big["ctas_per_sm"]
    waves = big["ctas"] / resident
    assert waves / -(-big["ctas"] // resident) > 0.95, "last wave of the N=2^20 plan should be nearly full"


@pytest.mark.parametrize("prec", [0, 1])
def test_forced_shape_is_honoured(ppgrav, prec):
    try:
        for key, name in ((ppgrav.SHAPE_LARGE, "large"), (ppgrav.SHAPE_MID, "mid"), (ppgrav.SHAPE_SMALL, "small")):
            ppgrav.pp_configure(ppgrav.PP_CFG_SHAPE, key)
            for n in (3, 3000, 2 ** 20):
                p = ppgrav.pp_plan_query(n, prec, True)
                assert (p["i_per_cta"], p["tile_j"]) == SHAPES[prec][name] and p["shape"] == key - 1
        with pytest.raises(ppgrav.PPGravError):
            ppgrav.pp_configure(ppgrav.PP_CFG_SHAPE, 4)
    finally:
        ppgrav.pp_configure(ppgrav.PP_CFG_SHAPE, 0)


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
    out = (ctypes.c_int64 * 16)()
    assert lib.pp_plan_query(0, 0, 0, out) == -1
    assert lib.pp_plan_query(2 ** 28 + 1, 0, 0, out) == -1          # beyond the maximum size (2^28 bodies)
    assert b"2^28" in lib.pp_last_error()
    assert lib.pp_plan_query(2 ** 28, 1, 1, out) == 0 and out[0] * out[11] >= 2 ** 28     # the maximum size plans
    # ... and its workspace fits the GPU: the banded symmetric sweep reuses its rows AND its partial sums, so the
    # demand does not grow with the number of bands (round 2 first kept one set of partials per band: 137 GB at 2^25)
    for n, cap in ((2 ** 20, 12), (2 ** 21, 40), (2 ** 23, 20), (2 ** 25, 24), (2 ** 28, 64)):
        for prec in (0, 1):
            q = ppgrav.pp_plan_query(n, prec, True)
            assert q["shape"] == 3 and q["workspace_bytes"] <= cap << 30, (n, prec, q["workspace_bytes"] / 2 ** 30)
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
