"""MEASUREMENT TOOLING, not part of the product path: ctypes front-end of libppprobe.so (probe/pipe_probe.cu), the
pipe-throughput microbenchmarks behind the ALU roofline denominators.

    python -m paper_1803_01190_b200.probe.pipe_probe          # prints every probe (what profiles/r1_pipe_probes.md lists)
"""
import ctypes
import os

KINDS = {"ffma": 0, "ffma2": 1, "dfma": 2, "mufu_rsq": 3, "mufu_rsq64h": 4, "force_mix_f32": 5,
         "ffma2_dfma_const": 6, "ffma2_3reg": 7, "ffma2_dfma_3reg": 8}
LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libppprobe.so")
_lib = None


def pp_probe_pipe(kind, iters=1 << 14):
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libppprobe.so not found -- run `python -m paper_1803_01190_b200.build`")
        _lib = ctypes.CDLL(LIB_PATH)
        _lib.pp_probe_pipe.restype = ctypes.c_int
        _lib.pp_probe_pipe.argtypes = [ctypes.c_int, ctypes.c_int64, ctypes.c_void_p]
    k = KINDS[kind] if isinstance(kind, str) else int(kind)
    out = (ctypes.c_double * 4)()
    rc = _lib.pp_probe_pipe(k, int(iters), out)
    if rc != 0:
        raise RuntimeError("pp_probe_pipe failed (%d)" % rc)
    return dict(seconds=out[0], lane_ops=out[1], sm_mhz=out[2], lane_ops_per_clk_per_sm=out[3])


if __name__ == "__main__":
    for name in KINDS:
        print(name, pp_probe_pipe(name, 1 << 16))
