"""libppgrav: B200-native (sm_100a) direct particle-particle gravity, FP32 and FP64, with KDK leapfrog and
conservation diagnostics -- the hot path of Khrapov, Khoperskov & Khoperskov (2018), eqs. (1)-(2), (5)-(10).

`paper_1803_01190_b200.ppgrav` is the thin binding over the C-ABI library (include/ppgrav.h);
`paper_1803_01190_b200.workloads` holds the seeded input generators.  Importing the package does not load
the CUDA library; the first call through `ppgrav` does, and fails loudly if it is missing.
"""
__all__ = ["ppgrav", "workloads", "build"]
