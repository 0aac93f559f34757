"""Build libppgrav.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1803_01190_b200.build [--force] [--verbose]

No GPU is needed (nvcc cross-compiles).  The .so is git-ignored but travels to the GPU box with the snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(ROOT, "include")
LIB = os.path.join(HERE, "libppgrav.so")
SOURCES = ("api.cu", "api_host.cu", "plan.cu", "update.cu", "invariants.cu", "density.cu", "force_f32.cu", "force_f64.cu",
           "force_sym_f32.cu", "force_sym_f64.cu")
# measurement tooling, NOT part of libppgrav: the pipe microbenchmarks of probe/ get a library of their own
PROBE_SRC = os.path.join(HERE, "probe", "pipe_probe.cu")
PROBE_LIB = os.path.join(HERE, "probe", "libppprobe.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
              "--ftz=false", "--prec-div=true", "--prec-sqrt=true", "--fmad=true"]


def _nvcc():
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(INCLUDE, "ppgrav.h"), __file__]
    if any(os.path.getmtime(d) > t for d in deps):
        return True
    return not os.path.exists(PROBE_LIB) or os.path.getmtime(PROBE_SRC) > os.path.getmtime(PROBE_LIB)


def build(force=False, verbose=False, extra_flags=(), out=None):
    """Compile every translation unit and link paper_1803_01190_b200/libppgrav.so.  Returns its path.
    extra_flags / out: tuning builds with -DPP_F32_IPT=... shape overrides into another file."""
    if out is None and not force and not _stale():
        return LIB
    objdir = os.path.join(HERE, "build") if out is None else out + ".objs"
    out = LIB if out is None else out
    os.makedirs(objdir, exist_ok=True)
    flags = list(NVCC_FLAGS) + list(extra_flags) + (["-Xptxas", "-v"] if verbose else [])
    procs = []
    for src in SOURCES:
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        cmd = [_nvcc()] + flags + ["-I", INCLUDE, "-I", CSRC, "-c", os.path.join(CSRC, src), "-o", obj]
        procs.append((src, obj, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    objs = []
    for src, obj, p in procs:
        log, _ = p.communicate()
        if verbose or p.returncode != 0:
            sys.stderr.write(log)
        if p.returncode != 0:
            raise RuntimeError("nvcc failed on %s" % src)
        objs.append(obj)
    cmd = [_nvcc(), "-shared", "-o", out] + objs + ["-gencode", "arch=compute_100a,code=sm_100a", "-lcudart"]
    subprocess.run(cmd, check=True)
    if out == LIB:
        subprocess.run([_nvcc()] + list(NVCC_FLAGS) + ["-shared", "-o", PROBE_LIB, PROBE_SRC, "-lcudart"], check=True)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
