"""Thin ctypes binding over the C ABI of libppgrav (include/ppgrav.h) -- argument marshalling only.

Every step of the path (packing, pair sweep, split-j reduction, kick/drift, invariants) runs in the library's CUDA
kernels; PyTorch is used for device buffers and streams.  Function names mirror the C entry points:

    pp_forces      eq. (1)-(2), PAPER.md:41-48     pp_step_kdk   eqs. (5)-(7)
    pp_invariants  eqs. (8)-(10)

There is no CPU fallback: if libppgrav.so is missing the first call raises (build it with
`python -m paper_1803_01190_b200.build`), and without a CUDA device every compute call raises PPGravError.
This module never imports oracle/.
"""
import ctypes
import os

import numpy as np

PP_F32, PP_F64, PP_MIXED = 0, 1, 2
PP_ACC_VALID = 1
PP_CFG_SPLIT_J, PP_CFG_GRAPH, PP_CFG_PROFILE, PP_CFG_EQUAL_MASS, PP_CFG_SHAPE, PP_CFG_SYMMETRIC = 1, 2, 3, 4, 5, 6
PP_CFG_SYM_BAND_ROWS = 7
SHAPE_AUTO, SHAPE_LARGE, SHAPE_MID, SHAPE_SMALL = 0, 1, 2, 3
INVARIANT_NAMES = ("E", "K", "W", "Px", "Py", "Pz", "Lx", "Ly", "Lz", "Cx", "Cy", "Cz", "M")

LIB_PATH = os.environ.get("PPGRAV_LIB") or os.path.join(os.path.dirname(os.path.abspath(__file__)), "libppgrav.so")

# every symbol include/ppgrav.h declares: (restype, argtypes)
_i64, _dbl, _int, _vp, _u = ctypes.c_int64, ctypes.c_double, ctypes.c_int, ctypes.c_void_p, ctypes.c_uint
SIGNATURES = {
    "pp_version": (_int, []),
    "pp_last_error": (ctypes.c_char_p, []),
    "pp_release": (_int, [_int]),
    "pp_configure": (_int, [_int, _i64]),
    "pp_launch_count": (_i64, []),
    "pp_forces": (_int, [_vp, _vp, _vp, _vp, _i64, _dbl, _dbl, _int, _vp]),
    "pp_forces_range": (_int, [_vp, _vp, _vp, _vp, _i64, _i64, _i64, _dbl, _dbl, _int, _vp]),
    "pp_kick_drift": (_int, [_vp, _vp, _vp, _i64, _dbl, _dbl, _int, _vp]),
    "pp_step_kdk": (_int, [_vp, _vp, _vp, _vp, _vp, _i64, _dbl, _i64, _dbl, _dbl, _int, _u, _vp]),
    "pp_invariants": (_int, [_vp, _vp, _vp, _vp, _i64, _dbl, _dbl, _int, _vp, _vp]),
    "pp_invariants_noalloc": (_int, [_vp, _vp, _vp, _vp, _i64, _int, _vp, _vp]),
    "pp_surface_density": (_int, [_vp, _vp, _i64, _dbl, _dbl, _dbl, _int, _int, _int, _vp, _vp]),
    "pp_forces_host": (_int, [_vp, _vp, _vp, _vp, _i64, _dbl, _dbl, _int, _vp]),
    "pp_step_kdk_host": (_int, [_vp, _vp, _vp, _vp, _vp, _i64, _dbl, _i64, _dbl, _dbl, _int, _u, _vp]),
    "pp_invariants_host": (_int, [_vp, _vp, _vp, _vp, _i64, _dbl, _dbl, _int, _vp, _vp]),
    "pp_plan_query": (_int, [_i64, _int, _int, _vp]),
    "pp_equal_mass_tiles": (_int, [_vp, _i64, _int, _vp, _vp]),
    "pp_profile_read": (_int, [_vp]),
}


class PPGravError(RuntimeError):
    pass


_lib = None


def lib():
    """The loaded C library (loads it on first use; raises if it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise PPGravError("libppgrav.so not found at %s -- run `python -m paper_1803_01190_b200.build`; "
                              "there is no CPU fallback" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _check(rc, what):
    if rc != 0:
        raise PPGravError("%s failed (%d): %s" % (what, rc, lib().pp_last_error().decode()))


def _torch():
    import torch
    return torch


def _precision_of(t, mixed=False):
    """PP_F32 / PP_F64 from the dtype; mixed=True (float64 arrays only) selects PP_MIXED: FP64 state, FP32 sweep."""
    torch = _torch()
    if mixed:
        if t.dtype != torch.float64:
            raise TypeError("mixed=True needs float64 state arrays, got %s" % t.dtype)
        return PP_MIXED
    if t.dtype == torch.float32:
        return PP_F32
    if t.dtype == torch.float64:
        return PP_F64
    raise TypeError("state arrays must be float32 or float64, got %s" % t.dtype)


def _dev(t, shape, dtype, name):
    if not t.is_cuda or not t.is_contiguous() or t.dtype != dtype or tuple(t.shape) != tuple(shape):
        raise ValueError("%s must be a contiguous CUDA tensor of shape %s and dtype %s" % (name, tuple(shape), dtype))
    return t.data_ptr()


def _stream(stream):
    torch = _torch()
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def pp_version():
    return lib().pp_version()


def pp_launch_count():
    return int(lib().pp_launch_count())


def pp_configure(key, value):
    _check(lib().pp_configure(int(key), int(value)), "pp_configure")


def pp_release(device=-1):
    _check(lib().pp_release(int(device)), "pp_release")


def pp_plan_query(N, precision, with_pot=False):
    out = (ctypes.c_int64 * 16)()
    _check(lib().pp_plan_query(int(N), int(precision), int(bool(with_pot)), out), "pp_plan_query")
    keys = ("i_per_cta", "tile_j", "split", "ctas", "ctas_per_sm", "sm_count", "pipe_ops_per_evaluation",
            "mufu_per_evaluation", "shape", "threads", "ipt", "i_blocks", "pairs_per_evaluation", "sym_partner_blocks",
            "sym_bands", "workspace_bytes")
    d = dict(zip(keys, (int(v) for v in out)))
    # per ordered pair (pair interaction): what the roofline counts; one less on equal-mass tiles
    d["pipe_ops_per_pair"] = d["pipe_ops_per_evaluation"] / d["pairs_per_evaluation"]
    return d


def pp_equal_mass_tiles(mass, stream=None, mixed=False):
    """(j-tiles swept, j-tiles whose bodies have a common mass) for a gravity solve of these masses."""
    prec = _precision_of(mass, mixed)
    N = mass.shape[0]
    out = (ctypes.c_int64 * 2)()
    _check(lib().pp_equal_mass_tiles(_dev(mass, (N,), mass.dtype, "mass"), N, prec, out, _stream(stream)),
           "pp_equal_mass_tiles")
    return int(out[0]), int(out[1])


def pp_profile_read():
    """(summed milliseconds, number) of the pair-sweep launches recorded since the last read (PP_CFG_PROFILE)."""
    out = (ctypes.c_double * 2)()
    _check(lib().pp_profile_read(out), "pp_profile_read")
    return float(out[0]), int(out[1])


def pp_forces(pos, mass, G=1.0, delta=0.0, want_pot=False, acc=None, pot=None, stream=None, mixed=False):
    """Accelerations (and potentials) of all bodies.  pos [N,3], mass [N]: CUDA tensors of one dtype.
    Returns (acc [N,3], pot [N] or None); pass acc/pot to reuse buffers."""
    torch = _torch()
    prec = _precision_of(pos, mixed)
    N = pos.shape[0]
    p_pos = _dev(pos, (N, 3), pos.dtype, "pos")
    p_mass = _dev(mass, (N,), pos.dtype, "mass")
    if acc is None:
        acc = torch.empty((N, 3), dtype=pos.dtype, device=pos.device)
    if pot is None and want_pot:
        pot = torch.empty((N,), dtype=pos.dtype, device=pos.device)
    p_acc = _dev(acc, (N, 3), pos.dtype, "acc")
    p_pot = _dev(pot, (N,), pos.dtype, "pot") if pot is not None else None
    with torch.cuda.device(pos.device):
        _check(lib().pp_forces(p_pos, p_mass, p_acc, p_pot, N, float(G), float(delta), prec, _stream(stream)),
               "pp_forces")
    return acc, pot


def pp_forces_range(pos, mass, i_begin, i_count, G=1.0, delta=0.0, want_pot=False, acc=None, pot=None, stream=None,
                    mixed=False):
    """Accelerations (and potentials) of bodies [i_begin, i_begin + i_count) against all N bodies.
    Returns (acc [i_count,3], pot [i_count] or None)."""
    torch = _torch()
    prec = _precision_of(pos, mixed)
    N = pos.shape[0]
    n = int(i_count)
    p_pos = _dev(pos, (N, 3), pos.dtype, "pos")
    p_mass = _dev(mass, (N,), pos.dtype, "mass")
    if acc is None:
        acc = torch.empty((n, 3), dtype=pos.dtype, device=pos.device)
    if pot is None and want_pot:
        pot = torch.empty((n,), dtype=pos.dtype, device=pos.device)
    p_acc = _dev(acc, (n, 3), pos.dtype, "acc")
    p_pot = _dev(pot, (n,), pos.dtype, "pot") if pot is not None else None
    with torch.cuda.device(pos.device):
        _check(lib().pp_forces_range(p_pos, p_mass, p_acc, p_pot, N, int(i_begin), n, float(G), float(delta), prec,
                                     _stream(stream)), "pp_forces_range")
    return acc, pot


def pp_kick_drift(pos, vel, acc, kick, dt, stream=None):
    """vel += kick * acc; pos += dt * vel (skipped when dt == 0), in place on CUDA tensors [n,3]."""
    torch = _torch()
    prec = _precision_of(pos)
    n = pos.shape[0]
    with torch.cuda.device(pos.device):
        _check(lib().pp_kick_drift(_dev(pos, (n, 3), pos.dtype, "pos"), _dev(vel, (n, 3), pos.dtype, "vel"),
                                   _dev(acc, (n, 3), pos.dtype, "acc"), n, float(kick), float(dt), prec,
                                   _stream(stream)), "pp_kick_drift")


def pp_step_kdk(pos, vel, mass, acc, dt, nsteps, G=1.0, delta=0.0, acc_valid=False, pot=None, stream=None,
                mixed=False):
    """nsteps KDK steps in place on CUDA tensors pos, vel [N,3], mass [N], acc [N,3]; pot [N] (optional) receives
    the potential of the final state (see include/ppgrav.h)."""
    torch = _torch()
    prec = _precision_of(pos, mixed)
    N = pos.shape[0]
    ptrs = [_dev(pos, (N, 3), pos.dtype, "pos"), _dev(vel, (N, 3), pos.dtype, "vel"),
            _dev(mass, (N,), pos.dtype, "mass"), _dev(acc, (N, 3), pos.dtype, "acc"),
            _dev(pot, (N,), pos.dtype, "pot") if pot is not None else None]
    with torch.cuda.device(pos.device):
        _check(lib().pp_step_kdk(ptrs[0], ptrs[1], ptrs[2], ptrs[3], ptrs[4], N, float(dt), int(nsteps), float(G),
                                 float(delta), prec, PP_ACC_VALID if acc_valid else 0, _stream(stream)),
               "pp_step_kdk")


def pp_invariants(pos, vel, mass, G=1.0, delta=0.0, pot=None, out16=None, stream=None):
    """out16 (CUDA float64 tensor of 16): E, K, W, P, L, COM, M.  pot=None runs the O(N^2) FP64 potential pass."""
    torch = _torch()
    prec = _precision_of(pos)
    N = pos.shape[0]
    if out16 is None:
        out16 = torch.empty(16, dtype=torch.float64, device=pos.device)
    p_pot = _dev(pot, (N,), pos.dtype, "pot") if pot is not None else None
    with torch.cuda.device(pos.device):
        _check(lib().pp_invariants(_dev(pos, (N, 3), pos.dtype, "pos"), _dev(vel, (N, 3), pos.dtype, "vel"),
                                   _dev(mass, (N,), pos.dtype, "mass"), p_pot, N, float(G), float(delta), prec,
                                   _dev(out16, (16,), torch.float64, "out16"), _stream(stream)), "pp_invariants")
    return out16


PP_NOALLOC_MAX_N = 1 << 28


def pp_invariants_noalloc(pos, vel, mass, pot, out16, stream=None):
    """pp_invariants without any allocation inside the library (its scratch is a static device array of 75,776 bytes;
    include/ppgrav.h): pot [N] is required, out16 (CUDA float64 tensor of 16) is supplied by the caller, N at most
    PP_NOALLOC_MAX_N.  Calls that overlap on the GPU race on the shared scratch."""
    torch = _torch()
    prec = _precision_of(pos)
    N = pos.shape[0]
    with torch.cuda.device(pos.device):
        _check(lib().pp_invariants_noalloc(_dev(pos, (N, 3), pos.dtype, "pos"), _dev(vel, (N, 3), pos.dtype, "vel"),
                                           _dev(mass, (N,), pos.dtype, "mass"), _dev(pot, (N,), pos.dtype, "pot"), N,
                                           prec, _dev(out16, (16,), torch.float64, "out16"), _stream(stream)),
               "pp_invariants_noalloc")
    return out16


def pp_surface_density(pos, mass, x0, y0, cell, nx, ny, sigma=None, stream=None):
    """Surface-density map sigma [ny, nx] (CUDA float64) of the bodies, Fig. 7."""
    torch = _torch()
    prec = _precision_of(pos)
    N = pos.shape[0]
    if sigma is None:
        sigma = torch.empty((int(ny), int(nx)), dtype=torch.float64, device=pos.device)
    with torch.cuda.device(pos.device):
        _check(lib().pp_surface_density(_dev(pos, (N, 3), pos.dtype, "pos"), _dev(mass, (N,), pos.dtype, "mass"), N,
                                        float(x0), float(y0), float(cell), int(nx), int(ny), prec,
                                        _dev(sigma, (ny, nx), torch.float64, "sigma"), _stream(stream)),
               "pp_surface_density")
    return sigma


def invariants_dict(out16):
    """Host-side view of an out16 tensor/array as a dict (synchronises if it is a CUDA tensor)."""
    a = out16.detach().cpu().numpy() if hasattr(out16, "detach") else np.asarray(out16)
    d = {k: float(a[i]) for i, k in enumerate(INVARIANT_NAMES)}
    d["P"], d["L"], d["COM"] = a[3:6].copy(), a[6:9].copy(), a[9:12].copy()
    return d


# ---- host-buffer entry points (numpy in, numpy out; copies are inside the C call) ---------------------------------
def _np_prec(a):
    if a.dtype == np.float32:
        return PP_F32
    if a.dtype == np.float64:
        return PP_F64
    raise TypeError("host arrays must be float32 or float64")


def _host(a, shape, dtype, name):
    if not isinstance(a, np.ndarray) or a.dtype != dtype or a.shape != tuple(shape) or not a.flags.c_contiguous:
        raise ValueError("%s must be a C-contiguous numpy array of shape %s and dtype %s" % (name, shape, dtype))
    return a.ctypes.data


def pp_forces_host(pos, mass, G=1.0, delta=0.0, want_pot=False, acc=None, pot=None, stream=None):
    prec = _np_prec(pos)
    N = pos.shape[0]
    if acc is None:
        acc = np.empty((N, 3), dtype=pos.dtype)
    if pot is None and want_pot:
        pot = np.empty((N,), dtype=pos.dtype)
    _check(lib().pp_forces_host(_host(pos, (N, 3), pos.dtype, "pos"), _host(mass, (N,), pos.dtype, "mass"),
                                _host(acc, (N, 3), pos.dtype, "acc"),
                                _host(pot, (N,), pos.dtype, "pot") if pot is not None else None, N, float(G),
                                float(delta), prec, _stream(stream)), "pp_forces_host")
    return acc, pot


def pp_step_kdk_host(pos, vel, mass, acc, dt, nsteps, G=1.0, delta=0.0, acc_valid=False, pot=None, stream=None):
    prec = _np_prec(pos)
    N = pos.shape[0]
    _check(lib().pp_step_kdk_host(_host(pos, (N, 3), pos.dtype, "pos"), _host(vel, (N, 3), pos.dtype, "vel"),
                                  _host(mass, (N,), pos.dtype, "mass"), _host(acc, (N, 3), pos.dtype, "acc"),
                                  _host(pot, (N,), pos.dtype, "pot") if pot is not None else None, N, float(dt), int(nsteps), float(G), float(delta), prec,
                                  PP_ACC_VALID if acc_valid else 0, _stream(stream)), "pp_step_kdk_host")


def pp_invariants_host(pos, vel, mass, G=1.0, delta=0.0, pot=None, stream=None):
    prec = _np_prec(pos)
    N = pos.shape[0]
    out16 = np.empty(16, dtype=np.float64)
    _check(lib().pp_invariants_host(_host(pos, (N, 3), pos.dtype, "pos"), _host(vel, (N, 3), pos.dtype, "vel"),
                                    _host(mass, (N,), pos.dtype, "mass"),
                                    _host(pot, (N,), pos.dtype, "pot") if pot is not None else None, N, float(G),
                                    float(delta), prec, out16.ctypes.data, _stream(stream)), "pp_invariants_host")
    return out16
