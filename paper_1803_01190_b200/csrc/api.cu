// api.cu -- the C ABI of libppgrav (include/ppgrav.h): argument checking, the per-device workspace, and the
// sequencing of the kernels.  No arithmetic of the method lives here.
//
//   pp_forces     = pack -> force sweep over (i-block, j-split) units -> finalize
//   pp_step_kdk   = [initial solve] -> nsteps x { kick+drift+pack -> force sweep -> finalize+kick }
//   pp_invariants = [FP64 potential sweep -> finalize] -> block partials -> final sum
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <utility>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "ppgrav_internal.h"

namespace ppgrav {

namespace {

// NVTX range around an ABI call (header-only nvtx3: a no-op unless a profiler is attached)
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

thread_local char t_err[512] = "";
std::atomic<int64_t> g_launches{0};
std::atomic<int64_t> g_cfg_split{0};
std::atomic<int64_t> g_cfg_graph{1};
std::atomic<int64_t> g_cfg_profile{0};
std::atomic<int64_t> g_cfg_equal_mass{1};
std::atomic<int64_t> g_cfg_shape{0};
std::atomic<int64_t> g_cfg_symmetric{1};
std::atomic<int64_t> g_cfg_band_rows{0};
std::vector<std::pair<cudaEvent_t, cudaEvent_t>> g_prof;   // guarded by g_mu (every sweep is launched under it)

constexpr int kMaxDevices = 64;
constexpr int64_t kMaxN = (int64_t)1 << 28;
constexpr int kNumBuf = 8;
enum { B_PACKED = 0, B_PARTIAL, B_INV, B_POT64, B_TILE_MASS, B_PARTIAL_J, B_BLOCK_MASS, B_ACC_J };
// the j-side rows of the symmetric sweep grow as N^2 / (2 x 2048) x 16 B (FP64: 32 B): 4.3 GB at N = 2^20, 17 GB at 2^21.  Up to
// kMaxPartialJBytes they are kept whole (one sweep launch, finalize reads them directly); beyond, the partner offsets
// are cut into bands of at most kBandBytes whose rows are reused and folded into running sums
constexpr size_t kMaxPartialJBytes = (size_t)48 << 30;
constexpr size_t kBandBytes = (size_t)16 << 30;

// one instantiated CUDA graph of an interior KDK step (sweep + finalize_kick_drift_pack), reused while every
// kernel argument it was recorded with is unchanged
struct StepGraph {
    cudaGraphExec_t exec = nullptr;
    const void *pos = nullptr, *vel = nullptr, *mass = nullptr, *acc = nullptr, *packed = nullptr, *partial = nullptr,
               *tm = nullptr;
    int64_t N = 0, n_pad = 0, part_stride = 0;
    int precision = -1, cls = -1, split = 0, threads = 0, ipt = 0, sym = 0;
    const void* partial_j = nullptr;
    double dt = 0, G = 0, delta = 0;
};

struct Workspace {
    void* buf[kNumBuf] = {};
    size_t cap[kNumBuf] = {};
    int sm_count = 0;
    // stream-ordered reuse: the workspace belongs to the stream of the last call; a call on another stream first
    // waits (on the device) for `done`, recorded at the end of every call that touched the workspace
    cudaStream_t last_stream = nullptr;
    bool used = false;
    cudaEvent_t done = nullptr;
    // graph replay from the legacy default stream goes through this internal stream (fork/join by events)
    cudaStream_t side = nullptr;
    cudaEvent_t fork = nullptr, join = nullptr;
    StepGraph graph;
};
Workspace g_ws[kMaxDevices];
std::mutex g_mu;

int current_workspace(Workspace** out) {
    int dev = -1;
    PP_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) {
        set_error("device ordinal %d out of range", dev);
        return PP_ECUDA;
    }
    Workspace* w = &g_ws[dev];
    if (w->sm_count == 0) {
        int sm = 0;
        PP_CUDA(cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev));
        w->sm_count = sm;
    }
    *out = w;
    return PP_OK;
}

// grow-only buffer; cudaFree synchronises the device, so work still reading the old block has finished
int ensure(Workspace* w, int which, size_t bytes, void** out) {
    if (bytes > w->cap[which]) {
        if (w->buf[which]) {
            cudaFree(w->buf[which]);
            w->buf[which] = nullptr;
            w->cap[which] = 0;
        }
        void* p = nullptr;
        const cudaError_t e = cudaMalloc(&p, bytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            set_error("workspace allocation of %zu bytes failed: %s", bytes, cudaGetErrorString(e));
            return PP_ENOMEM;
        }
        w->buf[which] = p;
        w->cap[which] = bytes;
    }
    *out = w->buf[which];
    return PP_OK;
}

bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }

int check_common(const char* fn, int64_t N, double G, double delta, int precision) {
    if (precision != PP_F32 && precision != PP_F64 && precision != PP_MIXED) {
        set_error("%s: precision must be PP_F32, PP_F64 or PP_MIXED (got %d)", fn, precision);
        return PP_EINVAL;
    }
    if (N < 1 || N > kMaxN) {
        set_error("%s: N = %lld outside [1, 2^28]", fn, (long long)N);
        return PP_EINVAL;
    }
    if (!std::isfinite(G) || !std::isfinite(delta) || delta < 0.0) {
        set_error("%s: G must be finite and delta finite and >= 0 (G = %g, delta = %g)", fn, G, delta);
        return PP_EINVAL;
    }
    return PP_OK;
}

int check_ptr(const char* fn, const char* name, const void* p, int precision, bool required) {
    if (!p) {
        if (!required) return PP_OK;
        set_error("%s: %s is NULL", fn, name);
        return PP_EINVAL;
    }
    if (!aligned(p, precision == PP_F32 ? 4 : 8)) {
        set_error("%s: %s is not aligned to its element size", fn, name);
        return PP_EINVAL;
    }
    return PP_OK;
}

#define PP_TRY(expr)              \
    do {                          \
        const int rc__ = (expr);  \
        if (rc__ != PP_OK) return rc__; \
    } while (0)

// precision of the pair sweep (packed copy, partial sums): PP_MIXED keeps an FP64 state but sweeps in FP32
int sweep_precision(int precision) { return precision == PP_F64 ? PP_F64 : PP_F32; }
size_t sweep_elem_bytes(int precision) { return precision == PP_F64 ? 8 : 4; }

// the pair sweep, optionally bracketed by events (PP_CFG_PROFILE)
int sweep(const Plan& p, int precision, const void* packed, const void* tile_mass, void* partial, int64_t N,
          double delta, int mode, cudaStream_t st, const void* block_mass = nullptr, void* partial_j = nullptr,
          void* acc_j = nullptr) {
    const bool prof = g_cfg_profile.load() != 0;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (prof) {
        PP_CUDA(cudaEventCreate(&e0));
        PP_CUDA(cudaEventCreate(&e1));
        PP_CUDA(cudaEventRecord(e0, st));
    }
    int rc;
    if (p.sym && sweep_precision(precision) == PP_F32)
        rc = launch_force_sym_f32(p, (const float*)packed, (const float*)tile_mass, (const float*)block_mass,
                                  (float4*)partial, (float4*)partial_j, (float4*)acc_j, delta, mode, st);
    else if (p.sym)
        rc = launch_force_sym_f64(p, (const double*)packed, (const double*)tile_mass, (const double*)block_mass,
                                  (double4*)partial, (double4*)partial_j, (double4*)acc_j, delta, mode, st);
    else
        rc = sweep_precision(precision) == PP_F32
                 ? launch_force_f32(p, (const float*)packed, (const float*)tile_mass, (float4*)partial, N, delta, mode, st)
                 : launch_force_f64(p, (const double*)packed, (const double*)tile_mass, (double4*)partial, N, delta, mode,
                                    st);
    if (prof) {
        PP_CUDA(cudaEventRecord(e1, st));
        g_prof.emplace_back(e0, e1);
    }
    return rc;
}

// where finalize finds the j-side sums of a symmetric sweep, and how many i-side partials there are per body
struct JSide {
    const void* ptr;
    int rows, split;
};
JSide jside(const Plan& p, const void* partial_j, const void* acc_j) {
    if (!p.sym) return {nullptr, 0, p.split};
    if (p.sym_bands > 1) return {acc_j, 2, 0};   // everything is already in the running TwoSum (value, error) sums
    return {partial_j, p.sym_h, p.split};
}

// one gravity solve on already packed bodies: sweep + finalize (optionally with the closing half-kick)
// (acc, pot, vel address the p.i_count bodies of the plan's i-range; p must be the plan of the mode pot selects;
// block_mass / partial_j: the symmetric sweep's extra input and j-side rows, unused otherwise)
int solve_packed(const Plan& p, int precision, const void* packed, const void* tile_mass, void* partial, int64_t N,
                 double G, double delta, void* acc, void* pot, void* vel, double kick, cudaStream_t st,
                 const void* block_mass = nullptr, void* partial_j = nullptr, void* acc_j = nullptr) {
    const int mode = pot ? MODE_FORCE_POT : MODE_FORCE;
    PP_TRY(sweep(p, precision, packed, tile_mass, partial, N, delta, mode, st, block_mass, partial_j, acc_j));
    const JSide j = jside(p, partial_j, acc_j);
    if (precision == PP_F32)
        return launch_finalize_f32((const float4*)partial, j.split, p.part_stride, p.i_count, G, (float*)acc,
                                   (float*)pot, (float*)vel, kick, st, (const float4*)j.ptr, j.rows, p.part_stride);
    if (precision == PP_MIXED)
        return launch_finalize_mixed((const float4*)partial, j.split, p.part_stride, p.i_count, G, (double*)acc,
                                     (double*)pot, (double*)vel, kick, st, (const float4*)j.ptr, j.rows,
                                     p.part_stride);
    return launch_finalize_f64((const double4*)partial, j.split, p.part_stride, p.i_count, G, (double*)acc,
                               (double*)pot, (double*)vel, kick, 0, st, (const double4*)j.ptr, j.rows,
                               p.part_stride);
}

int pack_state(int precision, const void* pos, const void* mass, void* packed, int64_t N, int64_t n_pad,
               cudaStream_t st) {
    if (precision == PP_F32) return launch_pack_f32((const float*)pos, (const float*)mass, (float*)packed, N, n_pad, st);
    if (precision == PP_MIXED)
        return launch_pack_f64_to_f32((const double*)pos, (const double*)mass, (float*)packed, N, n_pad, st);
    return launch_pack_f64((const double*)pos, (const double*)mass, (double*)packed, N, n_pad, st);
}

// per-j-tile common mass for the plan's tiles (the masses do not change inside an API call: computed once per call)
int tile_masses(Workspace* w, const Plan& p, int precision, const void* mass, int64_t N, int enable, void** out,
                cudaStream_t st) {
    PP_TRY(ensure(w, B_TILE_MASS, (size_t)p.n_tiles * sweep_elem_bytes(precision), out));
    if (precision == PP_F32)
        return launch_tile_mass_f32((const float*)mass, (float*)*out, N, p.tile_j, p.n_tiles, enable, st);
    if (precision == PP_MIXED)
        return launch_tile_mass_f64_to_f32((const double*)mass, (float*)*out, N, p.tile_j, p.n_tiles, enable, st);
    return launch_tile_mass_f64((const double*)mass, (double*)*out, N, p.tile_j, p.n_tiles, enable, st);
}

int kick_drift_pack(int precision, void* pos, void* vel, const void* acc, const void* mass, void* packed, int64_t N,
                    int64_t n_pad, double kick, double dt, cudaStream_t st) {
    if (precision == PP_F32)
        return launch_kick_drift_pack_f32((float*)pos, (float*)vel, (const float*)acc, (const float*)mass,
                                          (float*)packed, N, n_pad, kick, dt, st);
    if (precision == PP_MIXED)
        return launch_kick_drift_pack_mixed((double*)pos, (double*)vel, (const double*)acc, (const double*)mass,
                                            (float*)packed, N, n_pad, kick, dt, st);
    return launch_kick_drift_pack_f64((double*)pos, (double*)vel, (const double*)acc, (const double*)mass,
                                      (double*)packed, N, n_pad, kick, dt, st);
}

// Every API call that uses the workspace brackets its work with enter()/leave(): calls on ONE stream are ordered by
// the stream; a call on a different stream than the previous one waits on the device for the previous call's work
// (the packed bodies and partial sums are shared), so concurrent multi-stream use is serialised instead of racing.
int enter(Workspace* w, cudaStream_t st) {
    if (!w->done) PP_CUDA(cudaEventCreateWithFlags(&w->done, cudaEventDisableTiming));
    if (w->used && st != w->last_stream) PP_CUDA(cudaStreamWaitEvent(st, w->done, 0));
    return PP_OK;
}
int leave(Workspace* w, cudaStream_t st) {
    PP_CUDA(cudaEventRecord(w->done, st));
    w->last_stream = st;
    w->used = true;
    return PP_OK;
}

void drop_graph(Workspace* w) {
    if (w->graph.exec) cudaGraphExecDestroy(w->graph.exec);
    w->graph = StepGraph{};
}

// The plans, packed bodies, partial sums and tile masses of one API call.  `force` is the plan of the force-only
// sweep, `force_pot` of the sweep that also produces the potential; they share the shape class (hence tile_j and the
// tile masses) and differ at most in i-bodies per thread, so one packed array, padded for both, serves the call.
struct Solve {
    Plan force, force_pot;
    int64_t n_pad = 0;
    void *packed = nullptr, *partial = nullptr, *tm = nullptr;
    void *partial_j = nullptr, *bm = nullptr, *acc_j = nullptr;   // symmetric sweep only
    const Plan& plan(int mode) const { return mode == MODE_FORCE ? force : force_pot; }
};

int forced_class() { return (int)g_cfg_shape.load() - 1; }   // PP_CFG_SHAPE: 0 auto, 1 large, 2 mid, 3 small

// The symmetric sweep (every unordered pair once, force_sym_f32.cu / force_sym_f64.cu) serves full solves:
// PP_CFG_SYMMETRIC 0 = never, 1 = when the one-sided plan would take the large class and the j-side rows fit the cap,
// 2 = always (tests).  Returns true and fills *p if it is to be used.
bool symmetric_plan(int64_t N, int sweep_prec, int mode, int sm_count, bool full, Plan* p) {
    const int64_t cfg = g_cfg_symmetric.load();
    if (cfg == 0 || !full || (mode != MODE_FORCE && mode != MODE_FORCE_POT)) return false;
    if (cfg == 1) {   // automatic: not when a shape class is pinned (PP_CFG_SHAPE addresses the one-sided kernels)
        if (forced_class() >= 0) return false;
        // measured: faster than every one-sided class from N = 2^14 on (2^14: 140 against
        // 156 us, 2^15: 328 against 488 us in FP32), slower at 2^13 (101 against 56 us)
        if (N < 14000) return false;
    }
    size_t jbytes = 0, abytes = 0;
    // pinned symmetric sweep (PP_CFG_SYMMETRIC = 2): PP_CFG_SHAPE large / mid pins its 256- / 128-body tile variant
    const int fine = cfg == 2 ? (forced_class() == CLS_LARGE ? 0 : forced_class() == CLS_MID ? 1 : -1) : -1;
    const int64_t fs = g_cfg_split.load();
    Plan sp = make_sym_plan(N, sweep_prec, mode, sm_count, fs, kMaxPartialJBytes, &jbytes, &abytes, fine);
    if (sp.sym_bands > 1) sp = make_sym_plan(N, sweep_prec, mode, sm_count, fs, kBandBytes, &jbytes, &abytes, fine);
    const int64_t force_rows = g_cfg_band_rows.load();   // PP_CFG_SYM_BAND_ROWS (tests): at most that many rows per band
    if (force_rows >= 1) {
        const size_t row_bytes = (size_t)sp.part_stride * (sweep_prec == PP_F64 ? 32 : 16);
        sp = make_sym_plan(N, sweep_prec, mode, sm_count, fs, (size_t)force_rows * row_bytes, &jbytes, &abytes, fine);
    }
    *p = sp;
    return true;
}

int prepare_solve(Workspace* w, int64_t N, int precision, const void* mass, bool want_force_only, cudaStream_t st,
                  Solve* s, int64_t i_begin = 0, int64_t i_count = -1) {
    const int sp = sweep_precision(precision);
    const int64_t fs = g_cfg_split.load();
    const bool full = i_begin == 0 && (i_count < 0 || i_count == N);
    // the class is chosen for the mode that dominates the call
    const int lead = want_force_only ? MODE_FORCE : MODE_FORCE_POT;
    Plan first;
    bool sym = symmetric_plan(N, sp, lead, w->sm_count, full, &first);
    if (sym) {   // its j-side rows are the one big allocation of the library: if HBM cannot hold them, sweep one-sidedly
        const size_t row_bytes = (size_t)first.part_stride * 4 * sweep_elem_bytes(precision);
        const size_t jb = std::max<size_t>((size_t)std::min(first.sym_rows, std::max(first.sym_h, 1)) * row_bytes, 16);
        if (ensure(w, B_PARTIAL_J, jb, &s->partial_j) != PP_OK ||
            (first.sym_bands > 1 && ensure(w, B_ACC_J, 2 * row_bytes, &s->acc_j) != PP_OK)) {
            if (g_cfg_symmetric.load() == 2) return PP_ENOMEM;   // pinned by the caller: report, do not fall back
            set_error("");
            sym = false;
        }
    }
    if (sym) {
        s->force = s->force_pot = first;
        s->force.mode = MODE_FORCE;
        s->force_pot.mode = MODE_FORCE_POT;
    } else {
        first = make_plan(N, sp, lead, w->sm_count, fs, forced_class(), i_begin, i_count);
        s->force = lead == MODE_FORCE ? first : make_plan(N, sp, MODE_FORCE, w->sm_count, fs, first.cls, i_begin, i_count);
        s->force_pot = lead == MODE_FORCE_POT
                           ? first
                           : make_plan(N, sp, MODE_FORCE_POT, w->sm_count, fs, first.cls, i_begin, i_count);
    }
    s->n_pad = std::max(s->force.n_pad, s->force_pot.n_pad);
    const size_t body = 4 * sweep_elem_bytes(precision);
    const size_t part = std::max((size_t)s->force.split * (size_t)s->force.part_stride,
                                 (size_t)s->force_pot.split * (size_t)s->force_pot.part_stride);
    PP_TRY(ensure(w, B_PACKED, (size_t)s->n_pad * body, &s->packed));
    PP_TRY(ensure(w, B_PARTIAL, part * body, &s->partial));
    if (mass) PP_TRY(tile_masses(w, first, precision, mass, N, (int)g_cfg_equal_mass.load(), &s->tm, st));
    if (sym) {
        PP_TRY(ensure(w, B_BLOCK_MASS, (size_t)first.n_iblocks * sweep_elem_bytes(precision), &s->bm));
        if (mass) {   // common mass per i-block: the same kernel with tile = block
            const int em = (int)g_cfg_equal_mass.load();
            if (precision == PP_F32)
                PP_TRY(launch_tile_mass_f32((const float*)mass, (float*)s->bm, N, first.i_per_cta, first.n_iblocks, em, st));
            else if (precision == PP_MIXED)
                PP_TRY(launch_tile_mass_f64_to_f32((const double*)mass, (float*)s->bm, N, first.i_per_cta,
                                                   first.n_iblocks, em, st));
            else
                PP_TRY(launch_tile_mass_f64((const double*)mass, (double*)s->bm, N, first.i_per_cta, first.n_iblocks,
                                            em, st));
        }
    }
    return PP_OK;
}

// finalize + closing kick + opening kick + drift + re-pack (interior steps of pp_step_kdk)
int finalize_kick_drift_pack(const Plan& p, int precision, const void* partial, int64_t N, double G, void* acc,
                             void* vel, void* pos, const void* mass, void* packed, double kick, double dt,
                             cudaStream_t st, const void* partial_j = nullptr, const void* acc_j = nullptr) {
    const JSide j = jside(p, partial_j, acc_j);
    if (precision == PP_F32)
        return launch_finalize_kick_drift_pack_f32((const float4*)partial, j.split, p.part_stride, N, G, (float*)acc,
                                                   (float*)vel, (float*)pos, (const float*)mass, (float*)packed, kick,
                                                   dt, st, (const float4*)j.ptr, j.rows, p.part_stride);
    if (precision == PP_MIXED)
        return launch_finalize_kick_drift_pack_mixed((const float4*)partial, j.split, p.part_stride, N, G,
                                                     (double*)acc, (double*)vel, (double*)pos, (const double*)mass,
                                                     (float*)packed, kick, dt, st, (const float4*)j.ptr, j.rows,
                                                     p.part_stride);
    return launch_finalize_kick_drift_pack_f64((const double4*)partial, j.split, p.part_stride, N, G, (double*)acc,
                                               (double*)vel, (double*)pos, (const double*)mass, (double*)packed, kick,
                                               dt, st, (const double4*)j.ptr, j.rows, p.part_stride);
}

}  // namespace

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof(t_err), fmt, ap);
    va_end(ap);
}

int cuda_fail(cudaError_t e, const char* what) {
    cudaGetLastError();   // clear the sticky-less error state
    set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    return PP_ECUDA;
}

void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

}  // namespace ppgrav

using namespace ppgrav;

extern "C" {

int pp_version(void) { return PPGRAV_VERSION; }

const char* pp_last_error(void) { return t_err; }

int64_t pp_launch_count(void) { return g_launches.load(); }

int pp_configure(int key, int64_t value) {
    if (key == PP_CFG_SPLIT_J && value >= 0 && value <= 4096) { g_cfg_split.store(value); return PP_OK; }
    if (key == PP_CFG_GRAPH && (value == 0 || value == 1)) { g_cfg_graph.store(value); return PP_OK; }
    if (key == PP_CFG_PROFILE && (value == 0 || value == 1)) { g_cfg_profile.store(value); return PP_OK; }
    if (key == PP_CFG_EQUAL_MASS && (value == 0 || value == 1)) { g_cfg_equal_mass.store(value); return PP_OK; }
    if (key == PP_CFG_SHAPE && value >= 0 && value <= kNumClasses) { g_cfg_shape.store(value); return PP_OK; }
    if (key == PP_CFG_SYMMETRIC && value >= 0 && value <= 2) { g_cfg_symmetric.store(value); return PP_OK; }
    if (key == PP_CFG_SYM_BAND_ROWS && value >= 0 && value <= (1 << 20)) { g_cfg_band_rows.store(value); return PP_OK; }
    set_error("pp_configure: unknown key %d or value %lld out of range", key, (long long)value);
    return PP_EINVAL;
}

int pp_profile_read(double* out2) {
    if (!out2) { set_error("pp_profile_read: out2 is NULL"); return PP_EINVAL; }
    std::lock_guard<std::mutex> lk(g_mu);
    double total = 0.0;
    int rc = PP_OK;
    for (auto& ev : g_prof) {
        float ms = 0.f;
        cudaError_t e = cudaEventSynchronize(ev.second);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, ev.first, ev.second);
        if (e != cudaSuccess && rc == PP_OK) rc = cuda_fail(e, "pp_profile_read");
        total += ms;
        cudaEventDestroy(ev.first);
        cudaEventDestroy(ev.second);
    }
    out2[0] = total;
    out2[1] = (double)g_prof.size();
    g_prof.clear();
    return rc;
}

int pp_release(int device) {
    std::lock_guard<std::mutex> lk(g_mu);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess) { cudaGetLastError(); return PP_OK; }   // nothing was ever allocated
    if (device >= ndev || device >= kMaxDevices || device < -1) {
        set_error("pp_release: no device %d", device);
        return PP_EINVAL;
    }
    int prev = 0;
    PP_CUDA(cudaGetDevice(&prev));
    for (int d = 0; d < ndev && d < kMaxDevices; ++d) {
        if (device != -1 && d != device) continue;
        Workspace& w = g_ws[d];
        bool any = w.done || w.side || w.graph.exec;
        for (int b = 0; b < kNumBuf; ++b) any = any || w.buf[b];
        if (!any) continue;
        PP_CUDA(cudaSetDevice(d));
        PP_CUDA(cudaDeviceSynchronize());
        for (int b = 0; b < kNumBuf; ++b) {
            if (w.buf[b]) cudaFree(w.buf[b]);
            w.buf[b] = nullptr;
            w.cap[b] = 0;
        }
        drop_graph(&w);
        if (w.done) cudaEventDestroy(w.done);
        if (w.fork) cudaEventDestroy(w.fork);
        if (w.join) cudaEventDestroy(w.join);
        if (w.side) cudaStreamDestroy(w.side);
        w.done = w.fork = w.join = nullptr;
        w.side = nullptr;
        w.used = false;
        w.last_stream = nullptr;
    }
    PP_CUDA(cudaSetDevice(prev));
    return PP_OK;
}

int pp_plan_query(int64_t N, int precision, int with_pot, int64_t* out16) {
    int64_t* out12 = out16;
    if (!out16) { set_error("pp_plan_query: out16 is NULL"); return PP_EINVAL; }
    PP_TRY(check_common("pp_plan_query", N, 1.0, 0.0, precision));
    int sm = 148;   // B200; used when no device is present (host-side planning only)
    int dev = -1;
    if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) sm = v;
    }
    cudaGetLastError();
    precision = sweep_precision(precision);
    const int mode = with_pot ? MODE_FORCE_POT : MODE_FORCE;
    Plan p;
    if (!symmetric_plan(N, precision, mode, sm, true, &p))
        p = make_plan(N, precision, mode, sm, g_cfg_split.load(), forced_class());
    out12[0] = p.i_per_cta;
    out12[1] = p.tile_j;
    out12[2] = p.split;
    out12[3] = (int64_t)p.n_iblocks * p.split;
    out12[4] = p.ctas_per_sm;
    out12[5] = sm;
    // pipe operations per pair EVALUATION on a j-tile of mixed masses; the symmetric sweep's evaluation serves two
    // ordered pairs (out16[12])
    if (p.sym) out12[6] = precision == PP_F32 ? (with_pot ? 18 : 16) : (with_pot ? 23 : 20);
    else out12[6] = precision == PP_F32 ? (with_pot ? 13 : 12) : (with_pot ? 18 : 16);
    out12[7] = 1;
    out12[8] = p.sym ? 3 : p.cls;
    out12[9] = p.threads;
    out12[10] = p.ipt;
    out12[11] = p.n_iblocks;
    out16[12] = p.sym ? 2 : 1;
    out16[13] = p.sym ? p.sym_h : 0;
    out16[14] = p.sym ? p.sym_bands : 0;
    // bytes of workspace this solve keeps on the device: packed bodies, split-j partials, tile (and block) masses and,
    // for the symmetric sweep, the j-side rows of one band plus the running sums of a banded solve
    const size_t body = precision == PP_F64 ? 32 : 16;
    size_t bytes = (size_t)p.n_pad * body + (size_t)p.split * (size_t)p.part_stride * body + (size_t)p.n_tiles * (body / 4);
    if (p.sym) {
        const size_t row_bytes = (size_t)p.part_stride * body;
        bytes += (size_t)std::min(p.sym_rows, std::max(p.sym_h, 1)) * row_bytes + (size_t)p.n_iblocks * (body / 4);
        if (p.sym_bands > 1) bytes += 2 * row_bytes;
    }
    out16[15] = (int64_t)bytes;
    return PP_OK;
}

int pp_equal_mass_tiles(const void* mass, int64_t N, int precision, int64_t* out2, void* stream) {
    if (!out2) { set_error("pp_equal_mass_tiles: out2 is NULL"); return PP_EINVAL; }
    PP_TRY(check_common("pp_equal_mass_tiles", N, 1.0, 0.0, precision));
    PP_TRY(check_ptr("pp_equal_mass_tiles", "mass", mass, precision, true));
    std::lock_guard<std::mutex> lk(g_mu);
    Workspace* w = nullptr;
    PP_TRY(current_workspace(&w));
    cudaStream_t st = (cudaStream_t)stream;
    PP_TRY(enter(w, st));
    Plan plan;
    if (!symmetric_plan(N, sweep_precision(precision), MODE_FORCE, w->sm_count, true, &plan))
        plan = make_plan(N, sweep_precision(precision), MODE_FORCE, w->sm_count, g_cfg_split.load(), forced_class());
    void* tm;
    PP_TRY(tile_masses(w, plan, precision, mass, N, 1, &tm, st));
    const size_t eb = sweep_elem_bytes(precision);
    std::vector<unsigned char> host((size_t)plan.n_tiles * eb);
    PP_CUDA(cudaMemcpyAsync(host.data(), tm, host.size(), cudaMemcpyDeviceToHost, st));
    PP_TRY(leave(w, st));
    PP_CUDA(cudaStreamSynchronize(st));
    // (the symmetric plan also sweeps tiles that lie wholly in the padding; only tiles with a real body are counted)
    const int real_tiles = (int)((N + plan.tile_j - 1) / plan.tile_j);
    int64_t common = 0;
    for (int t = 0; t < real_tiles; ++t) {
        if (eb == 4) { float v; std::memcpy(&v, &host[(size_t)t * 4], 4); common += (v == v); }
        else { double v; std::memcpy(&v, &host[(size_t)t * 8], 8); common += (v == v); }
    }
    out2[0] = real_tiles;
    out2[1] = common;
    return PP_OK;
}

int pp_forces_range(const void* pos, const void* mass, void* acc, void* pot, int64_t N, int64_t i_begin,
                    int64_t i_count, double G, double delta, int precision, void* stream) {
    NvtxRange nvtx_range("pp_forces_range");
    PP_TRY(check_common("pp_forces_range", N, G, delta, precision));
    PP_TRY(check_ptr("pp_forces_range", "pos", pos, precision, true));
    PP_TRY(check_ptr("pp_forces_range", "mass", mass, precision, true));
    PP_TRY(check_ptr("pp_forces_range", "acc", acc, precision, true));
    PP_TRY(check_ptr("pp_forces_range", "pot", pot, precision, false));
    if (i_begin < 0 || i_count < 1 || i_begin > N - i_count) {
        set_error("pp_forces_range: i-range [%lld, %lld + %lld) outside [0, N = %lld) or empty", (long long)i_begin,
                  (long long)i_begin, (long long)i_count, (long long)N);
        return PP_EINVAL;
    }
    std::lock_guard<std::mutex> lk(g_mu);
    Workspace* w = nullptr;
    PP_TRY(current_workspace(&w));
    cudaStream_t st = (cudaStream_t)stream;
    PP_TRY(enter(w, st));
    Solve s;
    PP_TRY(prepare_solve(w, N, precision, mass, pot == nullptr, st, &s, i_begin, i_count));
    PP_TRY(pack_state(precision, pos, mass, s.packed, N, s.n_pad, st));
    PP_TRY(solve_packed(s.plan(pot ? MODE_FORCE_POT : MODE_FORCE), precision, s.packed, s.tm, s.partial, N, G, delta,
                        acc, pot, nullptr, 0.0, st, s.bm, s.partial_j, s.acc_j));
    return leave(w, st);
}

int pp_forces(const void* pos, const void* mass, void* acc, void* pot, int64_t N, double G, double delta,
              int precision, void* stream) {
    PP_TRY(check_common("pp_forces", N, G, delta, precision));
    return pp_forces_range(pos, mass, acc, pot, N, 0, N, G, delta, precision, stream);
}

int pp_kick_drift(void* pos, void* vel, const void* acc, int64_t n, double kick, double dt, int precision,
                  void* stream) {
    PP_TRY(check_common("pp_kick_drift", n, 1.0, 0.0, precision));
    PP_TRY(check_ptr("pp_kick_drift", "pos", pos, precision, true));
    PP_TRY(check_ptr("pp_kick_drift", "vel", vel, precision, true));
    PP_TRY(check_ptr("pp_kick_drift", "acc", acc, precision, true));
    if (!std::isfinite(kick) || !std::isfinite(dt)) {
        set_error("pp_kick_drift: kick and dt must be finite");
        return PP_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (precision == PP_F32)
        return launch_kick_drift_f32((float*)pos, (float*)vel, (const float*)acc, n, kick, dt, st);
    return launch_kick_drift_f64((double*)pos, (double*)vel, (const double*)acc, n, kick, dt, st);
}

int pp_step_kdk(void* pos, void* vel, const void* mass, void* acc, void* pot, int64_t N, double dt, int64_t nsteps,
                double G, double delta, int precision, unsigned flags, void* stream) {
    NvtxRange nvtx_range("pp_step_kdk");
    PP_TRY(check_common("pp_step_kdk", N, G, delta, precision));
    PP_TRY(check_ptr("pp_step_kdk", "pos", pos, precision, true));
    PP_TRY(check_ptr("pp_step_kdk", "vel", vel, precision, true));
    PP_TRY(check_ptr("pp_step_kdk", "mass", mass, precision, true));
    PP_TRY(check_ptr("pp_step_kdk", "acc", acc, precision, true));
    PP_TRY(check_ptr("pp_step_kdk", "pot", pot, precision, false));
    if (!std::isfinite(dt) || nsteps < 0 || (flags & ~PP_ACC_VALID)) {
        set_error("pp_step_kdk: dt must be finite, nsteps >= 0, flags a subset of PP_ACC_VALID");
        return PP_EINVAL;
    }
    std::lock_guard<std::mutex> lk(g_mu);
    Workspace* w = nullptr;
    PP_TRY(current_workspace(&w));
    cudaStream_t st = (cudaStream_t)stream;
    const bool cold = !(flags & PP_ACC_VALID);
    if (nsteps == 0 && !cold) return PP_OK;   // nothing to solve
    PP_TRY(enter(w, st));
    // gravity solves of this call: force-only ones and (at most one, the last) with the potential
    const int64_t n_pot = pot ? 1 : 0;
    const int64_t n_force = (cold ? 1 : 0) + nsteps - n_pot;
    Solve s;
    PP_TRY(prepare_solve(w, N, precision, mass, n_force >= n_pot, st, &s));
    if (cold) {   // a(t0): the one extra gravity solve of a cold start
        void* pot0 = nsteps == 0 ? pot : nullptr;
        PP_TRY(pack_state(precision, pos, mass, s.packed, N, s.n_pad, st));
        PP_TRY(solve_packed(s.plan(pot0 ? MODE_FORCE_POT : MODE_FORCE), precision, s.packed, s.tm, s.partial, N, G,
                            delta, acc, pot0, nullptr, 0.0, st, s.bm, s.partial_j, s.acc_j));
    }
    if (nsteps == 0) return leave(w, st);
    const double half = 0.5 * dt;
    // step 1 opens with kick + drift + pack (which also writes the padding of the packed array); every interior
    // boundary between two steps is ONE pass (finalize + closing kick + opening kick + drift + pack); the last
    // solve alone may carry the potential and ends with finalize + closing kick.
    PP_TRY(kick_drift_pack(precision, pos, vel, acc, mass, s.packed, N, s.n_pad, half, dt, st));
    const int64_t nbody = nsteps - 1;
    const Plan& pf = s.force;

    // Small N is launch-bound (a solve of 2048 bodies is a few microseconds of pipe time): the interior step
    // (sweep + update pass) is recorded into a CUDA graph once and replayed; the instantiated graph is kept while every
    // kernel argument is unchanged, so a caller that advances the same buffers call after call pays for it once.
    // The legacy default stream cannot be captured: its work is forked to an internal stream and joined back by events.
    StepGraph key;
    key.pos = pos; key.vel = vel; key.mass = mass; key.acc = acc; key.packed = s.packed; key.partial = s.partial;
    key.tm = s.tm; key.N = N; key.n_pad = s.n_pad; key.part_stride = pf.part_stride; key.precision = precision;
    key.cls = pf.cls; key.split = pf.split; key.threads = pf.threads; key.ipt = pf.ipt; key.dt = dt; key.G = G;
    key.delta = delta; key.sym = pf.sym * 1000 + pf.sym_bands; key.partial_j = s.partial_j;
    const StepGraph& g = w->graph;
    const bool hit = g.exec && g.pos == key.pos && g.vel == key.vel && g.mass == key.mass && g.acc == key.acc &&
                     g.packed == key.packed && g.partial == key.partial && g.tm == key.tm && g.N == key.N &&
                     g.n_pad == key.n_pad && g.part_stride == key.part_stride && g.precision == key.precision &&
                     g.cls == key.cls && g.split == key.split && g.threads == key.threads && g.ipt == key.ipt &&
                     g.dt == key.dt && g.G == key.G && g.delta == key.delta && g.sym == key.sym &&
                     g.partial_j == key.partial_j;
    const bool graph_ok = g_cfg_graph.load() && !g_cfg_profile.load() && N <= 65536;
    if (graph_ok && nbody >= 1 && (hit || nbody >= 4)) {
        const bool legacy = st == nullptr || st == cudaStreamLegacy;
        cudaStream_t run = st;
        if (legacy) {
            if (!w->side) {
                PP_CUDA(cudaStreamCreateWithFlags(&w->side, cudaStreamNonBlocking));
                PP_CUDA(cudaEventCreateWithFlags(&w->fork, cudaEventDisableTiming));
                PP_CUDA(cudaEventCreateWithFlags(&w->join, cudaEventDisableTiming));
            }
            run = w->side;
            PP_CUDA(cudaEventRecord(w->fork, st));
            PP_CUDA(cudaStreamWaitEvent(run, w->fork, 0));
        }
        if (!hit) {
            drop_graph(w);
            cudaGraph_t graph = nullptr;
            PP_CUDA(cudaStreamBeginCapture(run, cudaStreamCaptureModeThreadLocal));
            int rc = sweep(pf, precision, s.packed, s.tm, s.partial, N, delta, MODE_FORCE, run, s.bm, s.partial_j, s.acc_j);
            if (rc == PP_OK)
                rc = finalize_kick_drift_pack(pf, precision, s.partial, N, G, acc, vel, pos, mass, s.packed, half, dt,
                                              run, s.partial_j, s.acc_j);
            const cudaError_t ec = cudaStreamEndCapture(run, &graph);
            count_launch(-2);   // the two captured launches were recorded, not run
            if (rc != PP_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
            if (ec != cudaSuccess) return cuda_fail(ec, "cudaStreamEndCapture");
            cudaGraphExec_t exec = nullptr;
            const cudaError_t ei = cudaGraphInstantiate(&exec, graph, 0);
            cudaGraphDestroy(graph);
            if (ei != cudaSuccess) return cuda_fail(ei, "cudaGraphInstantiate");
            w->graph = key;
            w->graph.exec = exec;
        }
        for (int64_t k = 0; k < nbody; ++k) {
            const cudaError_t el = cudaGraphLaunch(w->graph.exec, run);
            if (el != cudaSuccess) { drop_graph(w); return cuda_fail(el, "cudaGraphLaunch"); }
            count_launch(2);
        }
        if (legacy) {
            PP_CUDA(cudaEventRecord(w->join, run));
            PP_CUDA(cudaStreamWaitEvent(st, w->join, 0));
        }
    } else {
        for (int64_t k = 0; k < nbody; ++k) {
            PP_TRY(sweep(pf, precision, s.packed, s.tm, s.partial, N, delta, MODE_FORCE, st, s.bm, s.partial_j, s.acc_j));
            PP_TRY(finalize_kick_drift_pack(pf, precision, s.partial, N, G, acc, vel, pos, mass, s.packed, half, dt, st,
                                            s.partial_j, s.acc_j));
        }
    }
    PP_TRY(solve_packed(s.plan(pot ? MODE_FORCE_POT : MODE_FORCE), precision, s.packed, s.tm, s.partial, N, G, delta,
                        acc, pot, vel, half, st, s.bm, s.partial_j, s.acc_j));
    return leave(w, st);
}

int pp_surface_density(const void* pos, const void* mass, int64_t N, double x0, double y0, double cell, int nx,
                       int ny, int precision, double* sigma, void* stream) {
    PP_TRY(check_common("pp_surface_density", N, 1.0, 0.0, precision));
    PP_TRY(check_ptr("pp_surface_density", "pos", pos, precision, true));
    PP_TRY(check_ptr("pp_surface_density", "mass", mass, precision, true));
    PP_TRY(check_ptr("pp_surface_density", "sigma", sigma, PP_F64, true));
    if (!std::isfinite(x0) || !std::isfinite(y0) || !std::isfinite(cell) || !(cell > 0.0) || nx < 1 || ny < 1 ||
        (int64_t)nx * ny > ((int64_t)1 << 26)) {
        set_error("pp_surface_density: need finite x0, y0, cell > 0 and 1 <= nx*ny <= 2^26");
        return PP_EINVAL;
    }
    Workspace* w = nullptr;
    PP_TRY(current_workspace(&w));
    cudaStream_t st = (cudaStream_t)stream;
    if (precision == PP_F32)
        return launch_density_f32((const float*)pos, (const float*)mass, N, x0, y0, cell, nx, ny, sigma, w->sm_count,
                                  st);
    return launch_density_f64((const double*)pos, (const double*)mass, N, x0, y0, cell, nx, ny, sigma, w->sm_count,
                              st);
}

int pp_invariants(const void* pos, const void* vel, const void* mass, const void* pot, int64_t N, double G,
                  double delta, int precision, double* out16, void* stream) {
    NvtxRange nvtx_range("pp_invariants");
    PP_TRY(check_common("pp_invariants", N, G, delta, precision));
    PP_TRY(check_ptr("pp_invariants", "pos", pos, precision, true));
    PP_TRY(check_ptr("pp_invariants", "vel", vel, precision, true));
    PP_TRY(check_ptr("pp_invariants", "mass", mass, precision, true));
    PP_TRY(check_ptr("pp_invariants", "pot", pot, precision, false));
    PP_TRY(check_ptr("pp_invariants", "out16", out16, PP_F64, true));
    std::lock_guard<std::mutex> lk(g_mu);
    Workspace* w = nullptr;
    PP_TRY(current_workspace(&w));
    cudaStream_t st = (cudaStream_t)stream;
    PP_TRY(enter(w, st));
    void* scratch;
    PP_TRY(ensure(w, B_INV, sizeof(double) * (size_t)invariants_scratch_doubles(N), &scratch));
    const double* pot64 = nullptr;
    if (!pot) {   // O(N^2) potential pass in FP64 with double-double partial sums, on the promoted state
        const Plan plan = make_plan(N, PP_F64, MODE_POT, w->sm_count, g_cfg_split.load(), forced_class());
        void *packed, *partial, *p64, *tm;
        PP_TRY(ensure(w, B_PACKED, (size_t)plan.n_pad * 32, &packed));
        PP_TRY(ensure(w, B_PARTIAL, (size_t)plan.split * (size_t)plan.part_stride * 32, &partial));
        PP_TRY(ensure(w, B_POT64, sizeof(double) * (size_t)N, &p64));
        PP_TRY(ensure(w, B_TILE_MASS, (size_t)plan.n_tiles * sizeof(double), &tm));
        const int em = (int)g_cfg_equal_mass.load();
        if (precision == PP_F32) {
            PP_TRY(launch_tile_mass_f32_to_f64((const float*)mass, (double*)tm, N, plan.tile_j, plan.n_tiles, em, st));
            PP_TRY(launch_pack_f32_to_f64((const float*)pos, (const float*)mass, (double*)packed, N, plan.n_pad, st));
        } else {
            PP_TRY(launch_tile_mass_f64((const double*)mass, (double*)tm, N, plan.tile_j, plan.n_tiles, em, st));
            PP_TRY(launch_pack_f64((const double*)pos, (const double*)mass, (double*)packed, N, plan.n_pad, st));
        }
        PP_TRY(sweep(plan, PP_F64, packed, tm, partial, N, delta, MODE_POT, st));
        PP_TRY(launch_finalize_f64((const double4*)partial, plan.split, plan.part_stride, N, G, nullptr, (double*)p64,
                                   nullptr, 0.0, 1, st));
        pot64 = (const double*)p64;
    }
    if (precision == PP_F32)
        PP_TRY(launch_invariants_f32((const float*)pos, (const float*)vel, (const float*)mass, (const float*)pot,
                                     pot64, N, (double*)scratch, out16, st));
    else
        PP_TRY(launch_invariants_f64((const double*)pos, (const double*)vel, (const double*)mass, (const double*)pot,
                                     pot64, N, (double*)scratch, out16, st));
    return leave(w, st);
}

}  // extern "C"
