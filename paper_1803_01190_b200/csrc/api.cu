// api.cu -- the C ABI of libppgrav (include/ppgrav.h): argument checking, the per-device workspace, and the
// sequencing of the kernels.  No arithmetic of the method lives here.
//
//   pp_forces     = pack -> force sweep over (i-block, j-split) units -> finalize
//   pp_step_kdk   = [initial solve] -> nsteps x { kick+drift+pack -> force sweep -> finalize+kick }
//   pp_invariants = [FP64 potential sweep -> finalize] -> block partials -> final sum
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <utility>
#include <vector>

#include "ppgrav_internal.h"

namespace ppgrav {

namespace {

thread_local char t_err[512] = "";
std::atomic<int64_t> g_launches{0};
std::atomic<int64_t> g_cfg_split{0};
std::atomic<int64_t> g_cfg_graph{1};
std::atomic<int64_t> g_cfg_profile{0};
std::atomic<int64_t> g_cfg_equal_mass{1};
std::vector<std::pair<cudaEvent_t, cudaEvent_t>> g_prof;   // guarded by g_mu (every sweep is launched under it)

constexpr int kMaxDevices = 64;
constexpr int64_t kMaxN = (int64_t)1 << 28;
constexpr int kNumBuf = 5;
enum { B_PACKED = 0, B_PARTIAL, B_INV, B_POT64, B_TILE_MASS };

struct Workspace {
    void* buf[kNumBuf] = {};
    size_t cap[kNumBuf] = {};
    int sm_count = 0;
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
          double delta, int mode, cudaStream_t st) {
    const bool prof = g_cfg_profile.load() != 0;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (prof) {
        PP_CUDA(cudaEventCreate(&e0));
        PP_CUDA(cudaEventCreate(&e1));
        PP_CUDA(cudaEventRecord(e0, st));
    }
    const int rc = sweep_precision(precision) == PP_F32
                       ? launch_force_f32(p, (const float*)packed, (const float*)tile_mass, (float4*)partial, N, delta,
                                          mode, st)
                       : launch_force_f64(p, (const double*)packed, (const double*)tile_mass, (double4*)partial, N,
                                          delta, mode, st);
    if (prof) {
        PP_CUDA(cudaEventRecord(e1, st));
        g_prof.emplace_back(e0, e1);
    }
    return rc;
}

// one gravity solve on already packed bodies: sweep + finalize (optionally with the closing half-kick)
// (acc, pot, vel address the p.i_count bodies of the plan's i-range)
int solve_packed(const Plan& p, int precision, const void* packed, const void* tile_mass, void* partial, int64_t N,
                 double G, double delta, void* acc, void* pot, void* vel, double kick, cudaStream_t st) {
    const int mode = pot ? MODE_FORCE_POT : MODE_FORCE;
    PP_TRY(sweep(p, precision, packed, tile_mass, partial, N, delta, mode, st));
    if (precision == PP_F32)
        return launch_finalize_f32((const float4*)partial, p.split, p.part_stride, p.i_count, G, (float*)acc,
                                   (float*)pot, (float*)vel, kick, st);
    if (precision == PP_MIXED)
        return launch_finalize_mixed((const float4*)partial, p.split, p.part_stride, p.i_count, G, (double*)acc,
                                     (double*)pot, (double*)vel, kick, st);
    return launch_finalize_f64((const double4*)partial, p.split, p.part_stride, p.i_count, G, (double*)acc,
                               (double*)pot, (double*)vel, kick, 0, st);
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

int prepare_solve(Workspace* w, int64_t N, int precision, Plan* plan, void** packed, void** partial,
                  int64_t i_begin = 0, int64_t i_count = -1) {
    *plan = make_plan(N, sweep_precision(precision), w->sm_count, g_cfg_split.load(), i_begin, i_count);
    const size_t body = 4 * sweep_elem_bytes(precision);
    PP_TRY(ensure(w, B_PACKED, (size_t)plan->n_pad * body, packed));
    PP_TRY(ensure(w, B_PARTIAL, (size_t)plan->split * (size_t)plan->part_stride * body, partial));
    return PP_OK;
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
        bool any = false;
        for (int b = 0; b < kNumBuf; ++b) any = any || w.buf[b];
        if (!any) continue;
        PP_CUDA(cudaSetDevice(d));
        PP_CUDA(cudaDeviceSynchronize());
        for (int b = 0; b < kNumBuf; ++b) {
            if (w.buf[b]) cudaFree(w.buf[b]);
            w.buf[b] = nullptr;
            w.cap[b] = 0;
        }
    }
    PP_CUDA(cudaSetDevice(prev));
    return PP_OK;
}

int pp_plan_query(int64_t N, int precision, int with_pot, int64_t* out8) {
    if (!out8) { set_error("pp_plan_query: out8 is NULL"); return PP_EINVAL; }
    PP_TRY(check_common("pp_plan_query", N, 1.0, 0.0, precision));
    int sm = 148;   // B200; used when no device is present (host-side planning only)
    int dev = -1;
    if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) sm = v;
    }
    cudaGetLastError();
    precision = sweep_precision(precision);
    const Plan p = make_plan(N, precision, sm, g_cfg_split.load());
    out8[0] = p.i_per_cta;
    out8[1] = p.tile_j;
    out8[2] = p.split;
    out8[3] = (int64_t)p.n_iblocks * p.split;
    out8[4] = p.ctas_per_sm;
    out8[5] = sm;
    out8[6] = precision == PP_F32 ? (with_pot ? 13 : 12) : (with_pot ? 18 : 16);
    out8[7] = 1;
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
    const Plan plan = make_plan(N, sweep_precision(precision), w->sm_count, g_cfg_split.load());
    void* tm;
    PP_TRY(tile_masses(w, plan, precision, mass, N, 1, &tm, st));
    const size_t eb = sweep_elem_bytes(precision);
    std::vector<unsigned char> host((size_t)plan.n_tiles * eb);
    PP_CUDA(cudaMemcpyAsync(host.data(), tm, host.size(), cudaMemcpyDeviceToHost, st));
    PP_CUDA(cudaStreamSynchronize(st));
    int64_t common = 0;
    for (int t = 0; t < plan.n_tiles; ++t) {
        if (eb == 4) { float v; std::memcpy(&v, &host[(size_t)t * 4], 4); common += (v == v); }
        else { double v; std::memcpy(&v, &host[(size_t)t * 8], 8); common += (v == v); }
    }
    out2[0] = plan.n_tiles;
    out2[1] = common;
    return PP_OK;
}

int pp_probe_pipe(int kind, int64_t iters, double* out4) {
    if (!out4) { set_error("pp_probe_pipe: out4 is NULL"); return PP_EINVAL; }
    Workspace* w = nullptr;
    PP_TRY(current_workspace(&w));
    return run_probe(kind, iters, w->sm_count, out4);
}

int pp_forces_range(const void* pos, const void* mass, void* acc, void* pot, int64_t N, int64_t i_begin,
                    int64_t i_count, double G, double delta, int precision, void* stream) {
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
    Plan plan;
    void *packed, *partial;
    PP_TRY(prepare_solve(w, N, precision, &plan, &packed, &partial, i_begin, i_count));
    void* tm;
    PP_TRY(tile_masses(w, plan, precision, mass, N, (int)g_cfg_equal_mass.load(), &tm, st));
    PP_TRY(pack_state(precision, pos, mass, packed, N, plan.n_pad, st));
    return solve_packed(plan, precision, packed, tm, partial, N, G, delta, acc, pot, nullptr, 0.0, st);
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
    Plan plan;
    void *packed, *partial;
    PP_TRY(prepare_solve(w, N, precision, &plan, &packed, &partial));
    if (nsteps == 0 && (flags & PP_ACC_VALID)) return PP_OK;   // nothing to solve
    void* tm;
    PP_TRY(tile_masses(w, plan, precision, mass, N, (int)g_cfg_equal_mass.load(), &tm, st));
    if (!(flags & PP_ACC_VALID)) {   // a(t0): the one extra gravity solve of a cold start
        PP_TRY(pack_state(precision, pos, mass, packed, N, plan.n_pad, st));
        PP_TRY(solve_packed(plan, precision, packed, tm, partial, N, G, delta, acc, nsteps == 0 ? pot : nullptr,
                            nullptr, 0.0, st));
    }
    if (nsteps == 0) return PP_OK;
    const double half = 0.5 * dt;
    // the last step is issued directly: it alone may carry the potential
    const int64_t nbody = nsteps - 1;

    // Small N is launch-bound (a solve of 2048 bodies is a few microseconds of pipe time): record one step into a
    // CUDA graph and replay it.  Needs a capturable (non-legacy) stream.
    const bool use_graph = g_cfg_graph.load() && !g_cfg_profile.load() && st != nullptr && st != cudaStreamLegacy && N <= 65536 && nbody >= 4;
    if (use_graph) {
        cudaGraph_t graph = nullptr;
        cudaGraphExec_t exec = nullptr;
        PP_CUDA(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
        int rc = kick_drift_pack(precision, pos, vel, acc, mass, packed, N, plan.n_pad, half, dt, st);
        if (rc == PP_OK)
            rc = solve_packed(plan, precision, packed, tm, partial, N, G, delta, acc, nullptr, vel, half, st);
        const cudaError_t ec = cudaStreamEndCapture(st, &graph);
        if (rc != PP_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (ec != cudaSuccess) return cuda_fail(ec, "cudaStreamEndCapture");
        const cudaError_t ei = cudaGraphInstantiate(&exec, graph, 0);
        if (ei != cudaSuccess) { cudaGraphDestroy(graph); return cuda_fail(ei, "cudaGraphInstantiate"); }
        count_launch(-3);   // the three captured launches were recorded, not run
        cudaError_t el = cudaSuccess;
        for (int64_t s = 0; s < nbody && el == cudaSuccess; ++s) {
            el = cudaGraphLaunch(exec, st);
            count_launch(3);
        }
        cudaGraphExecDestroy(exec);   // deferred by the runtime until the launches have drained
        cudaGraphDestroy(graph);
        if (el != cudaSuccess) return cuda_fail(el, "cudaGraphLaunch");
    } else {
        for (int64_t s = 0; s < nbody; ++s) {
            PP_TRY(kick_drift_pack(precision, pos, vel, acc, mass, packed, N, plan.n_pad, half, dt, st));
            PP_TRY(solve_packed(plan, precision, packed, tm, partial, N, G, delta, acc, nullptr, vel, half, st));
        }
    }
    PP_TRY(kick_drift_pack(precision, pos, vel, acc, mass, packed, N, plan.n_pad, half, dt, st));
    return solve_packed(plan, precision, packed, tm, partial, N, G, delta, acc, pot, vel, half, st);
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
    void* scratch;
    PP_TRY(ensure(w, B_INV, sizeof(double) * (size_t)invariants_scratch_doubles(N), &scratch));
    const double* pot64 = nullptr;
    if (!pot) {   // O(N^2) potential pass in FP64 with double-double partial sums, on the promoted state
        Plan plan;
        void *packed, *partial, *p64;
        PP_TRY(prepare_solve(w, N, PP_F64, &plan, &packed, &partial));
        PP_TRY(ensure(w, B_POT64, sizeof(double) * (size_t)N, &p64));
        if (precision == PP_F32)
            PP_TRY(launch_pack_f32_to_f64((const float*)pos, (const float*)mass, (double*)packed, N, plan.n_pad, st));
        else
            PP_TRY(launch_pack_f64((const double*)pos, (const double*)mass, (double*)packed, N, plan.n_pad, st));
        PP_TRY(sweep(plan, PP_F64, packed, nullptr, partial, N, delta, MODE_POT, st));
        PP_TRY(launch_finalize_f64((const double4*)partial, plan.split, plan.part_stride, N, G, nullptr, (double*)p64,
                                   nullptr, 0.0, 1, st));
        pot64 = (const double*)p64;
    }
    if (precision == PP_F32)
        return launch_invariants_f32((const float*)pos, (const float*)vel, (const float*)mass, (const float*)pot,
                                     pot64, N, (double*)scratch, out16, st);
    return launch_invariants_f64((const double*)pos, (const double*)vel, (const double*)mass, (const double*)pot,
                                 pot64, N, (double*)scratch, out16, st);
}

}  // extern "C"
