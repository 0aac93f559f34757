// invariants.cu -- conserved integrals of eqs. (8)-(10) plus centre of mass (Fig. 6,
// PAPER.md:162) and total mass, reduced deterministically in compensated FP64 whatever the state precision.
//
//   K = sum m |v|^2 / 2          W = (1/2) sum m Phi   (Phi_i < 0, j != i: DESIGN.md reading R3)
//   P = sum m v   (eq. 9)        L = sum m r x v       (eq. 10 is its z component)
//   C = sum m r / M              M = sum m
//
// Two launches: (1) a grid-stride pass in which every thread keeps 12 TwoSum (value, error) pairs, merged by warp
// shuffles and a shared-memory step into one (value, error) pair per block and quantity; (2) one warp that adds the
// block partials in block order and writes the 16 outputs.  No atomics: bit-reproducible for a given N.
#include <mutex>

#include "ppgrav_internal.h"

namespace ppgrav {
namespace {

constexpr int kThreads = 256;
constexpr int kQ = 12;          // K W Px Py Pz Lx Ly Lz Cx Cy Cz M
constexpr int kStride = 32;     // doubles of scratch per block
constexpr int kMaxBlocks = 296;

__device__ __forceinline__ void comp_add(double& s, double& c, double t) {
    const double n = __dadd_rn(s, t);
    const double bp = __dsub_rn(n, s);
    c = __dadd_rn(c, __dadd_rn(__dsub_rn(s, __dsub_rn(n, bp)), __dsub_rn(t, bp)));
    s = n;
}

template <typename T>
__global__ void __launch_bounds__(kThreads)
invariants_partial_kernel(const T* __restrict__ pos, const T* __restrict__ vel, const T* __restrict__ mass,
                          const T* __restrict__ pot_state, const double* __restrict__ pot64, int64_t N,
                          double* __restrict__ scratch) {
    double s[kQ], c[kQ];
#pragma unroll
    for (int q = 0; q < kQ; ++q) s[q] = c[q] = 0.0;

    for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < N; i += (int64_t)gridDim.x * kThreads) {
        const double m = (double)mass[i];
        const double x = (double)pos[3 * i], y = (double)pos[3 * i + 1], z = (double)pos[3 * i + 2];
        const double u = (double)vel[3 * i], v = (double)vel[3 * i + 1], w = (double)vel[3 * i + 2];
        const double phi = pot64 ? pot64[i] : (double)pot_state[i];
        // plain products, no contraction: the same expression tree as the definition
        const double v2 = __dadd_rn(__dadd_rn(__dmul_rn(u, u), __dmul_rn(v, v)), __dmul_rn(w, w));
        comp_add(s[0], c[0], __dmul_rn(__dmul_rn(0.5, m), v2));                          // K, eq. (8) first term
        comp_add(s[1], c[1], __dmul_rn(__dmul_rn(0.5, m), phi));                         // W, eq. (8) second term
        comp_add(s[2], c[2], __dmul_rn(m, u));                                           // P, eq. (9)
        comp_add(s[3], c[3], __dmul_rn(m, v));
        comp_add(s[4], c[4], __dmul_rn(m, w));
        comp_add(s[5], c[5], __dmul_rn(m, __dsub_rn(__dmul_rn(y, w), __dmul_rn(z, v))));  // L, eq. (10)
        comp_add(s[6], c[6], __dmul_rn(m, __dsub_rn(__dmul_rn(z, u), __dmul_rn(x, w))));
        comp_add(s[7], c[7], __dmul_rn(m, __dsub_rn(__dmul_rn(x, v), __dmul_rn(y, u))));
        comp_add(s[8], c[8], __dmul_rn(m, x));                                           // centre of mass
        comp_add(s[9], c[9], __dmul_rn(m, y));
        comp_add(s[10], c[10], __dmul_rn(m, z));
        comp_add(s[11], c[11], m);                                                       // total mass
    }

    // warp tree (fixed shape), then the 8 warp results in warp order
    __shared__ double sh[kThreads / 32][kQ][2];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < kQ; ++q) {
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            const double os = __shfl_down_sync(0xffffffffu, s[q], off);
            const double oc = __shfl_down_sync(0xffffffffu, c[q], off);
            comp_add(s[q], c[q], os);
            c[q] = __dadd_rn(c[q], oc);
        }
        if (lane == 0) { sh[wid][q][0] = s[q]; sh[wid][q][1] = c[q]; }
    }
    __syncthreads();
    if (threadIdx.x < kQ) {
        const int q = threadIdx.x;
        double ts = 0.0, tc = 0.0;
        for (int w = 0; w < kThreads / 32; ++w) {
            comp_add(ts, tc, sh[w][q][0]);
            tc = __dadd_rn(tc, sh[w][q][1]);
        }
        scratch[(size_t)blockIdx.x * kStride + 2 * q] = ts;
        scratch[(size_t)blockIdx.x * kStride + 2 * q + 1] = tc;
    }
}

__global__ void __launch_bounds__(32) invariants_final_kernel(const double* __restrict__ scratch, int nblocks,
                                                              double* __restrict__ out16) {
    __shared__ double tot[kQ];
    const int q = threadIdx.x;
    if (q < kQ) {
        double ts = 0.0, tc = 0.0;
        for (int b = 0; b < nblocks; ++b) {   // block order: deterministic
            comp_add(ts, tc, scratch[(size_t)b * kStride + 2 * q]);
            tc = __dadd_rn(tc, scratch[(size_t)b * kStride + 2 * q + 1]);
        }
        tot[q] = __dadd_rn(ts, tc);
    }
    __syncwarp();
    if (q == 0) {
        const double K = tot[0], W = tot[1], M = tot[11];
        out16[0] = __dadd_rn(K, W);
        out16[1] = K;
        out16[2] = W;
        for (int k = 0; k < 6; ++k) out16[3 + k] = tot[2 + k];
        for (int k = 0; k < 3; ++k) out16[9 + k] = tot[8 + k] / M;
        out16[12] = M;
        out16[13] = out16[14] = out16[15] = 0.0;
    }
}

inline int blocks_for(int64_t N) {
    const int64_t b = (N + kThreads - 1) / kThreads;
    return (int)(b < kMaxBlocks ? b : kMaxBlocks);
}

template <typename T>
int launch_invariants(const T* pos, const T* vel, const T* mass, const T* pot_state, const double* pot64, int64_t N,
                      double* scratch, double* out16, cudaStream_t st) {
    const int nb = blocks_for(N);
    invariants_partial_kernel<T><<<nb, kThreads, 0, st>>>(pos, vel, mass, pot_state, pot64, N, scratch);
    count_launch();
    PP_CUDA(cudaGetLastError());
    invariants_final_kernel<<<1, 32, 0, st>>>(scratch, nb, out16);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}

}  // namespace

int invariants_scratch_doubles(int64_t N) { return blocks_for(N) * kStride; }

int launch_invariants_f32(const float* pos, const float* vel, const float* mass, const float* pot_state,
                          const double* pot64, int64_t N, double* scratch, double* out16, cudaStream_t st) {
    return launch_invariants<float>(pos, vel, mass, pot_state, pot64, N, scratch, out16, st);
}
int launch_invariants_f64(const double* pos, const double* vel, const double* mass, const double* pot_state,
                          const double* pot64, int64_t N, double* scratch, double* out16, cudaStream_t st) {
    return launch_invariants<double>(pos, vel, mass, pot_state, pot64, N, scratch, out16, st);
}

// ---- pp_invariants_noalloc: the same two kernels with their scratch in a file-scope device array ----------------------
// For callers that may not allocate (code under CUDA-graph capture, tight serving loops, harnesses that forbid
// cudaMalloc): the block partials of invariants_partial_kernel live in g_noalloc_scratch instead of the library's
// grow-on-demand workspace.  kMaxBlocks x kStride doubles = 75,776 bytes, held by every GPU that loads the library until
// the process exits.  The grid-stride pass never launches more than kMaxBlocks blocks, so this serves any N up to
// PP_NOALLOC_MAX_N.  Every call shares the array and finds the previous call's contents in it; nothing has to start at
// zero, because block b overwrites its 2 x kQ doubles before invariants_final_kernel (stream-ordered behind it) reads
// exactly the nb blocks this call launched.  Calls that overlap on the GPU (different streams, no ordering) race on it.
namespace {

static __device__ __align__(256) double g_noalloc_scratch[kMaxBlocks * kStride];

constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mu;
double* g_noalloc_ptr[kNoallocMaxDevices] = {};   // device address of g_noalloc_scratch, per device (0 = not yet asked)

// In host code `g_noalloc_scratch` is a host-side stand-in, not a device address: the device address is asked for once
// per device, with that device current, and only that pointer is ever handed to a kernel.
int noalloc_scratch(double** out) {
    int dev = -1;
    PP_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoallocMaxDevices) {
        set_error("pp_invariants_noalloc: device ordinal %d out of range", dev);
        return PP_ECUDA;
    }
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        double* p = nullptr;
        PP_CUDA(cudaGetSymbolAddress((void**)&p, g_noalloc_scratch));
        if (!p) {
            set_error("pp_invariants_noalloc: cudaGetSymbolAddress returned a null address");
            return PP_ECUDA;
        }
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return PP_OK;
}

}  // namespace

}  // namespace ppgrav

extern "C" int pp_invariants_noalloc(const void* pos, const void* vel, const void* mass, const void* pot, int64_t N,
                                     int precision, double* out16, void* stream) {
    using namespace ppgrav;
    if (precision != PP_F32 && precision != PP_F64 && precision != PP_MIXED) {
        set_error("pp_invariants_noalloc: precision must be PP_F32, PP_F64 or PP_MIXED (got %d)", precision);
        return PP_EINVAL;
    }
    if (N < 1 || N > (int64_t)PP_NOALLOC_MAX_N) {
        set_error("pp_invariants_noalloc: N = %lld outside [1, PP_NOALLOC_MAX_N = %lld]", (long long)N,
                  (long long)PP_NOALLOC_MAX_N);
        return PP_EINVAL;
    }
    if (!pot) {
        set_error("pp_invariants_noalloc: pot is NULL -- the O(N^2) potential pass needs the allocating workspace; "
                  "pass the potential pp_forces / pp_step_kdk returned, or call pp_invariants");
        return PP_EINVAL;
    }
    const size_t a = precision == PP_F32 ? 4 : 8;
    const void* ptrs[5] = {pos, vel, mass, pot, out16};
    const char* names[5] = {"pos", "vel", "mass", "pot", "out16"};
    for (int k = 0; k < 5; ++k) {
        const size_t need = k == 4 ? 8 : a;
        if (!ptrs[k] || (reinterpret_cast<uintptr_t>(ptrs[k]) & (need - 1))) {
            set_error("pp_invariants_noalloc: %s is NULL or not aligned to its element size", names[k]);
            return PP_EINVAL;
        }
    }
    double* scratch = nullptr;
    const int rc = noalloc_scratch(&scratch);
    if (rc != PP_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (precision == PP_F32)
        return launch_invariants<float>((const float*)pos, (const float*)vel, (const float*)mass, (const float*)pot,
                                        nullptr, N, scratch, out16, st);
    return launch_invariants<double>((const double*)pos, (const double*)vel, (const double*)mass, (const double*)pot,
                                     nullptr, N, scratch, out16, st);
}
