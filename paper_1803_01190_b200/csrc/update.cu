// update.cu -- the O(N) kernels around the gravity solve: packing, split-j finalize, and the paper's "Update
// System" kernel in half-kick form (eqs. (5)-(7); reading R4).
//
// All of them are HBM-bound element-wise passes (<= 200 B per body per step against >= N x 12 pipe operations per
// body in the force kernel), so they are written for coalescing and fusion, not for arithmetic:
//   pack            pos[N,3], mass[N] -> packed tile layout (float pairs interleaved / double4), padding included
//   finalize        acc = G sum_s partial[s] (fixed order, compensated) [, pot = -G sum_s] [, vel += kick acc]
//   kick_drift_pack vel += kick acc; pos += dt vel; packed = pack(pos, mass)   -- one pass instead of three
//   finalize_kick_drift_pack  the two above back to back, for the interior steps of a pp_step_kdk call
#include "ppgrav_internal.h"

namespace ppgrav {
namespace {

constexpr int kThreads = 256;

inline int grid_for(int64_t n) { return (int)((n + kThreads - 1) / kThreads); }

// FP32 packed layout: body i lives in pair i>>1, lane i&1 of {x0 x1 y0 y1 z0 z1 m0 m1}
__device__ __forceinline__ void store_packed(float* packed, int64_t i, float x, float y, float z, float m) {
    float* q = packed + (i >> 1) * 8 + (i & 1);
    q[0] = x; q[2] = y; q[4] = z; q[6] = m;
}
__device__ __forceinline__ void store_packed(double* packed, int64_t i, double x, double y, double z, double m) {
    reinterpret_cast<double4*>(packed)[i] = make_double4(x, y, z, m);
}

template <typename TIn, typename TOut>
__global__ void __launch_bounds__(kThreads) pack_kernel(const TIn* __restrict__ pos, const TIn* __restrict__ mass,
                                                        TOut* __restrict__ packed, int64_t N, int64_t n_pad) {
    const int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (i >= n_pad) return;
    if (i < N)
        store_packed(packed, i, (TOut)pos[3 * i], (TOut)pos[3 * i + 1], (TOut)pos[3 * i + 2], (TOut)mass[i]);
    else
        store_packed(packed, i, (TOut)0, (TOut)0, (TOut)0, (TOut)0);   // padding: massless, contributes nothing
}

// tile_mass[t] = m if all tile_j bodies of j-tile t have the same mass m in the sweep's precision (bodies >= N are
// padding of mass 0), NaN otherwise.  One warp per tile.  The sweeps (force_f32.cu / force_f64.cu) take m_j out of
// the pair loop on tiles that have a common mass.  enable == 0 writes NaN everywhere (PP_CFG_EQUAL_MASS off).
template <typename TIn, typename TOut>
__global__ void __launch_bounds__(kThreads) tile_mass_kernel(const TIn* __restrict__ mass, TOut* __restrict__ tile_mass,
                                                             int64_t N, int tile_j, int n_tiles, int enable) {
    const int t = (int)(((int64_t)blockIdx.x * kThreads + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (t >= n_tiles) return;                                  // whole warps leave together
    const int64_t j0 = (int64_t)t * tile_j;
    const TOut first = j0 < N ? (TOut)mass[j0] : (TOut)0;     // tiles wholly inside the padding have the common mass 0
    bool same = enable != 0;
    for (int j = lane; j < tile_j; j += 32) {
        const TOut m = (j0 + j < N) ? (TOut)mass[j0 + j] : (TOut)0;
        same = same && (m == first);
    }
    same = __all_sync(0xffffffffu, same);
    if (lane == 0) tile_mass[t] = same ? first : (TOut)NAN;
}

// error-free s + t -> (s, err accumulated into c); intrinsics keep the compiler from contracting/reassociating
__device__ __forceinline__ void comp_add(float& s, float& c, float t) {
    const float n = __fadd_rn(s, t);
    const float bp = __fsub_rn(n, s);
    c = __fadd_rn(c, __fadd_rn(__fsub_rn(s, __fsub_rn(n, bp)), __fsub_rn(t, bp)));
    s = n;
}
__device__ __forceinline__ void comp_add(double& s, double& c, double t) {
    const double n = __dadd_rn(s, t);
    const double bp = __dsub_rn(n, s);
    c = __dadd_rn(c, __dadd_rn(__dsub_rn(s, __dsub_rn(n, bp)), __dsub_rn(t, bp)));
    s = n;
}

template <typename T> struct Vec4;
template <> struct Vec4<float> { using type = float4; };
template <> struct Vec4<double> { using type = double4; };

// POT_DD: partial.x/.y are the hi/lo words of a double-double potential sum (MODE_POT of force_f64.cu)
// TP: scalar type of the partial sums (the sweep's precision); T: scalar type of the state (acc, pot, vel).  They
// differ only in PP_MIXED (FP32 sweep, FP64 state), where the S partial sums are added and scaled in FP64.
template <typename TP, typename T, bool POT_DD>
__global__ void __launch_bounds__(kThreads)
finalize_kernel(const typename Vec4<TP>::type* __restrict__ partial, int split, int64_t n_pad, int64_t N, T G,
                T* __restrict__ acc, T* __restrict__ pot, T* __restrict__ vel, T kick,
                const typename Vec4<TP>::type* __restrict__ partial_j, int jrows, int64_t jstride) {
    const int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (i >= N) return;
    T sx = 0, sy = 0, sz = 0, sw = 0, cx = 0, cy = 0, cz = 0, cw = 0;
    for (int s = 0; s < split; ++s) {   // fixed order s = 0..S-1: run-to-run deterministic
        const typename Vec4<TP>::type v = partial[(size_t)s * n_pad + i];
        if (POT_DD) {
            comp_add(sx, cx, (T)v.x);
            comp_add(sx, cx, (T)v.y);
        } else {
            comp_add(sx, cx, (T)v.x);
            comp_add(sy, cy, (T)v.y);
            comp_add(sz, cz, (T)v.z);
            comp_add(sw, cw, (T)v.w);
        }
    }
    // symmetric sweep (force_sym_*.cu): what the blocks I - d, d = 1..jrows, gathered for body i, in fixed order d
    for (int d = 0; d < jrows; ++d) {
        const typename Vec4<TP>::type v = partial_j[(size_t)d * jstride + i];
        comp_add(sx, cx, (T)v.x);
        comp_add(sy, cy, (T)v.y);
        comp_add(sz, cz, (T)v.z);
        comp_add(sw, cw, (T)v.w);
    }
    if (POT_DD) {
        if (pot) pot[i] = -G * (sx + cx);
        return;
    }
    const T ax = G * (sx + cx), ay = G * (sy + cy), az = G * (sz + cz);
    if (acc) { acc[3 * i] = ax; acc[3 * i + 1] = ay; acc[3 * i + 2] = az; }
    if (pot) pot[i] = -G * (sw + cw);
    if (vel) {   // closing half-kick of eq. (7): v(t+dt) = v~ + dt/2 a(t+dt)
        vel[3 * i] = fma(kick, ax, vel[3 * i]);
        vel[3 * i + 1] = fma(kick, ay, vel[3 * i + 1]);
        vel[3 * i + 2] = fma(kick, az, vel[3 * i + 2]);
    }
}

// Symmetric sweep in bands (force_sym_*.cu): acc_j[0][i] + acc_j[1][i] (TwoSum value and error) += sum_r rows[r][i],
// in row order -- the j-side sums of one band of partner offsets, so that the rows can be reused by the next band.
template <typename T4, typename T>
__global__ void __launch_bounds__(kThreads)
fold_rows_kernel(const T4* __restrict__ rows, int nrows, int64_t stride, T4* __restrict__ acc_j, int first) {
    const int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (i >= stride) return;
    T4 s, c;
    if (first) { s.x = s.y = s.z = s.w = 0; c = s; }
    else { s = acc_j[i]; c = acc_j[stride + i]; }
    for (int r = 0; r < nrows; ++r) {
        const T4 v = rows[(size_t)r * stride + i];
        comp_add(s.x, c.x, v.x);
        comp_add(s.y, c.y, v.y);
        comp_add(s.z, c.z, v.z);
        comp_add(s.w, c.w, v.w);
    }
    acc_j[i] = s;
    acc_j[stride + i] = c;
}

// TK: scalar type of the packed copy (the sweep's precision; float for a double state in PP_MIXED)
template <typename T, typename TK>
__global__ void __launch_bounds__(kThreads)
kick_drift_pack_kernel(T* __restrict__ pos, T* __restrict__ vel, const T* __restrict__ acc,
                       const T* __restrict__ mass, TK* __restrict__ packed, int64_t N, int64_t n_pad, T kick, T dt) {
    const int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (i >= n_pad) return;
    if (i >= N) { store_packed(packed, i, (TK)0, (TK)0, (TK)0, (TK)0); return; }
    T r[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T v = fma(kick, acc[3 * i + c], vel[3 * i + c]);   // opening half-kick, eq. (5) halved
        vel[3 * i + c] = v;
        r[c] = fma(dt, v, pos[3 * i + c]);                       // drift, eq. (6)
        pos[3 * i + c] = r[c];
    }
    store_packed(packed, i, (TK)r[0], (TK)r[1], (TK)r[2], (TK)mass[i]);
}

// Between two gravity solves of one pp_step_kdk call the closing half-kick of step n (eq. (7)), the opening half-kick
// and drift of step n+1 (eqs. (5)-(6)) and the re-packing all touch the same body: one pass instead of two launches
// (finalize+kick, then kick+drift+pack).  The arithmetic is the same sequence of roundings as the two separate
// kernels -- acc = G sum_s partial; v = fma(kick, acc, v); v = fma(kick, acc, v); r = fma(dt, v, r) -- so a run is
// bit-identical whichever way the steps are issued.  Padding bodies (>= N) of `packed` are not touched: they were
// written by the pass that opened the call and never change.
template <typename TP, typename T, typename TK>
__global__ void __launch_bounds__(kThreads)
finalize_kick_drift_pack_kernel(const typename Vec4<TP>::type* __restrict__ partial, int split, int64_t part_stride,
                                int64_t N, T G, T* __restrict__ acc, T* __restrict__ vel, T* __restrict__ pos,
                                const T* __restrict__ mass, TK* __restrict__ packed, T kick, T dt,
                                const typename Vec4<TP>::type* __restrict__ partial_j, int jrows, int64_t jstride) {
    const int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (i >= N) return;
    T sx = 0, sy = 0, sz = 0, cx = 0, cy = 0, cz = 0;
    for (int s = 0; s < split; ++s) {   // fixed order s = 0..S-1: run-to-run deterministic
        const typename Vec4<TP>::type v = partial[(size_t)s * part_stride + i];
        comp_add(sx, cx, (T)v.x);
        comp_add(sy, cy, (T)v.y);
        comp_add(sz, cz, (T)v.z);
    }
    for (int d = 0; d < jrows; ++d) {   // j-side rows of the symmetric sweep, fixed order
        const typename Vec4<TP>::type v = partial_j[(size_t)d * jstride + i];
        comp_add(sx, cx, (T)v.x);
        comp_add(sy, cy, (T)v.y);
        comp_add(sz, cz, (T)v.z);
    }
    const T a[3] = {G * (sx + cx), G * (sy + cy), G * (sz + cz)};
    T r[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        acc[3 * i + c] = a[c];
        T v = fma(kick, a[c], vel[3 * i + c]);    // closing half-kick of this step, eq. (7)
        v = fma(kick, a[c], v);                   // opening half-kick of the next step, eq. (5) halved
        vel[3 * i + c] = v;
        r[c] = fma(dt, v, pos[3 * i + c]);        // drift, eq. (6)
        pos[3 * i + c] = r[c];
    }
    store_packed(packed, i, (TK)r[0], (TK)r[1], (TK)r[2], (TK)mass[i]);
}

// the sharded step's own-bodies update: opening half-kick + drift (dt != 0) or closing half-kick alone (dt == 0);
// the same two fused multiply-adds per component as kick_drift_pack_kernel, so a sharded run rounds identically
template <typename T>
__global__ void __launch_bounds__(kThreads)
kick_drift_kernel(T* __restrict__ pos, T* __restrict__ vel, const T* __restrict__ acc, int64_t n, T kick, T dt,
                  bool drift) {
    const int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x;
    if (i >= n) return;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T v = fma(kick, acc[3 * i + c], vel[3 * i + c]);
        vel[3 * i + c] = v;
        if (drift) pos[3 * i + c] = fma(dt, v, pos[3 * i + c]);
    }
}

}  // namespace

int launch_fold_rows(const float4* rows, int nrows, int64_t stride, float4* acc_j, bool first, cudaStream_t st) {
    fold_rows_kernel<float4, float><<<grid_for(stride), kThreads, 0, st>>>(rows, nrows, stride, acc_j, first ? 1 : 0);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}
int launch_fold_rows(const double4* rows, int nrows, int64_t stride, double4* acc_j, bool first, cudaStream_t st) {
    fold_rows_kernel<double4, double><<<grid_for(stride), kThreads, 0, st>>>(rows, nrows, stride, acc_j, first ? 1 : 0);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}

int launch_kick_drift_f32(float* pos, float* vel, const float* acc, int64_t n, double kick, double dt,
                          cudaStream_t st) {
    kick_drift_kernel<float><<<grid_for(n), kThreads, 0, st>>>(pos, vel, acc, n, (float)kick, (float)dt, dt != 0.0);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}
int launch_kick_drift_f64(double* pos, double* vel, const double* acc, int64_t n, double kick, double dt,
                          cudaStream_t st) {
    kick_drift_kernel<double><<<grid_for(n), kThreads, 0, st>>>(pos, vel, acc, n, kick, dt, dt != 0.0);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}

int launch_pack_f32(const float* pos, const float* mass, float* packed, int64_t N, int64_t n_pad, cudaStream_t st) {
    pack_kernel<float, float><<<grid_for(n_pad), kThreads, 0, st>>>(pos, mass, packed, N, n_pad);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}
int launch_pack_f64(const double* pos, const double* mass, double* packed, int64_t N, int64_t n_pad,
                    cudaStream_t st) {
    pack_kernel<double, double><<<grid_for(n_pad), kThreads, 0, st>>>(pos, mass, packed, N, n_pad);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}
int launch_pack_f32_to_f64(const float* pos, const float* mass, double* packed, int64_t N, int64_t n_pad,
                           cudaStream_t st) {
    pack_kernel<float, double><<<grid_for(n_pad), kThreads, 0, st>>>(pos, mass, packed, N, n_pad);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}

int launch_finalize_f32(const float4* partial, int split, int64_t n_pad, int64_t N, double G, float* acc, float* pot,
                        float* vel, double kick, cudaStream_t st, const float4* partial_j, int jrows, int64_t jstride) {
    finalize_kernel<float, float, false><<<grid_for(N), kThreads, 0, st>>>(partial, split, n_pad, N, (float)G, acc,
                                                                           pot, kick != 0.0 ? vel : nullptr,
                                                                           (float)kick, partial_j, jrows, jstride);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}
int launch_finalize_mixed(const float4* partial, int split, int64_t n_pad, int64_t N, double G, double* acc,
                          double* pot, double* vel, double kick, cudaStream_t st, const float4* partial_j, int jrows,
                          int64_t jstride) {
    finalize_kernel<float, double, false><<<grid_for(N), kThreads, 0, st>>>(partial, split, n_pad, N, G, acc, pot,
                                                                            kick != 0.0 ? vel : nullptr, kick,
                                                                            partial_j, jrows, jstride);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}
int launch_finalize_f64(const double4* partial, int split, int64_t n_pad, int64_t N, double G, double* acc,
                        double* pot, double* vel, double kick, int pot_is_dd, cudaStream_t st, const double4* partial_j,
                        int jrows, int64_t jstride) {
    if (pot_is_dd)
        finalize_kernel<double, double, true><<<grid_for(N), kThreads, 0, st>>>(partial, split, n_pad, N, G, nullptr, pot,
                                                                        nullptr, 0.0, nullptr, 0, 0);
    else
        finalize_kernel<double, double, false><<<grid_for(N), kThreads, 0, st>>>(partial, split, n_pad, N, G, acc, pot,
                                                                         kick != 0.0 ? vel : nullptr, kick,
                                                                         partial_j, jrows, jstride);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}

int launch_kick_drift_pack_f32(float* pos, float* vel, const float* acc, const float* mass, float* packed, int64_t N,
                               int64_t n_pad, double kick, double dt, cudaStream_t st) {
    kick_drift_pack_kernel<float, float><<<grid_for(n_pad), kThreads, 0, st>>>(pos, vel, acc, mass, packed, N, n_pad,
                                                                        (float)kick, (float)dt);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}
int launch_kick_drift_pack_f64(double* pos, double* vel, const double* acc, const double* mass, double* packed,
                               int64_t N, int64_t n_pad, double kick, double dt, cudaStream_t st) {
    kick_drift_pack_kernel<double, double><<<grid_for(n_pad), kThreads, 0, st>>>(pos, vel, acc, mass, packed, N, n_pad,
                                                                                 kick, dt);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}
int launch_kick_drift_pack_mixed(double* pos, double* vel, const double* acc, const double* mass, float* packed,
                                 int64_t N, int64_t n_pad, double kick, double dt, cudaStream_t st) {
    kick_drift_pack_kernel<double, float><<<grid_for(n_pad), kThreads, 0, st>>>(pos, vel, acc, mass, packed, N, n_pad,
                                                                                kick, dt);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}
int launch_pack_f64_to_f32(const double* pos, const double* mass, float* packed, int64_t N, int64_t n_pad,
                           cudaStream_t st) {
    pack_kernel<double, float><<<grid_for(n_pad), kThreads, 0, st>>>(pos, mass, packed, N, n_pad);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}

int launch_finalize_kick_drift_pack_f32(const float4* partial, int split, int64_t part_stride, int64_t N, double G,
                                        float* acc, float* vel, float* pos, const float* mass, float* packed,
                                        double kick, double dt, cudaStream_t st, const float4* partial_j,
                                        int jrows, int64_t jstride) {
    finalize_kick_drift_pack_kernel<float, float, float><<<grid_for(N), kThreads, 0, st>>>(
        partial, split, part_stride, N, (float)G, acc, vel, pos, mass, packed, (float)kick, (float)dt, partial_j, jrows,
        jstride);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}
int launch_finalize_kick_drift_pack_f64(const double4* partial, int split, int64_t part_stride, int64_t N, double G,
                                        double* acc, double* vel, double* pos, const double* mass, double* packed,
                                        double kick, double dt, cudaStream_t st, const double4* partial_j,
                                        int jrows, int64_t jstride) {
    finalize_kick_drift_pack_kernel<double, double, double><<<grid_for(N), kThreads, 0, st>>>(
        partial, split, part_stride, N, G, acc, vel, pos, mass, packed, kick, dt, partial_j, jrows, jstride);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}
int launch_finalize_kick_drift_pack_mixed(const float4* partial, int split, int64_t part_stride, int64_t N, double G,
                                          double* acc, double* vel, double* pos, const double* mass, float* packed,
                                          double kick, double dt, cudaStream_t st, const float4* partial_j,
                                        int jrows, int64_t jstride) {
    finalize_kick_drift_pack_kernel<float, double, float><<<grid_for(N), kThreads, 0, st>>>(
        partial, split, part_stride, N, G, acc, vel, pos, mass, packed, kick, dt, partial_j, jrows, jstride);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}

template <typename TIn, typename TOut>
static int launch_tile_mass(const TIn* mass, TOut* tile_mass, int64_t N, int tile_j, int n_tiles, int enable,
                            cudaStream_t st) {
    tile_mass_kernel<TIn, TOut><<<grid_for((int64_t)n_tiles * 32), kThreads, 0, st>>>(mass, tile_mass, N, tile_j,
                                                                                      n_tiles, enable);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}
int launch_tile_mass_f32(const float* mass, float* tile_mass, int64_t N, int tile_j, int n_tiles, int enable,
                         cudaStream_t st) {
    return launch_tile_mass(mass, tile_mass, N, tile_j, n_tiles, enable, st);
}
int launch_tile_mass_f64(const double* mass, double* tile_mass, int64_t N, int tile_j, int n_tiles, int enable,
                         cudaStream_t st) {
    return launch_tile_mass(mass, tile_mass, N, tile_j, n_tiles, enable, st);
}
int launch_tile_mass_f64_to_f32(const double* mass, float* tile_mass, int64_t N, int tile_j, int n_tiles, int enable,
                                cudaStream_t st) {
    return launch_tile_mass(mass, tile_mass, N, tile_j, n_tiles, enable, st);
}
int launch_tile_mass_f32_to_f64(const float* mass, double* tile_mass, int64_t N, int tile_j, int n_tiles, int enable,
                                cudaStream_t st) {
    return launch_tile_mass(mass, tile_mass, N, tile_j, n_tiles, enable, st);
}

}  // namespace ppgrav
