// ppgrav_internal.h -- declarations shared by the translation units of libppgrav (not part of the C ABI).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "ppgrav.h"

namespace ppgrav {

// ---- error plumbing (api.cu) ------------------------------------------------------------------------------
void set_error(const char* fmt, ...);
int cuda_fail(cudaError_t e, const char* what);   // records the message, returns PP_ECUDA
void count_launch(int n = 1);

#define PP_CUDA(call)                                            \
    do {                                                         \
        cudaError_t e__ = (call);                                \
        if (e__ != cudaSuccess) return ::ppgrav::cuda_fail(e__, #call); \
    } while (0)

// ---- kernel shapes: one table read by both the plan (plan.cu) and the instantiations (force_f32.cu/force_f64.cu) -------
// "large" = the throughput shape used whenever it fills the machine, "small" = the fallback for tiny N.
// Overridable at compile time (-DPP_F32_IPT=2 ...) for tuning sweeps; the defaults are the measured best.
#ifndef PP_F32_THREADS
#define PP_F32_THREADS 256
#endif
#ifndef PP_F32_IPT
#define PP_F32_IPT 7
#endif
#ifndef PP_F32_TJ
#define PP_F32_TJ 512
#endif
#ifndef PP_F32_MINB
#define PP_F32_MINB 1
#endif
#ifndef PP_F32_UNROLL
#define PP_F32_UNROLL 2
#endif
#ifndef PP_F64_THREADS
#define PP_F64_THREADS 256
#endif
#ifndef PP_F64_IPT
#define PP_F64_IPT 6
#endif
#ifndef PP_F64_TJ
#define PP_F64_TJ 256
#endif
#ifndef PP_F64_MINB
#define PP_F64_MINB 1
#endif
#ifndef PP_F64_UNROLL
#define PP_F64_UNROLL 2
#endif
constexpr int kF32Unroll = PP_F32_UNROLL;   // j-pairs (FP32) / j-bodies (FP64) per unrolled loop body
constexpr int kF64Unroll = PP_F64_UNROLL;
struct KernelShape {
    int threads, ipt, tile_j, stages, ctas_per_sm;
};
constexpr KernelShape kShapeF32Large = {PP_F32_THREADS, PP_F32_IPT, PP_F32_TJ, 4, PP_F32_MINB};
constexpr KernelShape kShapeF32Small = {128, 1, 128, 4, 4};
constexpr KernelShape kShapeF64Large = {PP_F64_THREADS, PP_F64_IPT, PP_F64_TJ, 4, PP_F64_MINB};
constexpr KernelShape kShapeF64Small = {128, 1, 128, 4, 4};

// ---- launch plan of one gravity solve (plan.cu) --------------------------------------------------------------
// The all-pairs sweep is cut into work units (i-block, j-split): CTA (ib, s) sweeps the j-tiles of split s for the
// bodies of i-block ib and writes one partial sum per body; a finalize kernel adds the S partials in fixed order.
struct Plan {
    int variant;        // 0 = large shape, 1 = small shape (see KernelShape above)
    int threads;        // threads per CTA
    int ipt;            // i-bodies per thread
    int i_per_cta;      // threads * ipt
    int tile_j;         // j-bodies per shared-memory tile
    int stages;         // depth of the TMA ring
    int ctas_per_sm;    // residency the kernel is built for
    int64_t n_pad;      // length of the packed array: covers every j-tile and every launched i-block, padded with
                        // massless bodies (N, or N + i_per_cta for an i-range that starts off a block boundary,
                        // rounded up to a multiple of i_per_cta, which tile_j divides)
    int64_t i_begin;    // first i-body of the solve (0 for a full solve; pp_forces_range shards the i-range)
    int64_t i_count;    // i-bodies of the solve
    int n_iblocks;      // ceil(i_count / i_per_cta): i-blocks launched
    int64_t part_stride;   // n_iblocks * i_per_cta: bodies per split in the partial-sum workspace (local index i - i_begin)
    int n_tiles;        // ceil(N / tile_j): j-tiles that contain a real body
    int split;          // S
    int sm_count;
};
Plan make_plan(int64_t N, int precision, int sm_count, int64_t forced_split, int64_t i_begin = 0, int64_t i_count = -1);

// modes of the pair sweep
enum { MODE_FORCE = 0, MODE_FORCE_POT = 1, MODE_POT = 2 };

// ---- kernels (one launcher per translation unit) -----------------------------------------------------------------
// Packed bodies.  FP32: pairs of bodies interleaved, 8 floats {x0 x1 y0 y1 z0 z1 m0 m1} per pair (so that one
// 64-bit shared-memory word feeds one packed f32x2 operand).  FP64: double4 {x y z m} per body.  Bodies N..n_pad-1
// are padding: mass 0 at the origin.
int launch_pack_f32(const float* pos, const float* mass, float* packed, int64_t N, int64_t n_pad, cudaStream_t st);
int launch_pack_f64(const double* pos, const double* mass, double* packed, int64_t N, int64_t n_pad, cudaStream_t st);
int launch_pack_f32_to_f64(const float* pos, const float* mass, double* packed, int64_t N, int64_t n_pad,
                           cudaStream_t st);
int launch_pack_f64_to_f32(const double* pos, const double* mass, float* packed, int64_t N, int64_t n_pad,
                           cudaStream_t st);   // PP_MIXED: FP64 state, FP32 sweep

// tile_mass[t] (sweep precision) = common mass of the tile_j bodies of j-tile t, NaN if they differ (or !enable)
int launch_tile_mass_f32(const float* mass, float* tile_mass, int64_t N, int tile_j, int n_tiles, int enable,
                         cudaStream_t st);
int launch_tile_mass_f64(const double* mass, double* tile_mass, int64_t N, int tile_j, int n_tiles, int enable,
                         cudaStream_t st);
int launch_tile_mass_f64_to_f32(const double* mass, float* tile_mass, int64_t N, int tile_j, int n_tiles, int enable,
                                cudaStream_t st);

// PP_MIXED variants of finalize and kick_drift_pack: FP32 partial sums / packed copy, FP64 state
int launch_finalize_mixed(const float4* partial, int split, int64_t n_pad, int64_t N, double G, double* acc,
                          double* pot, double* vel, double kick, cudaStream_t st);
int launch_kick_drift_pack_mixed(double* pos, double* vel, const double* acc, const double* mass, float* packed,
                                 int64_t N, int64_t n_pad, double kick, double dt, cudaStream_t st);

// partial[s * part_stride + (i - i_begin)] = {sum_x, sum_y, sum_z, sum_pot} over the j-tiles of split s, without G and with the
// sign convention  sum = sum_j m_j (r_j - r_i) w^3,  sum_pot = sum_j m_j w   (w = (r^2+delta^2)^{-1/2}).
// tile_mass: per-j-tile common mass (launch_tile_mass_*), or NULL = treat every tile as mixed.
int launch_force_f32(const Plan& p, const float* packed, const float* tile_mass, float4* partial, int64_t N,
                     double delta, int mode, cudaStream_t st);
// MODE_POT writes {pot_hi, pot_lo, 0, 0} (double-double partial of the potential sum).
int launch_force_f64(const Plan& p, const double* packed, const double* tile_mass, double4* partial, int64_t N,
                     double delta, int mode, cudaStream_t st);

// acc = G * sum_s partial (fixed order, compensated), pot = -G * sum_s partial.w; optional fused kick
// vel += kick * acc (kick = 0: none).  acc/pot/vel may be NULL where not wanted.
int launch_finalize_f32(const float4* partial, int split, int64_t n_pad, int64_t N, double G, float* acc, float* pot,
                        float* vel, double kick, cudaStream_t st);
int launch_finalize_f64(const double4* partial, int split, int64_t n_pad, int64_t N, double G, double* acc,
                        double* pot, double* vel, double kick, int pot_is_dd, cudaStream_t st);

// v += kick * a;  r += dt * v   on n bodies, no packing (the sharded step kicks and drifts its own bodies only)
int launch_kick_drift_f32(float* pos, float* vel, const float* acc, int64_t n, double kick, double dt, cudaStream_t st);
int launch_kick_drift_f64(double* pos, double* vel, const double* acc, int64_t n, double kick, double dt,
                          cudaStream_t st);

// v += kick * a;  r += dt * v;  packed = pack(r, m)      (eqs. (5)-(6) in half-kick form)
int launch_kick_drift_pack_f32(float* pos, float* vel, const float* acc, const float* mass, float* packed, int64_t N,
                               int64_t n_pad, double kick, double dt, cudaStream_t st);
int launch_kick_drift_pack_f64(double* pos, double* vel, const double* acc, const double* mass, double* packed,
                               int64_t N, int64_t n_pad, double kick, double dt, cudaStream_t st);

// eqs. (8)-(10): block partials (double-double) then a single-block fixed-order sum into out16.
int invariants_scratch_doubles(int64_t N);
int launch_invariants_f32(const float* pos, const float* vel, const float* mass, const float* pot_state,
                          const double* pot64, int64_t N, double* scratch, double* out16, cudaStream_t st);
int launch_invariants_f64(const double* pos, const double* vel, const double* mass, const double* pot_state,
                          const double* pot64, int64_t N, double* scratch, double* out16, cudaStream_t st);

// Fig. 7 surface-density map (density.cu): sigma[iy * nx + ix] = sum of m in the cell / cell^2
int launch_density_f32(const float* pos, const float* mass, int64_t N, double x0, double y0, double cell, int nx,
                       int ny, double* sigma, int sm_count, cudaStream_t st);
int launch_density_f64(const double* pos, const double* mass, int64_t N, double x0, double y0, double cell, int nx,
                       int ny, double* sigma, int sm_count, cudaStream_t st);

// pipe microbenchmarks (probe.cu)
int run_probe(int kind, int64_t iters, int sm_count, double* out4);

}  // namespace ppgrav
