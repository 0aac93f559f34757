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

#define PP_TRY_RC(expr)                 \
    do {                                \
        const int rc__ = (expr);        \
        if (rc__ != PP_OK) return rc__; \
    } while (0)

#define PP_CUDA(call)                                            \
    do {                                                         \
        cudaError_t e__ = (call);                                \
        if (e__ != cudaSuccess) return ::ppgrav::cuda_fail(e__, #call); \
    } while (0)

// ---- kernel shapes: one table read by both the plan (plan.cu) and the instantiations (force_f32.cu/force_f64.cu) -------
// Three shape classes per precision:
//   large  the throughput shape, 1 CTA per SM, whenever it fills the machine (N >~ 2^16)
//   mid    ~512 i-bodies per CTA, several CTAs per SM: N = 2^13 .. 2^16, where the large shape has too few i-blocks
//   small  one i-body per thread: tiny N
// A class fixes tile_j (the per-tile blocking of the sums, hence the bits of the result); threads and i-bodies per
// thread may differ between the sweep modes of a class (FP64 large: 7 i-bodies force-only, 6 with the potential).
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
#ifndef PP_F32_MID_THREADS
#define PP_F32_MID_THREADS 128
#endif
#ifndef PP_F32_MID_IPT
#define PP_F32_MID_IPT 4
#endif
#ifndef PP_F32_MID_TJ
#define PP_F32_MID_TJ 256
#endif
#ifndef PP_F32_MID_MINB
#define PP_F32_MID_MINB 3
#endif
#ifndef PP_F64_THREADS
#define PP_F64_THREADS 256
#endif
#ifndef PP_F64_IPT
#define PP_F64_IPT 6
#endif
#ifndef PP_F64_IPT_FORCE
#define PP_F64_IPT_FORCE 7
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
#ifndef PP_F64_MID_THREADS
#define PP_F64_MID_THREADS 128
#endif
#ifndef PP_F64_MID_IPT
#define PP_F64_MID_IPT 4
#endif
#ifndef PP_F64_MID_TJ
#define PP_F64_MID_TJ 128
#endif
#ifndef PP_F64_MID_MINB
#define PP_F64_MID_MINB 3
#endif
constexpr int kF32Unroll = PP_F32_UNROLL;   // j-pairs (FP32) / j-bodies (FP64) per unrolled loop body
constexpr int kF64Unroll = PP_F64_UNROLL;
struct KernelShape {
    int threads, ipt, tile_j, stages, ctas_per_sm;
};
enum { CLS_LARGE = 0, CLS_MID = 1, CLS_SMALL = 2, kNumClasses = 3 };
// modes of the pair sweep
enum { MODE_FORCE = 0, MODE_FORCE_POT = 1, MODE_POT = 2, kNumModes = 3 };
// kShapes[precision][class][mode]
constexpr KernelShape kShapeF32Large = {PP_F32_THREADS, PP_F32_IPT, PP_F32_TJ, 4, PP_F32_MINB};
constexpr KernelShape kShapeF32Mid = {PP_F32_MID_THREADS, PP_F32_MID_IPT, PP_F32_MID_TJ, 4, PP_F32_MID_MINB};
constexpr KernelShape kShapeF32Small = {128, 1, 128, 4, 4};
constexpr KernelShape kShapeF64Large = {PP_F64_THREADS, PP_F64_IPT, PP_F64_TJ, 4, PP_F64_MINB};
constexpr KernelShape kShapeF64LargeForce = {PP_F64_THREADS, PP_F64_IPT_FORCE, PP_F64_TJ, 4, PP_F64_MINB};
constexpr KernelShape kShapeF64Mid = {PP_F64_MID_THREADS, PP_F64_MID_IPT, PP_F64_MID_TJ, 4, PP_F64_MID_MINB};
constexpr KernelShape kShapeF64Small = {128, 1, 128, 4, 4};
// shape of the symmetric (every unordered pair once) sweeps: the block must be a whole number of tiles and a tile has
// one body per thread (its j-side sums are reduced one thread per body)
#ifndef PP_SYM32_THREADS
#define PP_SYM32_THREADS 256
#endif
#ifndef PP_SYM32_IPT
#define PP_SYM32_IPT 8
#endif
#ifndef PP_SYM32_JP
#define PP_SYM32_JP 1
#endif
#ifndef PP_SYM32_UNROLL
#define PP_SYM32_UNROLL 2
#endif
#ifndef PP_SYM64_IPT
#define PP_SYM64_IPT 8
#endif
#ifndef PP_SYM64_UNROLL
#define PP_SYM64_UNROLL 2
#endif
constexpr int kSymF32Jp = PP_SYM32_JP;          // j-pairs a lane keeps in flight (force_sym_f32.cu)
constexpr int kSymF32Unroll = PP_SYM32_UNROLL;  // systolic steps per unrolled loop body
constexpr int kSymF64Unroll = PP_SYM64_UNROLL;
constexpr KernelShape kShapeF32Sym = {PP_SYM32_THREADS, PP_SYM32_IPT, 256, 4, 1};
constexpr KernelShape kShapeF64Sym = {256, PP_SYM64_IPT, 256, 4, 1};
// the same kernels on 128-body tiles: half the work unit, for the sizes (N < 2^17) where a solve is only 1-2 waves of
// CTAs and the granularity of a 29-us tile costs more than the doubled per-tile overhead
constexpr KernelShape kShapeF32SymFine = {PP_SYM32_THREADS, PP_SYM32_IPT, 128, 4, 1};
constexpr KernelShape kShapeF64SymFine = {256, PP_SYM64_IPT, 128, 4, 1};
constexpr int64_t kSymFineBelow = 98304;
constexpr KernelShape kShapes[2][kNumClasses][kNumModes] = {
    {{kShapeF32Large, kShapeF32Large, kShapeF32Large},
     {kShapeF32Mid, kShapeF32Mid, kShapeF32Mid},
     {kShapeF32Small, kShapeF32Small, kShapeF32Small}},
    {{kShapeF64LargeForce, kShapeF64Large, kShapeF64Large},
     {kShapeF64Mid, kShapeF64Mid, kShapeF64Mid},
     {kShapeF64Small, kShapeF64Small, kShapeF64Small}},
};

// ---- launch plan of one gravity solve (plan.cu) --------------------------------------------------------------
// The all-pairs sweep is cut into work units (i-block, j-split): CTA (ib, s) sweeps the j-tiles of split s for the
// bodies of i-block ib and writes one partial sum per body; a finalize kernel adds the S partials in fixed order.
struct Plan {
    int cls;            // CLS_LARGE / CLS_MID / CLS_SMALL
    int mode;           // MODE_* the plan was made for (selects the shape within the class)
    int threads;        // threads per CTA
    int ipt;            // i-bodies per thread
    int i_per_cta;      // threads * ipt
    int tile_j;         // j-bodies per shared-memory tile
    int stages;         // depth of the TMA ring
    int ctas_per_sm;    // residency the kernel is built for
    int64_t n_pad;      // length of the packed array this plan needs: covers every j-tile and every launched i-block,
                        // padded with massless bodies (N, or i_begin + part_stride for an i-range that starts off a
                        // block boundary, rounded up to a multiple of tile_j)
    int64_t i_begin;    // first i-body of the solve (0 for a full solve; pp_forces_range shards the i-range)
    int64_t i_count;    // i-bodies of the solve
    int n_iblocks;      // ceil(i_count / i_per_cta): i-blocks launched
    int64_t part_stride;   // n_iblocks * i_per_cta: bodies per split in the partial-sum workspace (local index i - i_begin)
    int n_tiles;        // ceil(N / tile_j): j-tiles that contain a real body
    int split;          // S
    int sm_count;
    // symmetric sweep (force_sym_*.cu): every unordered pair once.  Blocks = i-blocks; block I sweeps the blocks
    // I+1 .. I+sym_h two-sidedly; j-side sums go to partial_j[sym_h][part_stride].
    int sym;            // 1 = this plan runs the symmetric kernel
    int sym_h;          // floor((n_iblocks - 1) / 2): partner offsets d = 1 .. sym_h
    int sym_rows;       // partner offsets per band (= rows of partial_j); sym_h when one band holds them all
    int sym_bands;      // ceil(sym_h / sym_rows), at least 1
};
// forced_split >= 1 pins S (capped by the tile count); forced_cls in {0,1,2} pins the shape class, -1 = choose.
Plan make_plan(int64_t N, int precision, int mode, int sm_count, int64_t forced_split, int forced_cls,
               int64_t i_begin = 0, int64_t i_count = -1);
// plan of the symmetric sweep for a full solve of N bodies; bytes of its j-side workspace in *jbytes
// (rows_cap_bytes: the j-side rows of one band may take that much; *jbytes = bytes of partial_j, *abytes = bytes of
// the running j-side sums acc_j that bands need, 0 for a single band)
// fine_tiles: 1 = 128-body j-tiles, 0 = 256-body, -1 = by size (128 below kSymFineBelow)
Plan make_sym_plan(int64_t N, int precision, int mode, int sm_count, int64_t forced_split, size_t rows_cap_bytes,
                   size_t* jbytes, size_t* abytes, int fine_tiles = -1);

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
int launch_tile_mass_f32_to_f64(const float* mass, double* tile_mass, int64_t N, int tile_j, int n_tiles, int enable,
                                cudaStream_t st);   // pp_invariants' FP64 potential sweep on an FP32 state

// PP_MIXED variants of finalize and kick_drift_pack: FP32 partial sums / packed copy, FP64 state
int launch_finalize_mixed(const float4* partial, int split, int64_t n_pad, int64_t N, double G, double* acc,
                          double* pot, double* vel, double kick, cudaStream_t st, const float4* partial_j = nullptr,
                          int jrows = 0, int64_t jstride = 0);
int launch_kick_drift_pack_mixed(double* pos, double* vel, const double* acc, const double* mass, float* packed,
                                 int64_t N, int64_t n_pad, double kick, double dt, cudaStream_t st);

// partial[s * part_stride + (i - i_begin)] = {sum_x, sum_y, sum_z, sum_pot} over the j-tiles of split s, without G and with the
// sign convention  sum = sum_j m_j (r_j - r_i) w^3,  sum_pot = sum_j m_j w   (w = (r^2+delta^2)^{-1/2}).
// tile_mass: per-j-tile common mass (launch_tile_mass_*), or NULL = treat every tile as mixed.
int launch_force_f32(const Plan& p, const float* packed, const float* tile_mass, float4* partial, int64_t N,
                     double delta, int mode, cudaStream_t st);
// symmetric sweep: i-side sums to partial[S][part_stride], j-side sums to partial_j[sym_h][part_stride] (same sign
// convention, ready to be added); block_mass[I] = common mass of i-block I or NaN (launch_tile_mass_* with tile = block)
// With p.sym_bands > 1 the partials and the rows are reused band after band and summed into acc_j[2][part_stride]
// (TwoSum value / error), which is then all that finalize reads (split = 0, two j-side "rows").
int launch_force_sym_f32(const Plan& p, const float* packed, const float* tile_mass, const float* block_mass,
                         float4* partial, float4* partial_j, float4* acc_j, double delta, int mode, cudaStream_t st);
int launch_fold_rows(const float4* rows, int nrows, int64_t stride, float4* acc_j, bool first, cudaStream_t st);
int launch_fold_rows(const double4* rows, int nrows, int64_t stride, double4* acc_j, bool first, cudaStream_t st);
int launch_force_sym_f64(const Plan& p, const double* packed, const double* tile_mass, const double* block_mass,
                         double4* partial, double4* partial_j, double4* acc_j, double delta, int mode, cudaStream_t st);
// MODE_POT writes {pot_hi, pot_lo, 0, 0} (double-double partial of the potential sum).
int launch_force_f64(const Plan& p, const double* packed, const double* tile_mass, double4* partial, int64_t N,
                     double delta, int mode, cudaStream_t st);

// acc = G * sum_s partial (fixed order, compensated), pot = -G * sum_s partial.w; optional fused kick
// vel += kick * acc (kick = 0: none).  acc/pot/vel may be NULL where not wanted.
// partial_j / jrows / jstride: the j-side rows of the symmetric sweep (force_sym_*.cu), added after the S partials.
int launch_finalize_f32(const float4* partial, int split, int64_t n_pad, int64_t N, double G, float* acc, float* pot,
                        float* vel, double kick, cudaStream_t st, const float4* partial_j = nullptr, int jrows = 0,
                        int64_t jstride = 0);
int launch_finalize_f64(const double4* partial, int split, int64_t n_pad, int64_t N, double G, double* acc,
                        double* pot, double* vel, double kick, int pot_is_dd, cudaStream_t st,
                        const double4* partial_j = nullptr, int jrows = 0, int64_t jstride = 0);

// v += kick * a;  r += dt * v   on n bodies, no packing (the sharded step kicks and drifts its own bodies only)
int launch_kick_drift_f32(float* pos, float* vel, const float* acc, int64_t n, double kick, double dt, cudaStream_t st);
int launch_kick_drift_f64(double* pos, double* vel, const double* acc, int64_t n, double kick, double dt,
                          cudaStream_t st);

// v += kick * a;  r += dt * v;  packed = pack(r, m)      (eqs. (5)-(6) in half-kick form)
int launch_kick_drift_pack_f32(float* pos, float* vel, const float* acc, const float* mass, float* packed, int64_t N,
                               int64_t n_pad, double kick, double dt, cudaStream_t st);
int launch_kick_drift_pack_f64(double* pos, double* vel, const double* acc, const double* mass, double* packed,
                               int64_t N, int64_t n_pad, double kick, double dt, cudaStream_t st);

// finalize + closing half-kick + opening half-kick + drift + re-pack in one pass (interior steps of pp_step_kdk)
int launch_finalize_kick_drift_pack_f32(const float4* partial, int split, int64_t part_stride, int64_t N, double G,
                                        float* acc, float* vel, float* pos, const float* mass, float* packed,
                                        double kick, double dt, cudaStream_t st,
                                        const float4* partial_j = nullptr, int jrows = 0, int64_t jstride = 0);
int launch_finalize_kick_drift_pack_f64(const double4* partial, int split, int64_t part_stride, int64_t N, double G,
                                        double* acc, double* vel, double* pos, const double* mass, double* packed,
                                        double kick, double dt, cudaStream_t st,
                                        const double4* partial_j = nullptr, int jrows = 0, int64_t jstride = 0);
int launch_finalize_kick_drift_pack_mixed(const float4* partial, int split, int64_t part_stride, int64_t N, double G,
                                          double* acc, double* vel, double* pos, const double* mass, float* packed,
                                          double kick, double dt, cudaStream_t st,
                                        const float4* partial_j = nullptr, int jrows = 0, int64_t jstride = 0);

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

}  // namespace ppgrav
