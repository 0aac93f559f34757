// force_f64.cu -- FP64 all-pairs gravity sweep for sm_100a (eq. (1)-(2); the paper's
// double-precision "Gravity Force Computation" kernel).
//
// Same structure as force_f32.cu (TMA ring of j-tiles, IPT i-bodies per thread in registers, (i-block, j-split)
// work units, fixed-order finalize).  What is specific to FP64:
//  * there is no FP64 reciprocal-square-root unit: the seed is one MUFU.RSQ64H (rsqrt.approx.ftz.f64, ~20 good
//    bits, reads only the high word) and ONE third-order correction brings it to full double precision.  With
//    y the seed and e = 1 - x y^2:  x^{-1/2} = y (1 + e/2 + 3e^2/8 + O(e^3)),  x^{-3/2} = y^3 (1 + 3e/2 + 15e^2/8 +
//    O(e^3)).  MODE_FORCE fuses the correction with the cube: 16 FP64-pipe operations per interaction
//    (3 DADD + 3 DFMA + 7 + 3 DFMA); with the potential 18; potential only (pp_invariants) 12.  Never 1.0/sqrt(x)
//    (~30 FP64 operations).
//  * equal-mass tiles (tile_mass[t] = the common mass, NaN otherwise; see force_f32.cu): the factor m_j is applied
//    once per tile in the fold -- 15 (17) instead of 16 (18) operations per interaction.  MODE_POT keeps m_j inside.
//  * blocked accumulation: per-tile sums are folded into outer sums after every tile (plain FP64 for the force,
//    TwoSum double-double for MODE_POT, which feeds the energy diagnostic).
#include "ppgrav_internal.h"
#include "tma_ring.cuh"

namespace ppgrav {
namespace {

__device__ __forceinline__ double rsqrt64h(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}

__device__ __forceinline__ void comp_add(double& s, double& c, double t) {
    const double n = __dadd_rn(s, t);
    const double bp = __dsub_rn(n, s);
    const double e = __dadd_rn(__dsub_rn(s, __dsub_rn(n, bp)), __dsub_rn(t, bp));
    s = n;
    c = __dadd_rn(c, e);
}

template <int IPT, int MODE, bool GUARD, bool DIAG, bool UNI>
__device__ __forceinline__ void sweep_tile(const double4* __restrict__ tp, const int nj, const double (&xi)[IPT],
                                           const double (&yi)[IPT], const double (&zi)[IPT], double (&ax)[IPT],
                                           double (&ay)[IPT], double (&az)[IPT], double (&ap)[IPT], const double eps2,
                                           const int jbase, const int (&iidx)[IPT]) {
#pragma unroll kF64Unroll
    for (int j = 0; j < nj; ++j) {
        const double4 b = tp[j];
#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            const double dx = b.x - xi[k];                    // r_j - r_i
            const double dy = b.y - yi[k];
            const double dz = b.z - zi[k];
            double r2 = fma(dx, dx, eps2);                    // |r_i - r_j|^2 + delta^2
            r2 = fma(dy, dy, r2);
            r2 = fma(dz, dz, r2);
            double y = rsqrt64h(r2);
            if (GUARD) y = r2 > 0.0 ? y : 0.0;                // delta == 0: zero-distance pairs contribute nothing
            const double t = y * y;
            const double e = fma(-r2, t, 1.0);                // 1 - x y^2
            if (MODE == MODE_FORCE) {
                const double p = fma(e, 1.875, 1.5);
                const double u = UNI ? y : b.w * y;           // equal-mass tile: m_j is applied in the fold
                const double w = u * t;                       // m y^3
                const double we = w * e;
                const double s = fma(p, we, w);               // m x^{-3/2}
                ax[k] = fma(s, dx, ax[k]);
                ay[k] = fma(s, dy, ay[k]);
                az[k] = fma(s, dz, az[k]);
            } else {
                const double q = fma(e, 0.375, 0.5);
                const double ye = y * e;
                const double yy = fma(q, ye, y);              // x^{-1/2} to full precision
                double u = UNI ? yy : b.w * yy;               // m / r
                if (MODE == MODE_FORCE_POT) {
                    const double s = u * (yy * yy);
                    ax[k] = fma(s, dx, ax[k]);
                    ay[k] = fma(s, dy, ay[k]);
                    az[k] = fma(s, dz, az[k]);
                }
                if (DIAG && (jbase + j == iidx[k])) u = 0.0;  // drop j == i from the potential
                ap[k] += u;
            }
        }
    }
}

template <int THREADS, int IPT, int TJ, int STAGES, int MINB, int MODE, bool GUARD>
__global__ void __launch_bounds__(THREADS, MINB)
force_f64_kernel(const double* __restrict__ packed, const double* __restrict__ tile_mass,
                 double4* __restrict__ partial, const int n_tiles, const int64_t part_stride, const int64_t i_begin,
                 const double eps2) {
    constexpr int NWARPS = THREADS / 32;
    constexpr uint32_t TILE_BYTES = TJ * 32u;
    __shared__ __align__(128) double tiles[STAGES][TJ * 4];
    __shared__ __align__(8) uint64_t full_bar[STAGES];
    __shared__ __align__(8) uint64_t empty_bar[STAGES];

    const int tid = threadIdx.x;
    const int ib = blockIdx.x;
    const int split = gridDim.y, sidx = blockIdx.y;
    const int t0 = (int)(((int64_t)n_tiles * sidx) / split);
    const int t1 = (int)(((int64_t)n_tiles * (sidx + 1)) / split);
    const int nt = t1 - t0;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], NWARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        const int pre = nt < STAGES ? nt : STAGES;
        for (int s = 0; s < pre; ++s) {
            mbar_expect_tx(&full_bar[s], TILE_BYTES);
            tma_load_1d(&tiles[s][0], packed + (size_t)(t0 + s) * TJ * 4, TILE_BYTES, &full_bar[s]);
        }
    }

    double xi[IPT], yi[IPT], zi[IPT];
    double ax[IPT], ay[IPT], az[IPT], ap[IPT];
    double sx[IPT], sy[IPT], sz[IPT], sp[IPT], cp[IPT];
    int iidx[IPT];
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const int i = (int)i_begin + ib * (THREADS * IPT) + k * THREADS + tid;   // global body index
        iidx[k] = i;
        const double4 q = reinterpret_cast<const double4*>(packed)[i];
        xi[k] = q.x; yi[k] = q.y; zi[k] = q.z;
        ax[k] = ay[k] = az[k] = ap[k] = 0.0;
        sx[k] = sy[k] = sz[k] = sp[k] = cp[k] = 0.0;
    }
    const int i_lo = (int)i_begin + ib * (THREADS * IPT), i_hi = i_lo + THREADS * IPT;

    // common mass of the bodies of tile t, NaN when they differ (fetched one tile ahead: no exposed latency)
    const double kNoCommonMass = __longlong_as_double(0x7ff8000000000000ll);
    const bool use_tm = (MODE != MODE_POT) && tile_mass != nullptr;
    double tm_next = (use_tm && nt > 0) ? __ldg(tile_mass + t0) : kNoCommonMass;

    for (int t = 0; t < nt; ++t) {
        const int s = t % STAGES;
        const double tm = tm_next;
        if (use_tm && t + 1 < nt) tm_next = __ldg(tile_mass + t0 + t + 1);
        const bool uni = (MODE != MODE_POT) && tm == tm;
        mbar_wait(&full_bar[s], (uint32_t)(t / STAGES) & 1u);
        const double4* tp = reinterpret_cast<const double4*>(&tiles[s][0]);
        const int jbase = (t0 + t) * TJ;
        const bool diag = (MODE != MODE_FORCE) && !GUARD && (jbase < i_hi) && (jbase + TJ > i_lo);
        if (MODE != MODE_POT && uni) {
            if (diag)
                sweep_tile<IPT, MODE, GUARD, true, true>(tp, TJ, xi, yi, zi, ax, ay, az, ap, eps2, jbase, iidx);
            else
                sweep_tile<IPT, MODE, GUARD, false, true>(tp, TJ, xi, yi, zi, ax, ay, az, ap, eps2, jbase, iidx);
        } else {
            if (diag)
                sweep_tile<IPT, MODE, GUARD, true, false>(tp, TJ, xi, yi, zi, ax, ay, az, ap, eps2, jbase, iidx);
            else
                sweep_tile<IPT, MODE, GUARD, false, false>(tp, TJ, xi, yi, zi, ax, ay, az, ap, eps2, jbase, iidx);
        }
        const double scale = uni ? tm : 1.0;   // x 1.0 is exact: the general path is unchanged bit for bit

        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty_bar[s]);
        if (tid == 0 && t >= 1 && t - 1 + STAGES < nt) {
            const int ps = (t - 1) % STAGES;
            mbar_wait(&empty_bar[ps], (uint32_t)((t - 1) / STAGES) & 1u);
            mbar_expect_tx(&full_bar[ps], TILE_BYTES);
            tma_load_1d(&tiles[ps][0], packed + (size_t)(t0 + t - 1 + STAGES) * TJ * 4, TILE_BYTES, &full_bar[ps]);
        }

#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            if (MODE != MODE_POT) {
                sx[k] = fma(scale, ax[k], sx[k]); sy[k] = fma(scale, ay[k], sy[k]); sz[k] = fma(scale, az[k], sz[k]);
                ax[k] = ay[k] = az[k] = 0.0;
            }
            if (MODE == MODE_FORCE_POT) { sp[k] = fma(scale, ap[k], sp[k]); ap[k] = 0.0; }
            if (MODE == MODE_POT) { comp_add(sp[k], cp[k], ap[k]); ap[k] = 0.0; }
        }
    }

#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        double4 o;
        if (MODE == MODE_POT) { o.x = sp[k]; o.y = cp[k]; o.z = 0.0; o.w = 0.0; }
        else { o.x = sx[k]; o.y = sy[k]; o.z = sz[k]; o.w = (MODE == MODE_FORCE_POT) ? sp[k] : 0.0; }
        partial[(size_t)sidx * part_stride + (iidx[k] - (int)i_begin)] = o;
    }
}

template <int THREADS, int IPT, int TJ, int STAGES, int MINB>
int launch_variant(const Plan& p, const double* packed, const double* tile_mass, double4* partial, int64_t N,
                   double eps2, bool guard, int mode, cudaStream_t st) {
    dim3 grid(p.n_iblocks, p.split);
#define PP_LAUNCH64(MODE_, GUARD_)                                                      \
    force_f64_kernel<THREADS, IPT, TJ, STAGES, MINB, MODE_, GUARD_>                     \
        <<<grid, THREADS, 0, st>>>(packed, tile_mass, partial, p.n_tiles, p.part_stride, p.i_begin, eps2)
    if (mode == MODE_FORCE) {
        if (guard) PP_LAUNCH64(MODE_FORCE, true); else PP_LAUNCH64(MODE_FORCE, false);
    } else if (mode == MODE_FORCE_POT) {
        if (guard) PP_LAUNCH64(MODE_FORCE_POT, true); else PP_LAUNCH64(MODE_FORCE_POT, false);
    } else {
        if (guard) PP_LAUNCH64(MODE_POT, true); else PP_LAUNCH64(MODE_POT, false);
    }
#undef PP_LAUNCH64
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}

}  // namespace

int launch_force_f64(const Plan& p, const double* packed, const double* tile_mass, double4* partial, int64_t N,
                     double delta, int mode, cudaStream_t st) {
    const double eps2 = delta * delta;
    const bool guard = !(eps2 >= 2.2250738585072014e-308);
    constexpr KernelShape L = kShapeF64Large, S = kShapeF64Small;
    if (p.variant == 0)
        return launch_variant<L.threads, L.ipt, L.tile_j, L.stages, L.ctas_per_sm>(p, packed, tile_mass, partial, N,
                                                                                    eps2, guard, mode, st);
    return launch_variant<S.threads, S.ipt, S.tile_j, S.stages, S.ctas_per_sm>(p, packed, tile_mass, partial, N, eps2,
                                                                                guard, mode, st);
}

}  // namespace ppgrav
