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
//    once per tile in the fold -- 15 (17) instead of 16 (18) operations per interaction.  MODE_POT (pp_invariants' potential sweep): 11 instead of 12.
//  * blocked accumulation: per-tile sums are folded into outer sums after every tile (plain FP64 for the force,
//    TwoSum double-double for MODE_POT, which feeds the energy diagnostic).
#include "force_f64_common.cuh"
#include "tma_ring.cuh"

namespace ppgrav {
namespace {

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
    const bool use_tm = tile_mass != nullptr;
    double tm_next = (use_tm && nt > 0) ? __ldg(tile_mass + t0) : kNoCommonMass;

    for (int t = 0; t < nt; ++t) {
        const int s = t % STAGES;
        const double tm = tm_next;
        if (use_tm && t + 1 < nt) tm_next = __ldg(tile_mass + t0 + t + 1);
        const bool uni = tm == tm;
        mbar_wait(&full_bar[s], (uint32_t)(t / STAGES) & 1u);
        const double4* tp = reinterpret_cast<const double4*>(&tiles[s][0]);
        const int jbase = (t0 + t) * TJ;
        const bool diag = (MODE != MODE_FORCE) && !GUARD && (jbase < i_hi) && (jbase + TJ > i_lo);
        if (uni) {
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
            if (MODE == MODE_POT) { comp_add(sp[k], cp[k], __dmul_rn(scale, ap[k])); ap[k] = 0.0; }
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

template <int CLS, int MODE, bool GUARD>
int launch_cmg(const Plan& p, const double* packed, const double* tile_mass, double4* partial, double eps2,
               cudaStream_t st) {
    constexpr KernelShape K = kShapes[1][CLS][MODE];
    if (p.threads != K.threads || p.ipt != K.ipt || p.tile_j != K.tile_j) {
        set_error("launch_force_f64: plan (%d x %d, tile %d) does not match the kernel shape of class %d mode %d",
                  p.threads, p.ipt, p.tile_j, CLS, MODE);
        return PP_EINVAL;
    }
    dim3 grid(p.n_iblocks, p.split);
    force_f64_kernel<K.threads, K.ipt, K.tile_j, K.stages, K.ctas_per_sm, MODE, GUARD>
        <<<grid, K.threads, 0, st>>>(packed, tile_mass, partial, p.n_tiles, p.part_stride, p.i_begin, eps2);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}

template <int CLS>
int launch_class(const Plan& p, const double* packed, const double* tile_mass, double4* partial, double eps2,
                 bool guard, int mode, cudaStream_t st) {
    if (mode == MODE_FORCE)
        return guard ? launch_cmg<CLS, MODE_FORCE, true>(p, packed, tile_mass, partial, eps2, st)
                     : launch_cmg<CLS, MODE_FORCE, false>(p, packed, tile_mass, partial, eps2, st);
    if (mode == MODE_FORCE_POT)
        return guard ? launch_cmg<CLS, MODE_FORCE_POT, true>(p, packed, tile_mass, partial, eps2, st)
                     : launch_cmg<CLS, MODE_FORCE_POT, false>(p, packed, tile_mass, partial, eps2, st);
    return guard ? launch_cmg<CLS, MODE_POT, true>(p, packed, tile_mass, partial, eps2, st)
                 : launch_cmg<CLS, MODE_POT, false>(p, packed, tile_mass, partial, eps2, st);
}

}  // namespace

int launch_force_f64(const Plan& p, const double* packed, const double* tile_mass, double4* partial, int64_t N,
                     double delta, int mode, cudaStream_t st) {
    (void)N;
    const double eps2 = delta * delta;
    const bool guard = !(eps2 >= kTinyR2F64);
    switch (p.cls) {
        case CLS_LARGE: return launch_class<CLS_LARGE>(p, packed, tile_mass, partial, eps2, guard, mode, st);
        case CLS_MID: return launch_class<CLS_MID>(p, packed, tile_mass, partial, eps2, guard, mode, st);
        default: return launch_class<CLS_SMALL>(p, packed, tile_mass, partial, eps2, guard, mode, st);
    }
}

}  // namespace ppgrav
