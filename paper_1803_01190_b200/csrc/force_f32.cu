// force_f32.cu -- FP32 all-pairs gravity sweep for sm_100a (the paper's "Gravity Force Computation" kernel,
// PAPER.md:110-112, eq. (1)-(2) PAPER.md:41-48), redesigned for Blackwell:
//
//  * j-bodies arrive in shared memory through a 4-stage TMA bulk-copy ring (tma_ring.cuh); no thread spends
//    issue slots on staging and warps only meet at mbarriers.
//  * each thread keeps IPT i-bodies in registers and processes TWO j-bodies per instruction with the packed
//    f32x2 pipe instructions sm_100 added (FADD2/FMUL2/FFMA2): the tile is stored pair-interleaved
//    {x0 x1 y0 y1 z0 z1 m0 m1}, so one LDS.128 yields two ready-made packed operands.  Per pair of interactions:
//    3 FADD2 + 3 FFMA2 + 2 MUFU.RSQ + 3 FMUL2 + 3 FFMA2 (+1 FADD2 with the potential) = 12 (13) FP32-pipe
//    operations per interaction in 7 (7.5) issue slots.
//  * accumulation is blocked: the packed accumulators only ever hold TJ/2 terms; after every tile they are folded
//    into a compensated (TwoSum) FP32 outer sum.  A single FP32 accumulator over 2^20 terms is wrong at the 1e-3
//    level; this keeps the whole solve at ~1e-7.
//  * equal-mass tiles: when every body of a j-tile has the same mass m (tile_mass[t] = m, written by
//    tile_mass_kernel in update.cu; NaN otherwise) the factor m_j leaves the pair loop -- the tile accumulates
//    sum_j w^3 (r_j - r_i) and sum_j w and is scaled by m once, in the fold.  11 (12) instead of 12 (13) FP32-pipe
//    operations per interaction; N-body workloads are made of a few mass species, so nearly every tile qualifies.
//  * the (i-block, j-split) decomposition gives the 148 SMs an even number of equal work units at any N; partial
//    sums go to a workspace and are added in fixed order by finalize (update.cu) -- no floating-point atomics.
#include "force_f32_common.cuh"
#include "tma_ring.cuh"

namespace ppgrav {
namespace {

template <int THREADS, int IPT, int TJ, int STAGES, int MINB, int MODE, bool GUARD>
__global__ void __launch_bounds__(THREADS, MINB)
force_f32_kernel(const float* __restrict__ packed, const float* __restrict__ tile_mass,
                 float4* __restrict__ partial, const int n_tiles, const int64_t part_stride, const int64_t i_begin,
                 const float eps2f) {
    constexpr int NWARPS = THREADS / 32;
    constexpr uint32_t TILE_BYTES = TJ * 16u;
    __shared__ __align__(128) float tiles[STAGES][TJ * 4];
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

    // this thread's i-bodies (negated and duplicated into both packed lanes)
    float2 nx[IPT], ny[IPT], nz[IPT];
    float2 ax[IPT], ay[IPT], az[IPT], ap[IPT];
    float sx[IPT], sy[IPT], sz[IPT], sp[IPT], cx[IPT], cy[IPT], cz[IPT], cp[IPT];
    int iidx[IPT];
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const int i = (int)i_begin + ib * (THREADS * IPT) + k * THREADS + tid;   // global body index
        iidx[k] = i;
        const float* q = packed + (size_t)(i >> 1) * 8 + (i & 1);
        const float xi = q[0], yi = q[2], zi = q[4];
        nx[k] = make_float2(-xi, -xi);
        ny[k] = make_float2(-yi, -yi);
        nz[k] = make_float2(-zi, -zi);
        ax[k] = ay[k] = az[k] = ap[k] = make_float2(0.f, 0.f);
        sx[k] = sy[k] = sz[k] = sp[k] = 0.f;
        cx[k] = cy[k] = cz[k] = cp[k] = 0.f;
    }
    const float2 eps2 = make_float2(eps2f, eps2f);
    const int i_lo = (int)i_begin + ib * (THREADS * IPT), i_hi = i_lo + THREADS * IPT;

    // common mass of the bodies of tile t, NaN when they differ (fetched one tile ahead: no exposed latency)
    const float kNoCommonMass = __int_as_float(0x7fc00000);
    float tm_next = (tile_mass && nt > 0) ? __ldg(tile_mass + t0) : kNoCommonMass;

    for (int t = 0; t < nt; ++t) {
        const int s = t % STAGES;
        const float tm = tm_next;
        if (tile_mass && t + 1 < nt) tm_next = __ldg(tile_mass + t0 + t + 1);
        const bool uni = tm == tm;
        mbar_wait(&full_bar[s], (uint32_t)(t / STAGES) & 1u);
        const float4* tp = reinterpret_cast<const float4*>(&tiles[s][0]);
        const int jbase = (t0 + t) * TJ;
        const bool diag = (MODE == MODE_FORCE_POT) && !GUARD && (jbase < i_hi) && (jbase + TJ > i_lo);
        if (uni) {
            if (diag)
                sweep_tile<IPT, MODE, GUARD, true, true>(tp, TJ / 2, nx, ny, nz, ax, ay, az, ap, eps2, jbase, iidx);
            else
                sweep_tile<IPT, MODE, GUARD, false, true>(tp, TJ / 2, nx, ny, nz, ax, ay, az, ap, eps2, jbase, iidx);
        } else {
            if (diag)
                sweep_tile<IPT, MODE, GUARD, true, false>(tp, TJ / 2, nx, ny, nz, ax, ay, az, ap, eps2, jbase, iidx);
            else
                sweep_tile<IPT, MODE, GUARD, false, false>(tp, TJ / 2, nx, ny, nz, ax, ay, az, ap, eps2, jbase, iidx);
        }
        const float scale = uni ? tm : 1.0f;   // x 1.0f is exact: the general path is unchanged bit for bit

        // release the stage, then (one tile late, so the wait is normally already satisfied) refill the stage
        // that held tile t-1 with tile t-1+STAGES
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty_bar[s]);
        if (tid == 0 && t >= 1 && t - 1 + STAGES < nt) {
            const int ps = (t - 1) % STAGES;
            mbar_wait(&empty_bar[ps], (uint32_t)((t - 1) / STAGES) & 1u);
            mbar_expect_tx(&full_bar[ps], TILE_BYTES);
            tma_load_1d(&tiles[ps][0], packed + (size_t)(t0 + t - 1 + STAGES) * TJ * 4, TILE_BYTES, &full_bar[ps]);
        }

        // blocked accumulation: fold the tile's packed partial sums into the compensated outer sums
#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            comp_add(sx[k], cx[k], __fmul_rn(scale, __fadd_rn(ax[k].x, ax[k].y)));
            comp_add(sy[k], cy[k], __fmul_rn(scale, __fadd_rn(ay[k].x, ay[k].y)));
            comp_add(sz[k], cz[k], __fmul_rn(scale, __fadd_rn(az[k].x, az[k].y)));
            ax[k] = ay[k] = az[k] = make_float2(0.f, 0.f);
            if (MODE == MODE_FORCE_POT) {
                comp_add(sp[k], cp[k], __fmul_rn(scale, __fadd_rn(ap[k].x, ap[k].y)));
                ap[k] = make_float2(0.f, 0.f);
            }
        }
    }

#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        float4 o;
        o.x = __fadd_rn(sx[k], cx[k]);
        o.y = __fadd_rn(sy[k], cy[k]);
        o.z = __fadd_rn(sz[k], cz[k]);
        o.w = (MODE == MODE_FORCE_POT) ? __fadd_rn(sp[k], cp[k]) : 0.f;
        partial[(size_t)sidx * part_stride + (iidx[k] - (int)i_begin)] = o;
    }
}

template <int CLS, int MODE, bool GUARD>
int launch_cmg(const Plan& p, const float* packed, const float* tile_mass, float4* partial, float eps2,
               cudaStream_t st) {
    constexpr KernelShape K = kShapes[0][CLS][MODE];
    if (p.threads != K.threads || p.ipt != K.ipt || p.tile_j != K.tile_j) {
        set_error("launch_force_f32: plan (%d x %d, tile %d) does not match the kernel shape of class %d mode %d",
                  p.threads, p.ipt, p.tile_j, CLS, MODE);
        return PP_EINVAL;
    }
    dim3 grid(p.n_iblocks, p.split);
    force_f32_kernel<K.threads, K.ipt, K.tile_j, K.stages, K.ctas_per_sm, MODE, GUARD>
        <<<grid, K.threads, 0, st>>>(packed, tile_mass, partial, p.n_tiles, p.part_stride, p.i_begin, eps2);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}

template <int CLS>
int launch_class(const Plan& p, const float* packed, const float* tile_mass, float4* partial, float eps2, bool guard,
                 int mode, cudaStream_t st) {
    if (mode == MODE_FORCE)
        return guard ? launch_cmg<CLS, MODE_FORCE, true>(p, packed, tile_mass, partial, eps2, st)
                     : launch_cmg<CLS, MODE_FORCE, false>(p, packed, tile_mass, partial, eps2, st);
    return guard ? launch_cmg<CLS, MODE_FORCE_POT, true>(p, packed, tile_mass, partial, eps2, st)
                 : launch_cmg<CLS, MODE_FORCE_POT, false>(p, packed, tile_mass, partial, eps2, st);
}

}  // namespace

int launch_force_f32(const Plan& p, const float* packed, const float* tile_mass, float4* partial, int64_t N,
                     double delta, int mode, cudaStream_t st) {
    (void)N;
    const float eps2 = (float)(delta * delta);
    const bool guard = !(eps2 >= kTinyR2F32);   // also catches NaN
    if (mode != MODE_FORCE && mode != MODE_FORCE_POT) {
        set_error("launch_force_f32: mode %d has no FP32 kernel", mode);
        return PP_EINVAL;
    }
    switch (p.cls) {
        case CLS_LARGE: return launch_class<CLS_LARGE>(p, packed, tile_mass, partial, eps2, guard, mode, st);
        case CLS_MID: return launch_class<CLS_MID>(p, packed, tile_mass, partial, eps2, guard, mode, st);
        default: return launch_class<CLS_SMALL>(p, packed, tile_mass, partial, eps2, guard, mode, st);
    }
}

}  // namespace ppgrav
