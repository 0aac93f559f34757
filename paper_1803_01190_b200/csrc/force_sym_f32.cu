// force_sym_f32.cu -- FP32 all-pairs gravity sweep that evaluates every UNORDERED pair once (sm_100a).
//
// eq. (2) is antisymmetric: m_i f_ij = -m_j f_ji.  The ordered-pair sweep of force_f32.cu spends 11 FP32-pipe
// operations on every (i <- j) and again on (j <- i); here one evaluation of r_j - r_i, r^2 + delta^2 and its -3/2 power
// feeds BOTH bodies: 14 packed operations per two ordered pairs (7 per ordered pair; 8 with the potential or with
// unequal masses) instead of 11 (12).  The work per pair interaction shrinks by a third; the pipe runs at ~0.76 instead
// of ~0.86 of its peak, because six of the fourteen instructions now read three distinct 64-bit register operands
// (ncu: math-pipe throttle and fixed-latency waits, profiles/r2_force_sym_f32_ncu.md).
//
//  * Bodies are cut into blocks of B = THREADS x IPT (256 x 8 = 2048).  Block I owns the unordered block pairs (I, I+d),
//    d = 1 .. H = floor((nb-1)/2), cyclically: every pair of distinct blocks exactly once, the same load for every I.
//    Its own block (and, for an even number of blocks, the block opposite, I + nb/2, which two CTAs share) is swept the
//    ordinary one-sided way (sweep_tile of force_f32_common.cuh): B/N of the work.  Split-j cuts the block's whole tile
//    list -- one-sided tiles first, then the partner tiles -- into S equal parts.
//  * j-tiles arrive through the same TMA ring as in force_f32.cu.  Inside a tile every lane of a warp takes one j-PAIR
//    (two bodies, one packed operand) into registers together with a packed accumulator for the pull of the warp's
//    i-bodies on it; 32 systolic steps rotate the j-pairs (and their accumulators) through the lanes by warp shuffles,
//    so after 32 steps each of the 64 j-bodies has met all 32 x IPT i-bodies of the warp.  No shared-memory traffic in
//    the pair loop at all; 12-16 shuffles per 14 pair evaluations.
//  * i-side per-tile packed sums stay in registers exactly as in force_f32.cu; the TwoSum outer sums they are folded
//    into once per tile live in shared memory, which frees the registers for 8 i-bodies per thread (measured: 7 % faster
//    than 7, the shuffles being shared by more pair work).
//    j-side sums of the 8 warps meet in shared memory once per tile and go to partial_j[d-1][j]; update.cu's finalize
//    adds, for every body, its S i-side partials and its H j-side partials in fixed order.  No atomics anywhere:
//    bit-reproducible run to run.
//  * Equal-mass shortcut as in force_f32.cu, now needing a common mass on both sides (the j-tile's, applied to the i-side
//    fold; the i-block's, applied to the j-side reduction).  Otherwise m_j w^3 and m_i w^3 are formed per pair.
#ifndef PP_SYM32_ORDER
#define PP_SYM32_ORDER 1   // measured: 267 against 274 ms force-only at N = 2^20 (profiles/r2_sym_tuning.md)
#endif
#include "force_f32_common.cuh"
#include <algorithm>

#include "tma_ring.cuh"

namespace ppgrav {
namespace {

__device__ __forceinline__ float2 rot(const float2 v, const int src) {
    return make_float2(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}

// One chunk of a tile: JP x 64 j-bodies (this lane starts with the j-pairs (xj, yj, zj, mj)[0..JP)) against the warp's
// 32 x IPT i-bodies.  On return (fx, fy, fz, fp)[q] holds, for the q-th j-pair this lane STARTED with,
// sum_i [m_i] w^3 (r_j - r_i) and sum_i [m_i] w over the warp's i-bodies ([m_i] only when !UNI), and the i-side packed
// sums have grown accordingly.  JP > 1 keeps independent j-pairs in flight, so that the shuffles of one overlap the
// arithmetic of the other.
template <int IPT, int JP, int MODE, bool GUARD, bool UNI>
__device__ __forceinline__ void sym_chunk(float2 (&xj)[JP], float2 (&yj)[JP], float2 (&zj)[JP], float2 (&mj)[JP],
                                          const float2 (&nx)[IPT], const float2 (&ny)[IPT], const float2 (&nz)[IPT],
                                          const float2 (&mi)[IPT], float2 (&ax)[IPT], float2 (&ay)[IPT],
                                          float2 (&az)[IPT], float2 (&ap)[IPT], float2 (&fx)[JP], float2 (&fy)[JP],
                                          float2 (&fz)[JP], float2 (&fp)[JP], const float2 eps2, const int lane) {
#pragma unroll
    for (int q = 0; q < JP; ++q) fx[q] = fy[q] = fz[q] = fp[q] = make_float2(0.f, 0.f);
    const int src = (lane + 1) & 31;
#pragma unroll kSymF32Unroll
    for (int step = 0; step < 32; ++step) {
#pragma unroll
        for (int q = 0; q < JP; ++q) {
#pragma unroll
            for (int k = 0; k < IPT; ++k) {
                const float2 dx = __fadd2_rn(xj[q], nx[k]);          // r_j - r_i (two j-bodies)
                const float2 dy = __fadd2_rn(yj[q], ny[k]);
                const float2 dz = __fadd2_rn(zj[q], nz[k]);
                float2 r2 = __ffma2_rn(dx, dx, eps2);                // |r_i - r_j|^2 + delta^2
                r2 = __ffma2_rn(dy, dy, r2);
                r2 = __ffma2_rn(dz, dz, r2);
                float2 w;
                w.x = rsqrt_approx(r2.x);
                w.y = rsqrt_approx(r2.y);
                if (GUARD) {
                    w.x = r2.x > kTinyR2F32 ? w.x : 0.f;
                    w.y = r2.y > kTinyR2F32 ? w.y : 0.f;
                }
                const float2 w3 = __fmul2_rn(w, __fmul2_rn(w, w));
                const float2 si = UNI ? w3 : __fmul2_rn(mj[q], w3);  // pull of j on i:  m_j w^3 (r_j - r_i)
                const float2 sj = UNI ? w3 : __fmul2_rn(mi[k], w3);  // pull of i on j: -m_i w^3 (r_j - r_i), sign in the reduction
#if PP_SYM32_ORDER == 1   // i-side and j-side update of one component back to back: they share two operands
                ax[k] = __ffma2_rn(si, dx, ax[k]);
                fx[q] = __ffma2_rn(sj, dx, fx[q]);
                ay[k] = __ffma2_rn(si, dy, ay[k]);
                fy[q] = __ffma2_rn(sj, dy, fy[q]);
                az[k] = __ffma2_rn(si, dz, az[k]);
                fz[q] = __ffma2_rn(sj, dz, fz[q]);
#else
                ax[k] = __ffma2_rn(si, dx, ax[k]);
                ay[k] = __ffma2_rn(si, dy, ay[k]);
                az[k] = __ffma2_rn(si, dz, az[k]);
                fx[q] = __ffma2_rn(sj, dx, fx[q]);
                fy[q] = __ffma2_rn(sj, dy, fy[q]);
                fz[q] = __ffma2_rn(sj, dz, fz[q]);
#endif
                if (MODE == MODE_FORCE_POT) {
                    ap[k] = UNI ? __fadd2_rn(ap[k], w) : __ffma2_rn(mj[q], w, ap[k]);
                    fp[q] = UNI ? __fadd2_rn(fp[q], w) : __ffma2_rn(mi[k], w, fp[q]);
                }
            }
            // systolic step: this j-pair, with the sums it has gathered, moves one lane down
            xj[q] = rot(xj[q], src); yj[q] = rot(yj[q], src); zj[q] = rot(zj[q], src);
            if (!UNI) mj[q] = rot(mj[q], src);
            fx[q] = rot(fx[q], src); fy[q] = rot(fy[q], src); fz[q] = rot(fz[q], src);
            if (MODE == MODE_FORCE_POT) fp[q] = rot(fp[q], src);
        }
    }   // after 32 rotations every pair is back in the lane it started in
}

template <int THREADS, int IPT, int TJ, int STAGES, int MODE, bool GUARD>
__global__ void __launch_bounds__(THREADS, 1)
force_sym_f32_kernel(const float* __restrict__ packed, const float* __restrict__ tile_mass,
                     const float* __restrict__ block_mass, float4* __restrict__ partial,
                     float4* __restrict__ partial_j, const int nb, const int d0, const int rows, const int first, const int64_t part_stride,
                     const int64_t n_padb, const float eps2f) {
    constexpr int NWARPS = THREADS / 32;
    constexpr int B = THREADS * IPT;
    constexpr int TPB = B / TJ;            // j-tiles per block
    constexpr int JP = kSymF32Jp;          // j-pairs a lane keeps in flight
    constexpr int CHUNKS = TJ / (64 * JP); // JP x 64 j-bodies (32 lanes x JP pairs) per systolic pass
    constexpr uint32_t TILE_BYTES = TJ * 16u;
    static_assert(B % TJ == 0 && TJ % (64 * JP) == 0 && TJ <= THREADS, "one thread per j-body in the tile reduction");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* tiles = reinterpret_cast<float*>(smem_raw);                                   // [STAGES][TJ*4]
    float2* jacc = reinterpret_cast<float2*>(smem_raw + STAGES * TILE_BYTES);            // [2][NWARPS][TJ/2][4]
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem_raw + STAGES * TILE_BYTES + 2 * NWARPS * (TJ / 2) * 32);
    uint64_t* empty_bar = full_bar + STAGES;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int I = blockIdx.x;
    const int S = gridDim.y, sidx = blockIdx.y;
    // The tiles of block I in this band: first the non-symmetric ones (own block, and for an even block count the
    // opposite block I + nb/2; they belong to the first band), then the symmetric partner tiles of blocks I+d0+1 ..
    // I+d0+rows (cyclic).  The S splits cut this ONE list evenly, so the one-sided tiles do not pile up on one CTA.
    // (A solve whose j-side rows do not fit the workspace at once is cut into bands of partner offsets.)
    const int n_ns = first ? TPB * ((nb > 1 && (nb & 1) == 0) ? 2 : 1) : 0;
    const int T = n_ns + rows * TPB;
    const int g0 = (int)(((int64_t)T * sidx) / S), g1 = (int)(((int64_t)T * (sidx + 1)) / S);
    const int nt = g1 - g0;
    auto tile_of = [&](int q) -> int {
        const int g = g0 + q;
        if (g < n_ns) return ((g < TPB ? I : (I + nb / 2) % nb)) * TPB + g % TPB;
        const int p = g - n_ns;
        return ((I + 1 + d0 + p / TPB) % nb) * TPB + p % TPB;
    };

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
            tma_load_1d(tiles + s * TJ * 4, packed + (size_t)tile_of(s) * TJ * 4, TILE_BYTES, &full_bar[s]);
        }
    }

    float2 nx[IPT], ny[IPT], nz[IPT], mi[IPT];
    float2 ax[IPT], ay[IPT], az[IPT], ap[IPT];
    // compensated outer sums (value, error) x (x, y, z, phi) per i-body: touched once per tile, so they live in shared
    // memory -- osum[q][k][tid], q = 0..7 -- and leave their 8 IPT registers to more i-bodies per thread
    float* osum = reinterpret_cast<float*>(empty_bar + STAGES);
    auto os = [&](int q, int k) -> float& { return osum[(q * IPT + k) * THREADS + tid]; };
    int iidx[IPT];
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const int i = I * B + k * THREADS + tid;
        iidx[k] = i;
        const float* q = packed + (size_t)(i >> 1) * 8 + (i & 1);
        const float xi = q[0], yi = q[2], zi = q[4], m = q[6];
        nx[k] = make_float2(-xi, -xi);
        ny[k] = make_float2(-yi, -yi);
        nz[k] = make_float2(-zi, -zi);
        mi[k] = make_float2(m, m);
        ax[k] = ay[k] = az[k] = ap[k] = make_float2(0.f, 0.f);
#pragma unroll
        for (int q = 0; q < 8; ++q) os(q, k) = 0.f;
    }
    const float2 eps2 = make_float2(eps2f, eps2f);
    const float bm = block_mass ? __ldg(block_mass + I) : __int_as_float(0x7fc00000);   // common mass of the own block
    const bool uni_i = bm == bm;
    const float kNoCommonMass = __int_as_float(0x7fc00000);
    float tm_next = (tile_mass && nt > 0) ? __ldg(tile_mass + tile_of(0)) : kNoCommonMass;
    int buf = 0;

    for (int t = 0; t < nt; ++t) {
        const int s = t % STAGES;
        const float tm = tm_next;
        if (tile_mass && t + 1 < nt) tm_next = __ldg(tile_mass + tile_of(t + 1));
        const int gt = tile_of(t);
        const int jbase = gt * TJ;
        mbar_wait(&full_bar[s], (uint32_t)(t / STAGES) & 1u);
        const float4* tp = reinterpret_cast<const float4*>(tiles + s * TJ * 4);
        const bool sym = g0 + t >= n_ns;
        const bool uni = (tm == tm) && (!sym || uni_i);
        if (!sym) {
            const bool diag = (MODE == MODE_FORCE_POT) && !GUARD && g0 + t < TPB;   // the own block holds j == i
            if (uni) {
                if (diag) sweep_tile<IPT, MODE, GUARD, true, true>(tp, TJ / 2, nx, ny, nz, ax, ay, az, ap, eps2, jbase, iidx);
                else sweep_tile<IPT, MODE, GUARD, false, true>(tp, TJ / 2, nx, ny, nz, ax, ay, az, ap, eps2, jbase, iidx);
            } else {
                if (diag) sweep_tile<IPT, MODE, GUARD, true, false>(tp, TJ / 2, nx, ny, nz, ax, ay, az, ap, eps2, jbase, iidx);
                else sweep_tile<IPT, MODE, GUARD, false, false>(tp, TJ / 2, nx, ny, nz, ax, ay, az, ap, eps2, jbase, iidx);
            }
        } else {
            float2* mine = jacc + ((size_t)(buf * NWARPS + warp) * (TJ / 2)) * 4;
#pragma unroll 1
            for (int c = 0; c < CHUNKS; ++c) {
                float2 xj[JP], yj[JP], zj[JP], mj[JP], fx[JP], fy[JP], fz[JP], fp[JP];
#pragma unroll
                for (int q = 0; q < JP; ++q) {
                    const float4 a = tp[2 * ((c * JP + q) * 32 + lane)];
                    const float4 b = tp[2 * ((c * JP + q) * 32 + lane) + 1];
                    xj[q] = make_float2(a.x, a.y); yj[q] = make_float2(a.z, a.w);
                    zj[q] = make_float2(b.x, b.y); mj[q] = make_float2(b.z, b.w);
                }
                if (uni)
                    sym_chunk<IPT, JP, MODE, GUARD, true>(xj, yj, zj, mj, nx, ny, nz, mi, ax, ay, az, ap, fx, fy, fz, fp,
                                                          eps2, lane);
                else
                    sym_chunk<IPT, JP, MODE, GUARD, false>(xj, yj, zj, mj, nx, ny, nz, mi, ax, ay, az, ap, fx, fy, fz, fp,
                                                           eps2, lane);
#pragma unroll
                for (int q = 0; q < JP; ++q) {
                    float4* o = reinterpret_cast<float4*>(mine + (size_t)((c * JP + q) * 32 + lane) * 4);
                    o[0] = make_float4(fx[q].x, fx[q].y, fy[q].x, fy[q].y);
                    o[1] = make_float4(fz[q].x, fz[q].y, (MODE == MODE_FORCE_POT) ? fp[q].x : 0.f,
                                       (MODE == MODE_FORCE_POT) ? fp[q].y : 0.f);
                }
            }
        }
        const float scale = uni ? tm : 1.0f;

        // release the stage, then (one tile late) refill the stage that held tile t-1 with tile t-1+STAGES
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[s]);
        if (tid == 0 && t >= 1 && t - 1 + STAGES < nt) {
            const int ps = (t - 1) % STAGES;
            mbar_wait(&empty_bar[ps], (uint32_t)((t - 1) / STAGES) & 1u);
            mbar_expect_tx(&full_bar[ps], TILE_BYTES);
            tma_load_1d(tiles + ps * TJ * 4, packed + (size_t)tile_of(t - 1 + STAGES) * TJ * 4, TILE_BYTES, &full_bar[ps]);
        }

        // i-side: fold the tile's packed partial sums into the compensated outer sums
#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            float v0 = os(0, k), e0 = os(1, k), v1 = os(2, k), e1 = os(3, k), v2 = os(4, k), e2 = os(5, k);
            comp_add(v0, e0, __fmul_rn(scale, __fadd_rn(ax[k].x, ax[k].y)));
            comp_add(v1, e1, __fmul_rn(scale, __fadd_rn(ay[k].x, ay[k].y)));
            comp_add(v2, e2, __fmul_rn(scale, __fadd_rn(az[k].x, az[k].y)));
            os(0, k) = v0; os(1, k) = e0; os(2, k) = v1; os(3, k) = e1; os(4, k) = v2; os(5, k) = e2;
            ax[k] = ay[k] = az[k] = make_float2(0.f, 0.f);
            if (MODE == MODE_FORCE_POT) {
                float v3 = os(6, k), e3 = os(7, k);
                comp_add(v3, e3, __fmul_rn(scale, __fadd_rn(ap[k].x, ap[k].y)));
                os(6, k) = v3; os(7, k) = e3;
                ap[k] = make_float2(0.f, 0.f);
            }
        }

        // j-side: the 8 warps' sums for the TJ bodies of this tile meet here, in warp order; one thread per j-body
        if (sym) {
            __syncthreads();
            const float2* base = jacc + ((size_t)(buf * NWARPS) * (TJ / 2)) * 4 + (size_t)((tid < TJ ? tid : 0) >> 1) * 4;
            const int h = tid & 1;
            float fx = 0.f, fy = 0.f, fz = 0.f, fp = 0.f;
#pragma unroll
            for (int w = 0; w < NWARPS; ++w) {
                const float2* e = base + (size_t)w * (TJ / 2) * 4;
                fx = __fadd_rn(fx, h ? e[0].y : e[0].x);
                fy = __fadd_rn(fy, h ? e[1].y : e[1].x);
                fz = __fadd_rn(fz, h ? e[2].y : e[2].x);
                if (MODE == MODE_FORCE_POT) fp = __fadd_rn(fp, h ? e[3].y : e[3].x);
            }
            const float sj = uni ? bm : 1.0f;
            const int row = (g0 + t - n_ns) / TPB;                       // d - 1
            if (tid < TJ)
                partial_j[(size_t)row * n_padb + jbase + tid] =
                    make_float4(-__fmul_rn(sj, fx), -__fmul_rn(sj, fy), -__fmul_rn(sj, fz), __fmul_rn(sj, fp));
            buf ^= 1;   // the other buffer is free: every thread passed the barrier of the tile before
        }
    }

#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        float4 o;
        o.x = __fadd_rn(os(0, k), os(1, k));
        o.y = __fadd_rn(os(2, k), os(3, k));
        o.z = __fadd_rn(os(4, k), os(5, k));
        o.w = (MODE == MODE_FORCE_POT) ? __fadd_rn(os(6, k), os(7, k)) : 0.f;
        partial[(size_t)sidx * part_stride + iidx[k]] = o;
    }
}

template <int FINE, int MODE, bool GUARD>
int launch_mg(const Plan& p, const float* packed, const float* tile_mass, const float* block_mass, float4* partial,
              float4* partial_j, float4* acc_j, float eps2, cudaStream_t st) {
    constexpr KernelShape K = FINE ? kShapeF32SymFine : kShapeF32Sym;
    // j-tile ring + two j-side reduction buffers + mbarriers + the outer sums
    constexpr size_t smem = (size_t)K.stages * K.tile_j * 16 + 2 * (K.threads / 32) * (K.tile_j / 2) * 32 + 2 * K.stages * 8 +
                            (size_t)8 * K.ipt * K.threads * 4;
    auto kern = force_sym_f32_kernel<K.threads, K.ipt, K.tile_j, K.stages, MODE, GUARD>;
    PP_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));   // > 48 KB: opt-in
    dim3 grid(p.n_iblocks, p.split);
    // bands of partner offsets (one band unless the j-side rows exceed the workspace cap): every band reuses BOTH the
    // i-side partials and the j-side rows; in between, fold_rows (update.cu) adds them -- the S i-side partials first,
    // then the band's rows, all in fixed order -- into the running TwoSum sums acc_j that finalize reads at the end
    for (int b = 0; b < p.sym_bands; ++b) {
        const int d0 = b * p.sym_rows, rows = std::min(p.sym_rows, p.sym_h - d0);
        kern<<<grid, K.threads, smem, st>>>(packed, tile_mass, block_mass, partial, partial_j, p.n_iblocks, d0, rows,
                                            b == 0, p.part_stride, p.part_stride, eps2);
        count_launch();
        PP_CUDA(cudaGetLastError());
        if (p.sym_bands > 1) {
            PP_TRY_RC(launch_fold_rows(partial, p.split, p.part_stride, acc_j, b == 0, st));
            PP_TRY_RC(launch_fold_rows(partial_j, rows, p.part_stride, acc_j, false, st));
        }
    }
    return PP_OK;
}

template <int FINE>
int launch_fine(const Plan& p, const float* packed, const float* tile_mass, const float* block_mass, float4* partial,
                float4* partial_j, float4* acc_j, float eps2, bool guard, int mode, cudaStream_t st) {
    if (mode == MODE_FORCE)
        return guard ? launch_mg<FINE, MODE_FORCE, true>(p, packed, tile_mass, block_mass, partial, partial_j, acc_j, eps2, st)
                     : launch_mg<FINE, MODE_FORCE, false>(p, packed, tile_mass, block_mass, partial, partial_j, acc_j, eps2, st);
    return guard ? launch_mg<FINE, MODE_FORCE_POT, true>(p, packed, tile_mass, block_mass, partial, partial_j, acc_j, eps2, st)
                 : launch_mg<FINE, MODE_FORCE_POT, false>(p, packed, tile_mass, block_mass, partial, partial_j, acc_j, eps2, st);
}

}  // namespace

int launch_force_sym_f32(const Plan& p, const float* packed, const float* tile_mass, const float* block_mass,
                         float4* partial, float4* partial_j, float4* acc_j, double delta, int mode, cudaStream_t st) {
    constexpr KernelShape K = kShapeF32Sym, F = kShapeF32SymFine;
    const bool fine = p.tile_j == F.tile_j;
    if (!p.sym || p.threads != K.threads || p.ipt != K.ipt || (p.tile_j != K.tile_j && !fine) || p.i_begin != 0 ||
        (mode != MODE_FORCE && mode != MODE_FORCE_POT)) {
        set_error("launch_force_sym_f32: not a symmetric FP32 plan");
        return PP_EINVAL;
    }
    const float eps2 = (float)(delta * delta);
    const bool guard = !(eps2 >= kTinyR2F32);
    return fine ? launch_fine<1>(p, packed, tile_mass, block_mass, partial, partial_j, acc_j, eps2, guard, mode, st)
                : launch_fine<0>(p, packed, tile_mass, block_mass, partial, partial_j, acc_j, eps2, guard, mode, st);
}

}  // namespace ppgrav
