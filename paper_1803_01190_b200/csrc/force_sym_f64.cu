// force_sym_f64.cu -- FP64 all-pairs gravity sweep that evaluates every UNORDERED pair once (sm_100a).
//
// The FP64 twin of force_sym_f32.cu (read its header for the block-pair decomposition, the systolic rotation of the
// j-bodies through the lanes of a warp, and the fixed-order j-side reduction).  What differs: one j-body per lane (no
// packed FP64 arithmetic exists), 32 j-bodies per systolic pass, and the
// RSQ64H-seed-plus-one-cubic-correction reciprocal square root of force_f64.cu.  FP64-pipe operations per evaluation,
// which serves the two ordered pairs (i <- j) and (j <- i): 18 force-only (15 one-sided per ORDERED pair), 21 with the
// potential (17), two more when the masses are not common to block and tile -- 9 / 10.5 instead of 15 / 17 per pair
// interaction.
#ifndef PP_SYM64_ORDER
#define PP_SYM64_ORDER 0
#endif
#include "force_f64_common.cuh"
#include <algorithm>

#include "tma_ring.cuh"

namespace ppgrav {
namespace {

__device__ __forceinline__ double rotd(const double v, const int src) {
    const int lo = __shfl_sync(0xffffffffu, __double2loint(v), src);
    const int hi = __shfl_sync(0xffffffffu, __double2hiint(v), src);
    return __hiloint2double(hi, lo);
}

template <int IPT, int MODE, bool GUARD, bool UNI>
__device__ __forceinline__ void sym_chunk(double xj, double yj, double zj, double mj, const double (&xi)[IPT],
                                          const double (&yi)[IPT], const double (&zi)[IPT], const double (&mi)[IPT],
                                          double (&ax)[IPT], double (&ay)[IPT], double (&az)[IPT], double (&ap)[IPT],
                                          double& fx, double& fy, double& fz, double& fp, const double eps2,
                                          const int lane) {
    fx = fy = fz = fp = 0.0;
    const int src = (lane + 1) & 31;
#pragma unroll kSymF64Unroll
    for (int step = 0; step < 32; ++step) {
#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            const double dx = xj - xi[k];                     // r_j - r_i
            const double dy = yj - yi[k];
            const double dz = zj - zi[k];
            double r2 = fma(dx, dx, eps2);                    // |r_i - r_j|^2 + delta^2
            r2 = fma(dy, dy, r2);
            r2 = fma(dz, dz, r2);
            double y = rsqrt64h(r2);
            if (GUARD) y = r2 > kTinyR2F64 ? y : 0.0;
            const double t = y * y;
            const double e = fma(-r2, t, 1.0);                // 1 - x y^2
            double s;                                         // x^{-3/2}
            if (MODE == MODE_FORCE) {
                const double p = fma(e, 1.875, 1.5);
                const double w = y * t;
                s = fma(p, w * e, w);
            } else {
                const double q = fma(e, 0.375, 0.5);
                const double yy = fma(q, y * e, y);           // x^{-1/2} to full precision
                s = yy * (yy * yy);
                ap[k] = UNI ? ap[k] + yy : fma(mj, yy, ap[k]);
                fp = UNI ? fp + yy : fma(mi[k], yy, fp);
            }
            const double si = UNI ? s : mj * s;               // pull of j on i:  m_j x^{-3/2} (r_j - r_i)
            const double sj = UNI ? s : mi[k] * s;            // pull of i on j: -m_i x^{-3/2} (r_j - r_i)
#if PP_SYM64_ORDER == 1   // i-side and j-side update of one component back to back: they share two operands
            ax[k] = fma(si, dx, ax[k]);
            fx = fma(sj, dx, fx);
            ay[k] = fma(si, dy, ay[k]);
            fy = fma(sj, dy, fy);
            az[k] = fma(si, dz, az[k]);
            fz = fma(sj, dz, fz);
#else
            ax[k] = fma(si, dx, ax[k]);
            ay[k] = fma(si, dy, ay[k]);
            az[k] = fma(si, dz, az[k]);
            fx = fma(sj, dx, fx);
            fy = fma(sj, dy, fy);
            fz = fma(sj, dz, fz);
#endif
        }
        xj = rotd(xj, src); yj = rotd(yj, src); zj = rotd(zj, src);
        if (!UNI) mj = rotd(mj, src);
        fx = rotd(fx, src); fy = rotd(fy, src); fz = rotd(fz, src);
        if (MODE == MODE_FORCE_POT) fp = rotd(fp, src);
    }   // after 32 rotations every j-body is back in the lane it started in
}

template <int THREADS, int IPT, int TJ, int STAGES, int MODE, bool GUARD>
__global__ void __launch_bounds__(THREADS, 1)
force_sym_f64_kernel(const double* __restrict__ packed, const double* __restrict__ tile_mass,
                     const double* __restrict__ block_mass, double4* __restrict__ partial,
                     double4* __restrict__ partial_j, const int nb, const int d0, const int rows, const int first, const int64_t part_stride,
                     const int64_t n_padb, const double eps2) {
    constexpr int NWARPS = THREADS / 32;
    constexpr int B = THREADS * IPT;
    constexpr int TPB = B / TJ;
    constexpr int CHUNKS = TJ / 32;
    constexpr uint32_t TILE_BYTES = TJ * 32u;
    static_assert(B % TJ == 0 && TJ % 32 == 0 && TJ <= THREADS, "one thread per j-body in the tile reduction");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* tiles = reinterpret_cast<double*>(smem_raw);                                  // [STAGES][TJ*4]
    double4* jacc = reinterpret_cast<double4*>(smem_raw + STAGES * TILE_BYTES);           // [2][NWARPS][TJ]
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem_raw + STAGES * TILE_BYTES + 2 * NWARPS * TJ * 32);
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

    double xi[IPT], yi[IPT], zi[IPT], mi[IPT];
    double ax[IPT], ay[IPT], az[IPT], ap[IPT];
    // outer sums (x, y, z, phi) per i-body: touched once per tile, so they live in shared memory (osum[q][k][tid])
    double* osum = reinterpret_cast<double*>(empty_bar + STAGES);
    auto os = [&](int q, int k) -> double& { return osum[(q * IPT + k) * THREADS + tid]; };
    int iidx[IPT];
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const int i = I * B + k * THREADS + tid;
        iidx[k] = i;
        const double4 q = reinterpret_cast<const double4*>(packed)[i];
        xi[k] = q.x; yi[k] = q.y; zi[k] = q.z; mi[k] = q.w;
        ax[k] = ay[k] = az[k] = ap[k] = 0.0;
        os(0, k) = os(1, k) = os(2, k) = os(3, k) = 0.0;
    }
    const double kNoCommonMass = __longlong_as_double(0x7ff8000000000000ll);
    const double bm = block_mass ? __ldg(block_mass + I) : kNoCommonMass;
    const bool uni_i = bm == bm;
    double tm_next = (tile_mass && nt > 0) ? __ldg(tile_mass + tile_of(0)) : kNoCommonMass;
    int buf = 0;

    for (int t = 0; t < nt; ++t) {
        const int s = t % STAGES;
        const double tm = tm_next;
        if (tile_mass && t + 1 < nt) tm_next = __ldg(tile_mass + tile_of(t + 1));
        const int gt = tile_of(t);
        const int jbase = gt * TJ;
        mbar_wait(&full_bar[s], (uint32_t)(t / STAGES) & 1u);
        const double4* tp = reinterpret_cast<const double4*>(tiles + s * TJ * 4);
        const bool sym = g0 + t >= n_ns;
        const bool uni = (tm == tm) && (!sym || uni_i);
        if (!sym) {
            const bool diag = (MODE == MODE_FORCE_POT) && !GUARD && g0 + t < TPB;
            if (uni) {
                if (diag) sweep_tile<IPT, MODE, GUARD, true, true>(tp, TJ, xi, yi, zi, ax, ay, az, ap, eps2, jbase, iidx);
                else sweep_tile<IPT, MODE, GUARD, false, true>(tp, TJ, xi, yi, zi, ax, ay, az, ap, eps2, jbase, iidx);
            } else {
                if (diag) sweep_tile<IPT, MODE, GUARD, true, false>(tp, TJ, xi, yi, zi, ax, ay, az, ap, eps2, jbase, iidx);
                else sweep_tile<IPT, MODE, GUARD, false, false>(tp, TJ, xi, yi, zi, ax, ay, az, ap, eps2, jbase, iidx);
            }
        } else {
            double4* mine = jacc + (size_t)(buf * NWARPS + warp) * TJ;
#pragma unroll 1
            for (int c = 0; c < CHUNKS; ++c) {
                const double4 b = tp[c * 32 + lane];
                double fx, fy, fz, fp;
                if (uni)
                    sym_chunk<IPT, MODE, GUARD, true>(b.x, b.y, b.z, b.w, xi, yi, zi, mi, ax, ay, az, ap, fx, fy, fz, fp,
                                                      eps2, lane);
                else
                    sym_chunk<IPT, MODE, GUARD, false>(b.x, b.y, b.z, b.w, xi, yi, zi, mi, ax, ay, az, ap, fx, fy, fz, fp,
                                                       eps2, lane);
                mine[c * 32 + lane] = make_double4(fx, fy, fz, (MODE == MODE_FORCE_POT) ? fp : 0.0);
            }
        }
        const double scale = uni ? tm : 1.0;

        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[s]);
        if (tid == 0 && t >= 1 && t - 1 + STAGES < nt) {
            const int ps = (t - 1) % STAGES;
            mbar_wait(&empty_bar[ps], (uint32_t)((t - 1) / STAGES) & 1u);
            mbar_expect_tx(&full_bar[ps], TILE_BYTES);
            tma_load_1d(tiles + ps * TJ * 4, packed + (size_t)tile_of(t - 1 + STAGES) * TJ * 4, TILE_BYTES, &full_bar[ps]);
        }

#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            os(0, k) = fma(scale, ax[k], os(0, k));
            os(1, k) = fma(scale, ay[k], os(1, k));
            os(2, k) = fma(scale, az[k], os(2, k));
            ax[k] = ay[k] = az[k] = 0.0;
            if (MODE == MODE_FORCE_POT) { os(3, k) = fma(scale, ap[k], os(3, k)); ap[k] = 0.0; }
        }

        if (sym) {   // j-side: the 8 warps' sums for the TJ bodies of this tile, added in warp order, one thread per body
            __syncthreads();
            const double4* base = jacc + (size_t)(buf * NWARPS) * TJ + (tid < TJ ? tid : 0);
            double fx = 0.0, fy = 0.0, fz = 0.0, fp = 0.0;
#pragma unroll
            for (int w = 0; w < NWARPS; ++w) {
                const double4 e = base[(size_t)w * TJ];
                fx += e.x; fy += e.y; fz += e.z;
                if (MODE == MODE_FORCE_POT) fp += e.w;
            }
            const double sj = uni ? bm : 1.0;
            const int row = (g0 + t - n_ns) / TPB;                       // d - 1
            if (tid < TJ)
                partial_j[(size_t)row * n_padb + jbase + tid] = make_double4(-(sj * fx), -(sj * fy), -(sj * fz), sj * fp);
            buf ^= 1;
        }
    }

#pragma unroll
    for (int k = 0; k < IPT; ++k)
        partial[(size_t)sidx * part_stride + iidx[k]] =
            make_double4(os(0, k), os(1, k), os(2, k), (MODE == MODE_FORCE_POT) ? os(3, k) : 0.0);
}

template <int FINE, int MODE, bool GUARD>
int launch_mg(const Plan& p, const double* packed, const double* tile_mass, const double* block_mass, double4* partial,
              double4* partial_j, double4* acc_j, double eps2, cudaStream_t st) {
    constexpr KernelShape K = FINE ? kShapeF64SymFine : kShapeF64Sym;
    // j-tile ring + two j-side reduction buffers + mbarriers + the outer sums
    constexpr size_t smem = (size_t)K.stages * K.tile_j * 32 + 2 * (K.threads / 32) * K.tile_j * 32 + 2 * K.stages * 8 +
                            (size_t)4 * K.ipt * K.threads * 8;
    static_assert(smem <= 227 * 1024, "shared memory of the symmetric FP64 sweep");
    auto kern = force_sym_f64_kernel<K.threads, K.ipt, K.tile_j, K.stages, MODE, GUARD>;
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
int launch_fine(const Plan& p, const double* packed, const double* tile_mass, const double* block_mass, double4* partial,
                double4* partial_j, double4* acc_j, double eps2, bool guard, int mode, cudaStream_t st) {
    if (mode == MODE_FORCE)
        return guard ? launch_mg<FINE, MODE_FORCE, true>(p, packed, tile_mass, block_mass, partial, partial_j, acc_j, eps2, st)
                     : launch_mg<FINE, MODE_FORCE, false>(p, packed, tile_mass, block_mass, partial, partial_j, acc_j, eps2, st);
    return guard ? launch_mg<FINE, MODE_FORCE_POT, true>(p, packed, tile_mass, block_mass, partial, partial_j, acc_j, eps2, st)
                 : launch_mg<FINE, MODE_FORCE_POT, false>(p, packed, tile_mass, block_mass, partial, partial_j, acc_j, eps2, st);
}

}  // namespace

int launch_force_sym_f64(const Plan& p, const double* packed, const double* tile_mass, const double* block_mass,
                         double4* partial, double4* partial_j, double4* acc_j, double delta, int mode, cudaStream_t st) {
    constexpr KernelShape K = kShapeF64Sym, F = kShapeF64SymFine;
    const bool fine = p.tile_j == F.tile_j;
    if (!p.sym || p.threads != K.threads || p.ipt != K.ipt || (p.tile_j != K.tile_j && !fine) || p.i_begin != 0 ||
        (mode != MODE_FORCE && mode != MODE_FORCE_POT)) {
        set_error("launch_force_sym_f64: not a symmetric FP64 plan");
        return PP_EINVAL;
    }
    const double eps2 = delta * delta;
    const bool guard = !(eps2 >= kTinyR2F64);
    return fine ? launch_fine<1>(p, packed, tile_mass, block_mass, partial, partial_j, acc_j, eps2, guard, mode, st)
                : launch_fine<0>(p, packed, tile_mass, block_mass, partial, partial_j, acc_j, eps2, guard, mode, st);
}

}  // namespace ppgrav
