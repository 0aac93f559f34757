// force_f64_common.cuh -- device helpers shared by the FP64 pair sweeps (force_f64.cu: every ordered pair; force_sym_f64.cu:
// every unordered pair once).  Included by those two translation units only.
#pragma once

#include "ppgrav_internal.h"

namespace ppgrav {
namespace {

// as kTinyR2F32 in force_f32.cu: below this softened squared distance a pair contributes nothing (guarded kernels,
// selected when delta^2 < kTinyR2F64); (1e-200)^{-3/2} = 1e300 is still finite
constexpr double kTinyR2F64 = 1e-200;

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
            if (GUARD) y = r2 > kTinyR2F64 ? y : 0.0;         // delta ~ 0: (near-)zero-distance pairs contribute nothing
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

}  // namespace
}  // namespace ppgrav
