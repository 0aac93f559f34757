// force_f32_common.cuh -- device helpers shared by the FP32 pair sweeps (force_f32.cu: every ordered pair; force_sym_f32.cu:
// every unordered pair once).  Included by those two translation units only.
#pragma once

#include "ppgrav_internal.h"

namespace ppgrav {
namespace {

// Softened squared distances below this select / trigger the guarded path: w^3 = r2^{-3/2} must stay finite in FP32
// (1e-20^{-3/2} = 1e30 leaves room for m_j up to ~1e8).  delta^2 >= kTinyR2F32 runs the unguarded kernels, in which
// the j == i term is exactly 0 x finite; below it (delta = 0 included) every pair with r^2 + delta^2 <= kTinyR2F32 --
// j == i, coincident bodies, padding -- contributes nothing (include/ppgrav.h, reading R2).
constexpr float kTinyR2F32 = 1e-20f;

__device__ __forceinline__ float rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// s + c += t with the rounding error of the addition captured in c (Knuth TwoSum; never contracted or reassociated)
__device__ __forceinline__ void comp_add(float& s, float& c, float t) {
    const float n = __fadd_rn(s, t);
    const float bp = __fsub_rn(n, s);
    const float e = __fadd_rn(__fsub_rn(s, __fsub_rn(n, bp)), __fsub_rn(t, bp));
    s = n;
    c = __fadd_rn(c, e);
}

template <int IPT, int MODE, bool GUARD, bool DIAG, bool UNI>
__device__ __forceinline__ void sweep_tile(const float4* __restrict__ tp, const int npairs, const float2 (&nx)[IPT],
                                           const float2 (&ny)[IPT], const float2 (&nz)[IPT], float2 (&ax)[IPT],
                                           float2 (&ay)[IPT], float2 (&az)[IPT], float2 (&ap)[IPT], const float2 eps2,
                                           const int jbase, const int (&iidx)[IPT]) {
#pragma unroll kF32Unroll
    for (int p = 0; p < npairs; ++p) {
        const float4 a = tp[2 * p];
        const float4 b = tp[2 * p + 1];
        const float2 xj = make_float2(a.x, a.y), yj = make_float2(a.z, a.w);
        const float2 zj = make_float2(b.x, b.y), mj = make_float2(b.z, b.w);
#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            const float2 dx = __fadd2_rn(xj, nx[k]);          // r_j - r_i (two j-bodies)
            const float2 dy = __fadd2_rn(yj, ny[k]);
            const float2 dz = __fadd2_rn(zj, nz[k]);
            float2 r2 = __ffma2_rn(dx, dx, eps2);             // |r_i - r_j|^2 + delta^2
            r2 = __ffma2_rn(dy, dy, r2);
            r2 = __ffma2_rn(dz, dz, r2);
            float2 w;
            w.x = rsqrt_approx(r2.x);
            w.y = rsqrt_approx(r2.y);
            if (GUARD) {                                      // delta ~ 0: (near-)zero-distance pairs contribute nothing
                w.x = r2.x > kTinyR2F32 ? w.x : 0.f;
                w.y = r2.y > kTinyR2F32 ? w.y : 0.f;
            }
            const float2 w2 = __fmul2_rn(w, w);
            float2 mw = UNI ? w : __fmul2_rn(mj, w);          // equal-mass tile: m_j is applied in the fold
            const float2 s = __fmul2_rn(mw, w2);              // m_j / (r^2 + delta^2)^{3/2}
            ax[k] = __ffma2_rn(s, dx, ax[k]);
            ay[k] = __ffma2_rn(s, dy, ay[k]);
            az[k] = __ffma2_rn(s, dz, az[k]);
            if (MODE == MODE_FORCE_POT) {
                if (DIAG) {                                   // tile overlaps this CTA's own bodies: drop j == i
                    const int j0 = jbase + 2 * p;
                    if (j0 == iidx[k]) mw.x = 0.f;
                    if (j0 + 1 == iidx[k]) mw.y = 0.f;
                }
                ap[k] = __fadd2_rn(ap[k], mw);                // m_j / (r^2 + delta^2)^{1/2}
            }
        }
    }
}

}  // namespace
}  // namespace ppgrav
