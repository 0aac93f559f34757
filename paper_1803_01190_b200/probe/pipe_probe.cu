// pipe_probe.cu -- MEASUREMENT TOOLING, NOT PART OF libppgrav: pipe-throughput microbenchmarks behind the ALU roofline
// denominators (profiles/r1_pipe_probes.md).  Built by paper_1803_01190_b200/build.py into its own
// libppprobe.so (one C entry point, pp_probe_pipe, below); nothing in the library, the binding, the tests of the hot
// path or bench.py's timed region links or calls it.
//
// The force kernels are bound by the FP32 / FP64 pipes, not by HBM or tensor cores, and MEASURED_PEAKS.json holds
// no CUDA-core peak.  Each probe runs a long, register-only dependent-chain loop (8 independent chains per thread,
// 32 warps per SM) of one instruction kind and reports lane-operations per clock per SM, with the SM clock taken
// from clock64()/globaltimer inside the kernel.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

constexpr int kThreads = 256;
constexpr int kCtasPerSm = 4;
constexpr int kChains = 8;
constexpr int kInner = 8;

__device__ __forceinline__ uint64_t globaltimer_ns() {
    uint64_t t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ float rsqrt_f32(float x) {
    float y;
    asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ double rsqrt_f64h(double x) {
    double y;
    asm volatile("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}

// KIND: 0 FFMA, 1 FFMA2, 2 DFMA, 3 MUFU.RSQ, 4 MUFU.RSQ64H, 5 the force kernel's mix (12 FFMA2 : 2 MUFU.RSQ = two pairs)
// 6-8 ask whether the idle FP64 pipe could carry extra i-bodies of an FP32 sweep:
//   6 two FFMA2 : one DFMA, every instruction a = a*b + c with loop-constant b, c (one register operand read each)
//   7 FFMA2 alone, three distinct rotating register operands per instruction (what a real pair loop reads)
//   8 two FFMA2 : one DFMA, three distinct rotating register operands per instruction
template <int KIND>
__global__ void __launch_bounds__(kThreads, kCtasPerSm)
probe_kernel(int64_t iters, float seed, float* __restrict__ sink, uint64_t* __restrict__ clk) {
    const uint64_t t0 = globaltimer_ns();
    const long long c0 = clock64();
    float acc = 0.f;
    if (KIND == 0) {
        float a[kChains];
        const float b = 1.0f + (seed + threadIdx.x) * 1e-9f, c = (seed + threadIdx.x) * 1e-9f;   // per-thread: 3-register form
#pragma unroll
        for (int k = 0; k < kChains; ++k) a[k] = seed + k + threadIdx.x;
        for (int64_t it = 0; it < iters; ++it)
#pragma unroll
            for (int u = 0; u < kInner; ++u)
#pragma unroll
                for (int k = 0; k < kChains; ++k) a[k] = __fmaf_rn(a[k], b, c);
#pragma unroll
        for (int k = 0; k < kChains; ++k) acc += a[k];
    } else if (KIND == 1) {
        float2 a[kChains];
        const float tx = (seed + threadIdx.x) * 1e-9f;
        const float2 b = make_float2(1.0f + tx, 1.0f - tx), c = make_float2(tx, seed + tx);
#pragma unroll
        for (int k = 0; k < kChains; ++k) a[k] = make_float2(seed + k, seed + threadIdx.x);
        for (int64_t it = 0; it < iters; ++it)
#pragma unroll
            for (int u = 0; u < kInner; ++u)
#pragma unroll
                for (int k = 0; k < kChains; ++k) a[k] = __ffma2_rn(a[k], b, c);
#pragma unroll
        for (int k = 0; k < kChains; ++k) acc += a[k].x + a[k].y;
    } else if (KIND == 2) {
        double a[kChains];
        const double b = 1.0 + (seed + threadIdx.x) * 1e-12, c = (seed + threadIdx.x) * 1e-12;
#pragma unroll
        for (int k = 0; k < kChains; ++k) a[k] = seed + k + threadIdx.x;
        for (int64_t it = 0; it < iters; ++it)
#pragma unroll
            for (int u = 0; u < kInner; ++u)
#pragma unroll
                for (int k = 0; k < kChains; ++k) a[k] = __fma_rn(a[k], b, c);
#pragma unroll
        for (int k = 0; k < kChains; ++k) acc += (float)a[k];
    } else if (KIND == 3) {
        float a[kChains];
#pragma unroll
        for (int k = 0; k < kChains; ++k) a[k] = 1.0f + seed + k + threadIdx.x;
        for (int64_t it = 0; it < iters; ++it)
#pragma unroll
            for (int u = 0; u < kInner; ++u)
#pragma unroll
                for (int k = 0; k < kChains; ++k) a[k] = rsqrt_f32(a[k]);
#pragma unroll
        for (int k = 0; k < kChains; ++k) acc += a[k];
    } else if (KIND == 4) {
        double a[kChains];
#pragma unroll
        for (int k = 0; k < kChains; ++k) a[k] = 1.0 + seed + k + threadIdx.x;
        for (int64_t it = 0; it < iters; ++it)
#pragma unroll
            for (int u = 0; u < kInner; ++u)
#pragma unroll
                for (int k = 0; k < kChains; ++k) a[k] = rsqrt_f64h(a[k]);
#pragma unroll
        for (int k = 0; k < kChains; ++k) acc += (float)a[k];
    } else if (KIND == 6) {
        float2 a[kChains];
        double d[kChains / 2];
        const float tx = (seed + threadIdx.x) * 1e-9f;
        const float2 b = make_float2(1.0f + tx, 1.0f - tx), c = make_float2(tx, seed + tx);
        const double bd = 1.0 + tx, cd = tx;
#pragma unroll
        for (int k = 0; k < kChains; ++k) a[k] = make_float2(seed + k, seed + threadIdx.x);
#pragma unroll
        for (int k = 0; k < kChains / 2; ++k) d[k] = seed + k;
        for (int64_t it = 0; it < iters; ++it)
#pragma unroll
            for (int u = 0; u < kInner; ++u)
#pragma unroll
                for (int k = 0; k < kChains / 2; ++k) {
                    a[2 * k] = __ffma2_rn(a[2 * k], b, c);
                    d[k] = __fma_rn(d[k], bd, cd);
                    a[2 * k + 1] = __ffma2_rn(a[2 * k + 1], b, c);
                }
#pragma unroll
        for (int k = 0; k < kChains; ++k) acc += a[k].x + a[k].y;
#pragma unroll
        for (int k = 0; k < kChains / 2; ++k) acc += (float)d[k];
    } else if (KIND == 7 || KIND == 8) {
        float2 a[kChains], x[kChains], y[kChains];
        double d[kChains / 2], xd[kChains / 2], yd[kChains / 2];
        const float tx = (seed + threadIdx.x) * 1e-9f;
#pragma unroll
        for (int k = 0; k < kChains; ++k) {
            a[k] = make_float2(seed + k, seed + threadIdx.x);
            x[k] = make_float2(1e-3f * k + tx, tx);
            y[k] = make_float2(tx + k, 1.f + tx);
        }
#pragma unroll
        for (int k = 0; k < kChains / 2; ++k) { d[k] = seed + k; xd[k] = 1e-3 * k + tx; yd[k] = tx + k; }
        for (int64_t it = 0; it < iters; ++it)
#pragma unroll
            for (int u = 0; u < kInner; ++u)
#pragma unroll
                for (int k = 0; k < kChains / 2; ++k) {
                    a[2 * k] = __ffma2_rn(x[(2 * k + u) % kChains], y[(2 * k + 3 + u) % kChains], a[2 * k]);
                    if (KIND == 8)
                        d[k] = __fma_rn(xd[(k + u) % (kChains / 2)], yd[(k + 1 + u) % (kChains / 2)], d[k]);
                    a[2 * k + 1] = __ffma2_rn(x[(2 * k + 1 + u) % kChains], y[(2 * k + 4 + u) % kChains], a[2 * k + 1]);
                }
#pragma unroll
        for (int k = 0; k < kChains; ++k) acc += a[k].x + a[k].y + x[k].x + y[k].y;
#pragma unroll
        for (int k = 0; k < kChains / 2; ++k) acc += (float)(d[k] + xd[k] + yd[k]);
    } else {
        float2 a[kChains];
        const float tx = (seed + threadIdx.x) * 1e-9f;
        const float2 b = make_float2(1.0f + tx, 1.0f - tx), c = make_float2(1.0f + tx, 1.0f + seed);
#pragma unroll
        for (int k = 0; k < kChains; ++k) a[k] = make_float2(1.0f + seed + k, 1.0f + threadIdx.x);
        for (int64_t it = 0; it < iters; ++it)
#pragma unroll
            for (int u = 0; u < kInner; ++u)
#pragma unroll
                for (int k = 0; k < kChains; ++k) {
                    float2 r = a[k];
#pragma unroll
                    for (int f = 0; f < 12; ++f) r = __ffma2_rn(r, b, c);
                    a[k] = make_float2(rsqrt_f32(r.x), rsqrt_f32(r.y));
                }
#pragma unroll
        for (int k = 0; k < kChains; ++k) acc += a[k].x + a[k].y;
    }
    const long long c1 = clock64();
    const uint64_t t1 = globaltimer_ns();
    if (acc == 123.456f) sink[0] = acc;   // keeps the chains alive; practically never true
    if (threadIdx.x == 0) {
        clk[2 * blockIdx.x] = (uint64_t)(c1 - c0);
        clk[2 * blockIdx.x + 1] = t1 - t0;
    }
}

template <int KIND>
void launch(int grid, int64_t iters, float* sink, uint64_t* clk) {
    probe_kernel<KIND><<<grid, kThreads>>>(iters, 0.5f, sink, clk);
}

}  // namespace

// kind: 0 FFMA, 1 FFMA2 (packed f32x2), 2 DFMA, 3 MUFU.RSQ, 4 MUFU.RSQ64H, 5 FFMA2+MUFU in the force kernel's mix (12 : 2),
//       6 two FFMA2 : one DFMA with loop-constant multiplier/addend (do the FP32 and FP64 pipes overlap?),
//       7 FFMA2 with three distinct register operands, 8 as 6 with three distinct register operands each
// out4 (host) = { seconds, lane-operations executed, SM clock in MHz during the run, lane-ops/clk/SM }; kinds 6-8
// count the FFMA2 lanes only.  Synchronous.  Returns 0, -1 (bad argument) or -2 (CUDA error).
extern "C" int pp_probe_pipe(int kind, int64_t iters, double* out4) {
    if (!out4 || kind < 0 || kind > 8 || iters < 1) return -1;
#define PROBE_CUDA(call) do { if ((call) != cudaSuccess) { cudaGetLastError(); return -2; } } while (0)
    int dev = 0, sm_count = 0;
    PROBE_CUDA(cudaGetDevice(&dev));
    PROBE_CUDA(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev));
    const int grid = sm_count * kCtasPerSm;
    float* sink = nullptr;
    uint64_t* clk = nullptr;
    PROBE_CUDA(cudaMalloc(&sink, 4));
    PROBE_CUDA(cudaMalloc(&clk, sizeof(uint64_t) * 2 * grid));
    cudaEvent_t e0, e1;
    PROBE_CUDA(cudaEventCreate(&e0));
    PROBE_CUDA(cudaEventCreate(&e1));
    float ms = 0.f;
    for (int rep = 0; rep < 2; ++rep) {   // first repetition warms up clocks and the instruction cache
        PROBE_CUDA(cudaEventRecord(e0));
        switch (kind) {
            case 0: launch<0>(grid, iters, sink, clk); break;
            case 1: launch<1>(grid, iters, sink, clk); break;
            case 2: launch<2>(grid, iters, sink, clk); break;
            case 3: launch<3>(grid, iters, sink, clk); break;
            case 4: launch<4>(grid, iters, sink, clk); break;
            case 5: launch<5>(grid, iters, sink, clk); break;
            case 6: launch<6>(grid, iters, sink, clk); break;
            case 7: launch<7>(grid, iters, sink, clk); break;
            default: launch<8>(grid, iters, sink, clk); break;
        }
        PROBE_CUDA(cudaGetLastError());
        PROBE_CUDA(cudaEventRecord(e1));
        PROBE_CUDA(cudaEventSynchronize(e1));
        PROBE_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    }
    uint64_t h[2];
    PROBE_CUDA(cudaMemcpy(h, clk, sizeof(h), cudaMemcpyDeviceToHost));
#undef PROBE_CUDA
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    cudaFree(clk);
    // lane-operations per chain step: packed instructions count 2 lanes; the mix counts its 12 FFMA2 (24 lane-ops);
    // kinds 6-8 count their FFMA2 lanes only (kinds 6 and 8 also run one DFMA per two FFMA2 on the FP64 pipe)
    const double per_step = (kind == 1 || kind >= 6) ? 2.0 : (kind == 5) ? 24.0 : 1.0;
    const double lane_ops = (double)grid * kThreads * (double)iters * kInner * kChains * per_step;
    const double sec = ms * 1e-3;
    const double mhz = h[1] ? (double)h[0] / (double)h[1] * 1e3 : 0.0;
    out4[0] = sec;
    out4[1] = lane_ops;
    out4[2] = mhz;
    out4[3] = (mhz > 0.0) ? lane_ops / (sec * mhz * 1e6 * sm_count) : 0.0;
    return 0;
}
