// api_host.cu -- the *_host entry points of include/ppgrav.h: HOST pointers in, the same device path, HOST pointers
// out.  Device staging comes from the stream-ordered allocator (cudaMallocAsync), so nothing is cached here; every
// call ends with a synchronisation of `stream`.  These are what bench.py's end-to-end figure times.
#include <cstddef>

#include "ppgrav_internal.h"

namespace {

using namespace ppgrav;

struct Stage {   // frees its device blocks (stream-ordered) when it goes out of scope
    cudaStream_t st;
    void* p[6] = {};
    int n = 0;
    explicit Stage(cudaStream_t s) : st(s) {}
    ~Stage() {
        for (int i = 0; i < n; ++i)
            if (p[i]) cudaFreeAsync(p[i], st);
    }
    int alloc(size_t bytes, void** out) {
        void* q = nullptr;
        const cudaError_t e = cudaMallocAsync(&q, bytes, st);
        if (e != cudaSuccess) {
            cudaGetLastError();
            set_error("staging allocation of %zu bytes failed: %s", bytes, cudaGetErrorString(e));
            return PP_ENOMEM;
        }
        p[n++] = q;
        *out = q;
        return PP_OK;
    }
    int upload(const void* host, size_t bytes, void** out) {
        const int rc = alloc(bytes, out);
        if (rc != PP_OK) return rc;
        PP_CUDA(cudaMemcpyAsync(*out, host, bytes, cudaMemcpyHostToDevice, st));
        return PP_OK;
    }
};

#define PP_TRYH(expr)                   \
    do {                                \
        const int rc__ = (expr);        \
        if (rc__ != PP_OK) return rc__; \
    } while (0)

bool host_args_ok(const char* fn, int64_t N, int precision) {
    if ((precision != PP_F32 && precision != PP_F64 && precision != PP_MIXED) || N < 1 || N > ((int64_t)1 << 28)) {
        set_error("%s: bad precision (%d) or N (%lld)", fn, precision, (long long)N);
        return false;
    }
    return true;
}

}  // namespace

extern "C" {

int pp_forces_host(const void* pos, const void* mass, void* acc, void* pot, int64_t N, double G, double delta,
                   int precision, void* stream) {
    if (!host_args_ok("pp_forces_host", N, precision)) return PP_EINVAL;
    if (!pos || !mass || !acc) { set_error("pp_forces_host: NULL pointer"); return PP_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t e = precision == PP_F32 ? 4 : 8, n = (size_t)N;
    Stage s(st);
    void *dpos, *dmass, *dacc, *dpot = nullptr;
    PP_TRYH(s.upload(pos, 3 * n * e, &dpos));
    PP_TRYH(s.upload(mass, n * e, &dmass));
    PP_TRYH(s.alloc(3 * n * e, &dacc));
    if (pot) PP_TRYH(s.alloc(n * e, &dpot));
    PP_TRYH(pp_forces(dpos, dmass, dacc, dpot, N, G, delta, precision, stream));
    PP_CUDA(cudaMemcpyAsync(acc, dacc, 3 * n * e, cudaMemcpyDeviceToHost, st));
    if (pot) PP_CUDA(cudaMemcpyAsync(pot, dpot, n * e, cudaMemcpyDeviceToHost, st));
    PP_CUDA(cudaStreamSynchronize(st));
    return PP_OK;
}

int pp_step_kdk_host(void* pos, void* vel, const void* mass, void* acc, void* pot, int64_t N, double dt,
                     int64_t nsteps, double G, double delta, int precision, unsigned flags, void* stream) {
    if (!host_args_ok("pp_step_kdk_host", N, precision)) return PP_EINVAL;
    if (!pos || !vel || !mass || !acc) { set_error("pp_step_kdk_host: NULL pointer"); return PP_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t e = precision == PP_F32 ? 4 : 8, n = (size_t)N;
    Stage s(st);
    void *dpos, *dvel, *dmass, *dacc, *dpot = nullptr;
    PP_TRYH(s.upload(pos, 3 * n * e, &dpos));
    PP_TRYH(s.upload(vel, 3 * n * e, &dvel));
    PP_TRYH(s.upload(mass, n * e, &dmass));
    if (flags & PP_ACC_VALID) PP_TRYH(s.upload(acc, 3 * n * e, &dacc));
    else PP_TRYH(s.alloc(3 * n * e, &dacc));
    const bool solves = nsteps > 0 || !(flags & PP_ACC_VALID);
    if (pot && solves) PP_TRYH(s.alloc(n * e, &dpot));
    PP_TRYH(pp_step_kdk(dpos, dvel, dmass, dacc, dpot, N, dt, nsteps, G, delta, precision, flags, stream));
    if (dpot) PP_CUDA(cudaMemcpyAsync(pot, dpot, n * e, cudaMemcpyDeviceToHost, st));
    PP_CUDA(cudaMemcpyAsync(pos, dpos, 3 * n * e, cudaMemcpyDeviceToHost, st));
    PP_CUDA(cudaMemcpyAsync(vel, dvel, 3 * n * e, cudaMemcpyDeviceToHost, st));
    PP_CUDA(cudaMemcpyAsync(acc, dacc, 3 * n * e, cudaMemcpyDeviceToHost, st));
    PP_CUDA(cudaStreamSynchronize(st));
    return PP_OK;
}

int pp_invariants_host(const void* pos, const void* vel, const void* mass, const void* pot, int64_t N, double G,
                       double delta, int precision, double* out16, void* stream) {
    if (!host_args_ok("pp_invariants_host", N, precision)) return PP_EINVAL;
    if (!pos || !vel || !mass || !out16) { set_error("pp_invariants_host: NULL pointer"); return PP_EINVAL; }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t e = precision == PP_F32 ? 4 : 8, n = (size_t)N;
    Stage s(st);
    void *dpos, *dvel, *dmass, *dpot = nullptr, *dout;
    PP_TRYH(s.upload(pos, 3 * n * e, &dpos));
    PP_TRYH(s.upload(vel, 3 * n * e, &dvel));
    PP_TRYH(s.upload(mass, n * e, &dmass));
    if (pot) PP_TRYH(s.upload(pot, n * e, &dpot));
    PP_TRYH(s.alloc(16 * sizeof(double), &dout));
    PP_TRYH(pp_invariants(dpos, dvel, dmass, dpot, N, G, delta, precision, (double*)dout, stream));
    PP_CUDA(cudaMemcpyAsync(out16, dout, 16 * sizeof(double), cudaMemcpyDeviceToHost, st));
    PP_CUDA(cudaStreamSynchronize(st));
    return PP_OK;
}

}  // extern "C"
