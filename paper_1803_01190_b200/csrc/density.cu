// density.cu -- face-on surface-density map, the diagnostic of Fig. 7: sigma(x, y) on a regular grid.
//
// HBM-bound O(N) pass: 16-32 B read per body, one FP64 atomic per body that lands on the grid.  Cells are tiny
// compared with L2 (a 1024^2 map is 8 MB), so the atomics resolve in L2; each CTA first bins into a shared-memory
// copy of the map when the map fits (<= 4096 cells), which turns the global atomics of a small map -- where many
// bodies hit the same cell -- into one per cell per CTA.
// The cell index is floor((x - x0) * (1/cell)) in FP64 on the promoted coordinate, so an FP32 state and its exact
// promotion land in the same cells.  Sums use floating-point atomics: equal to the oracle up to summation order.
#include "ppgrav_internal.h"

namespace ppgrav {
namespace {

constexpr int kThreads = 256;
constexpr int kSmemCells = 4096;

template <typename T, bool SMEM>
__global__ void __launch_bounds__(kThreads)
density_kernel(const T* __restrict__ pos, const T* __restrict__ mass, int64_t N, double x0, double y0, double inv,
               int nx, int ny, double scale, double* __restrict__ sigma) {
    __shared__ double local[SMEM ? kSmemCells : 1];
    const int cells = nx * ny;
    if (SMEM) {
        for (int c = threadIdx.x; c < cells; c += kThreads) local[c] = 0.0;
        __syncthreads();
    }
    for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < N; i += (int64_t)gridDim.x * kThreads) {
        const double fx = floor(((double)pos[3 * i] - x0) * inv);
        const double fy = floor(((double)pos[3 * i + 1] - y0) * inv);
        if (fx >= 0.0 && fx < (double)nx && fy >= 0.0 && fy < (double)ny) {
            const int c = (int)fy * nx + (int)fx;
            const double m = (double)mass[i] * scale;
            if (SMEM) atomicAdd(&local[c], m); else atomicAdd(&sigma[c], m);
        }
    }
    if (SMEM) {
        __syncthreads();
        for (int c = threadIdx.x; c < cells; c += kThreads)
            if (local[c] != 0.0) atomicAdd(&sigma[c], local[c]);
    }
}

template <typename T>
int launch(const T* pos, const T* mass, int64_t N, double x0, double y0, double cell, int nx, int ny, double* sigma,
           int sm_count, cudaStream_t st) {
    PP_CUDA(cudaMemsetAsync(sigma, 0, sizeof(double) * (size_t)nx * (size_t)ny, st));
    const int64_t want = (N + kThreads - 1) / kThreads;
    const int grid = (int)(want < (int64_t)sm_count * 8 ? want : (int64_t)sm_count * 8);
    const double inv = 1.0 / cell, scale = 1.0 / (cell * cell);
    if ((int64_t)nx * ny <= kSmemCells)
        density_kernel<T, true><<<grid, kThreads, 0, st>>>(pos, mass, N, x0, y0, inv, nx, ny, scale, sigma);
    else
        density_kernel<T, false><<<grid, kThreads, 0, st>>>(pos, mass, N, x0, y0, inv, nx, ny, scale, sigma);
    count_launch();
    PP_CUDA(cudaGetLastError());
    return PP_OK;
}

}  // namespace

int launch_density_f32(const float* pos, const float* mass, int64_t N, double x0, double y0, double cell, int nx,
                       int ny, double* sigma, int sm_count, cudaStream_t st) {
    return launch<float>(pos, mass, N, x0, y0, cell, nx, ny, sigma, sm_count, st);
}
int launch_density_f64(const double* pos, const double* mass, int64_t N, double x0, double y0, double cell, int nx,
                       int ny, double* sigma, int sm_count, cudaStream_t st) {
    return launch<double>(pos, mass, N, x0, y0, cell, nx, ny, sigma, sm_count, st);
}

}  // namespace ppgrav
