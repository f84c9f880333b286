// phx_aux.cu -- helper kernels off the stepping path: ensemble mean of |psi|^2 and the
// debug dump of the Philox words (same device function the stepping kernels call).
#include "phx_launch.h"
#include "phx_philox.cuh"

namespace phx {

template <typename T>
__global__ void ensemble_mean_kernel(const typename Cx<T>::type* __restrict__ psi, T* __restrict__ out, size_t plane, int batch) {
    const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= plane) return;
    double s = 0.0;   // plain sum over realisations r = 0..batch-1, accumulated in double
    for (int r = 0; r < batch; ++r) {
        const auto z = psi[(size_t)r * plane + k];
        s += (double)z.x * (double)z.x + (double)z.y * (double)z.y;
    }
    out[k] = (T)(s / (double)batch);
}

__global__ void noise_words_kernel(uint4* __restrict__ out, uint32_t seed, uint64_t step, size_t plane, uint32_t r0) {
    const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= plane) return;
    out[(size_t)blockIdx.y * plane + k] = noise_words(seed, r0 + blockIdx.y, step, (uint32_t)k);
}

cudaError_t launch_ensemble_mean(const void* psi, void* out, int prec64, size_t plane, int batch, cudaStream_t st) {
    const unsigned blocks = (unsigned)((plane + 255) / 256);
    if (prec64) ensemble_mean_kernel<double><<<blocks, 256, 0, st>>>((const double2*)psi, (double*)out, plane, batch);
    else ensemble_mean_kernel<float><<<blocks, 256, 0, st>>>((const float2*)psi, (float*)out, plane, batch);
    return cudaGetLastError();
}

// flag <- 1 if any of the n real values is NaN or +-Inf (the flag is zeroed by the caller)
template <typename T>
__global__ void check_finite_kernel(const T* data, size_t n, int* flag) {
    bool bad = false;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) bad |= !isfinite(data[i]);
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) *flag = 1;
}

cudaError_t launch_check_finite(const void* data, size_t n_reals, int prec64, int* flag, cudaStream_t st) {
    const size_t want = (n_reals + 255) / 256;
    const unsigned blocks = (unsigned)(want < 148u * 16u ? (want ? want : 1) : 148u * 16u);
    if (prec64) check_finite_kernel<double><<<blocks, 256, 0, st>>>((const double*)data, n_reals, flag);
    else check_finite_kernel<float><<<blocks, 256, 0, st>>>((const float*)data, n_reals, flag);
    return cudaGetLastError();
}

cudaError_t launch_noise_words(uint32_t* out, uint32_t seed, uint64_t step, size_t plane, int r0, int batch, cudaStream_t st) {
    const dim3 grid((unsigned)((plane + 255) / 256), (unsigned)batch);
    noise_words_kernel<<<grid, 256, 0, st>>>((uint4*)out, seed, step, plane, (uint32_t)r0);
    return cudaGetLastError();
}

}  // namespace phx
