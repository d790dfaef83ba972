// Test helper (not product, not oracle): runs cuRAND's own Philox4x32-10 block function ON THE DEVICE, as a black box, so the
// words libpimc's kernels draw can be compared with a library routine on the same GPU (pin P4 of SURVEY.md §8(c)).
#include <curand_kernel.h>
#include <curand_philox4x32_x.h>
#include <cstdint>

__global__ void curand_philox_kernel(uint64_t n, const uint32_t* ctrs, uint32_t k0, uint32_t k1, uint32_t* out) {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint4 r = curand_Philox4x32_10(make_uint4(ctrs[4 * i], ctrs[4 * i + 1], ctrs[4 * i + 2], ctrs[4 * i + 3]), make_uint2(k0, k1));
        out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
    }
}

// ctrs, out: device pointers.  Returns the CUDA error code of the launch + synchronisation.
extern "C" int curand_philox_device(uint64_t n, const uint32_t* ctrs, uint32_t k0, uint32_t k1, uint32_t* out) {
    curand_philox_kernel<<<296, 256>>>(n, ctrs, k0, k1, out);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    return (int)e;
}
