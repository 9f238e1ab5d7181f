// Test-only: cuRAND's own device implementation of Philox4x32-10 (curand_philox4x32_x.h), exposed through a
// C entry point so that tests can pin BOTH the oracle's and the library's Philox against a third party,
// including counter word 3 (which cuRAND's host generator API cannot reach).  Not part of the product.
#include <cuda_runtime.h>
#include <curand_kernel.h>
#include <stdint.h>

__global__ void k_curand_philox(const uint4 *ctr, const uint2 *key, uint4 *out, long long n)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        out[i] = curand_Philox4x32_10(ctr[i], key[i]);
}

extern "C" int curand_ref_philox(const uint32_t *ctr, const uint32_t *key, uint32_t *out, long long n)
{
    uint4 *dc = nullptr, *dout = nullptr;
    uint2 *dk = nullptr;
    cudaError_t e = cudaMalloc(&dc, n * 16);
    if (e == cudaSuccess) e = cudaMalloc(&dk, n * 8);
    if (e == cudaSuccess) e = cudaMalloc(&dout, n * 16);
    if (e == cudaSuccess) e = cudaMemcpy(dc, ctr, n * 16, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(dk, key, n * 8, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_curand_philox<<<1024, 256>>>(dc, dk, dout, n);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(out, dout, n * 16, cudaMemcpyDeviceToHost);
    cudaFree(dc); cudaFree(dk); cudaFree(dout);
    return (int)e;
}
