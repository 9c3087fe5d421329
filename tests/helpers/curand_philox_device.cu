// Test helper (pin P6): raw output of cuRAND's DEVICE-API
// Philox4_32_10 generator for chosen (seed, subsequence, offset).  Compiled by
// tests/test_gpu_parity.py with nvcc at test time; not part of the product and
// not part of the oracle -- it only calls the library generator.
//
// cuRAND documents curand_init(seed, subsequence, offset, &state) for this
// generator as: key = seed; the 128-bit counter is (offset / 4) in its low 64
// bits and the subsequence in its high 64 bits; curand4() returns the four
// 32-bit outputs of the current counter (offset % 4 == 0 here).
#include <cstdint>
#include <cuda_runtime.h>
#include <curand_kernel.h>

__global__ void k(const unsigned long long* seed, const unsigned long long* subseq,
                  const unsigned long long* offset4, uint4* out, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    curandStatePhilox4_32_10_t st;
    curand_init(seed[i], subseq[i], 4ull * offset4[i], &st);
    out[i] = curand4(&st);
}

extern "C" int curand_philox_device(const unsigned long long* seed, const unsigned long long* subseq,
                                    const unsigned long long* offset4, unsigned int* out, int n) {
    unsigned long long* d = nullptr;
    uint4* o = nullptr;
    if (cudaMalloc(&d, 3 * sizeof(unsigned long long) * n) != cudaSuccess) return 1;
    if (cudaMalloc(&o, sizeof(uint4) * n) != cudaSuccess) return 2;
    cudaMemcpy(d, seed, 8 * n, cudaMemcpyHostToDevice);
    cudaMemcpy(d + n, subseq, 8 * n, cudaMemcpyHostToDevice);
    cudaMemcpy(d + 2 * n, offset4, 8 * n, cudaMemcpyHostToDevice);
    k<<<(n + 63) / 64, 64>>>(d, d + n, d + 2 * n, o, n);
    const cudaError_t e = cudaMemcpy(out, o, sizeof(uint4) * n, cudaMemcpyDeviceToHost);
    cudaFree(d); cudaFree(o);
    return e == cudaSuccess ? 0 : 3;
}
