// TEST INFRASTRUCTURE (pin P1 on the GPU box): raw words of cuRAND's Philox4_32_10 device generator, a
// library routine independent of both the oracle and libtaiga.  curand_init(seed, subsequence, offset)
// sets key = (seed lo, hi) and counter = (offset lo, offset hi, subsequence lo, subsequence hi);
// curand4() returns the four output words of that block.
#include <cuda_runtime.h>
#include <curand_kernel.h>
#include <stdint.h>

__global__ void k_words(unsigned long long seed, const unsigned long long* sub, const unsigned long long* off, int n, uint4* out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    curandStatePhilox4_32_10_t st;
    curand_init(seed, sub[i], off[i] * 4ull, &st);      // offset counts single 32-bit outputs: 4 per block
    out[i] = curand4(&st);
}

extern "C" int philox_curand_words(unsigned long long seed, const unsigned long long* sub_host, const unsigned long long* off_host,
                                   int n, uint32_t* out_host /* [n][4] */) {
    unsigned long long *sub = nullptr, *off = nullptr;
    uint4* out = nullptr;
    if (cudaMalloc(&sub, n * 8) || cudaMalloc(&off, n * 8) || cudaMalloc(&out, n * 16)) return -1;
    cudaMemcpy(sub, sub_host, n * 8, cudaMemcpyHostToDevice);
    cudaMemcpy(off, off_host, n * 8, cudaMemcpyHostToDevice);
    k_words<<<(n + 127) / 128, 128>>>(seed, sub, off, n, out);
    int rc = cudaMemcpy(out_host, out, n * 16, cudaMemcpyDeviceToHost) != cudaSuccess ? -2 : 0;
    cudaFree(sub); cudaFree(off); cudaFree(out);
    return rc;
}
