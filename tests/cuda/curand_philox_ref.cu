// curand_philox_ref.cu -- TEST HELPER, not the product: raw words of cuRAND's device Philox4x32-10 for given counters and
// keys, as the independent implementation SURVEY.md 8(c).4 asks the GPU generator to be cross-checked against.
// cuRAND's state: key = (seed lo, seed hi); counter = (offset/4 lo, offset/4 hi, subsequence lo, subsequence hi); the
// first curand4() after curand_init returns the four words of that counter.
#include <cuda_runtime.h>
#include <curand_kernel.h>
#include <stdint.h>

__global__ void k_ref(int n, const uint32_t* __restrict__ in /* [n][6] */, uint32_t* __restrict__ out /* [n][4] */) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const unsigned long long seed = ((unsigned long long)in[6 * i + 5] << 32) | in[6 * i + 4];
    const unsigned long long ctr_lo = ((unsigned long long)in[6 * i + 1] << 32) | in[6 * i];     // must be < 2^62
    const unsigned long long subseq = ((unsigned long long)in[6 * i + 3] << 32) | in[6 * i + 2];
    curandStatePhilox4_32_10_t st;
    curand_init(seed, subseq, 4ull * ctr_lo, &st);
    const uint4 r = curand4(&st);
    out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

extern "C" int curand_philox_words(int n, const uint32_t* ctr_key_host, uint32_t* out_host) {
    uint32_t *din = nullptr, *dout = nullptr;
    if (cudaMalloc((void**)&din, (size_t)n * 24) != cudaSuccess || cudaMalloc((void**)&dout, (size_t)n * 16) != cudaSuccess) return -1;
    cudaMemcpy(din, ctr_key_host, (size_t)n * 24, cudaMemcpyHostToDevice);
    k_ref<<<(n + 127) / 128, 128>>>(n, din, dout);
    const cudaError_t e = cudaMemcpy(out_host, dout, (size_t)n * 16, cudaMemcpyDeviceToHost);
    cudaFree(din);
    cudaFree(dout);
    return e == cudaSuccess ? 0 : -2;
}
