// feds_peaks.cu — measured integer ceilings of this GPU for the SHA-256 arithmetic of the hot path (bench.py's ALU
// roofline context). Register-resident SHA-256 compressions with the library's own device function, no memory
// traffic: the most the chip can hash if nothing else ran. Prints one JSON line.
//   build: see paper_1512_02951_b200/build.py (target feds_peaks);  run: ./feds_peaks
#include <cuda_runtime.h>

#include <cstdio>

#include "feds_device.cuh"
using namespace feds;

template <int VARIANT>
__global__ void __launch_bounds__(256, 2) sha_peak_kernel(uint32_t *out, int n, uint32_t one) {
    uint32_t H[8], w[16];
    sha256_init(H);
    H[0] ^= threadIdx.x + blockIdx.x * 977u;
#pragma unroll 1
    for (int it = 0; it < n; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) w[i] = H[i & 7] + i * 0x01010101u + it;
        if (VARIANT == 0) sha256_compress(H, w);
        else if (VARIANT == 1) sha256_compress_rolled(H, w);
        else sha256_compress_rolled_fma(H, w, one);
    }
    uint32_t x = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) x ^= H[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = x;
}

template <int VARIANT>
static double run(int n_sm, int n, uint32_t *out) {
    const int ctas = n_sm * 2, threads = 256;
    sha_peak_kernel<VARIANT><<<ctas, threads>>>(out, n, 1u);
    cudaDeviceSynchronize();
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0);
        sha_peak_kernel<VARIANT><<<ctas, threads>>>(out, n, 1u);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        const double gbs = (double)ctas * threads * n * 64.0 / (ms * 1e-3) / 1e9;
        if (gbs > best) best = gbs;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return best;
}

int main() {
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, 0) != cudaSuccess) { printf("{\"error\": \"no CUDA device\"}\n"); return 1; }
    const int n_sm = prop.multiProcessorCount;
    uint32_t *out;
    cudaMalloc(&out, (size_t)n_sm * 2 * 256 * 4);
    const double a = run<0>(n_sm, 512, out), b = run<1>(n_sm, 512, out), c = run<2>(n_sm, 512, out);
    printf("{\"gpu\": \"%s\", \"sms\": %d, \"warps_per_sm\": 16, \"sha256_GBps_unrolled64\": %.1f, \"sha256_GBps_rolled16\": %.1f, "
           "\"sha256_GBps_rolled16_fma_adds\": %.1f}\n", prop.name, n_sm, a, b, c);
    cudaFree(out);
    return cudaGetLastError() == cudaSuccess ? 0 : 1;
}
