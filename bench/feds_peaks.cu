// feds_peaks.cu — measured integer ceilings of this GPU for the SHA-256 arithmetic of the hot path (bench.py's ALU
// roofline context). Register-resident SHA-256 compressions with the library's own device function, no memory
// traffic: the most the chip can hash if nothing else ran. Prints one JSON line.
//   build: see paper_1512_02951_b200/build.py (target feds_peaks);  run: ./feds_peaks  |  ./feds_peaks pipes
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

// ---- per-SM, per-clock issue rate of the integer instructions SHA-256 and AES are made of (clock64-based, so independent
// of the SM frequency): 8 independent chains per thread, 512 threads on every SM. `./feds_peaks pipes`
template <int OP>
__global__ void __launch_bounds__(512, 1) pipe_kernel(uint32_t *out, long long *cyc, int n, uint32_t y, uint32_t z) {
    uint32_t x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = threadIdx.x * 31 + i;
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < n; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (OP == 0) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[i]) : "r"(y), "r"(z));
                if (OP == 1) asm volatile("shf.r.wrap.b32 %0, %0, %0, 7;" : "+r"(x[i]));
                if (OP == 2) asm volatile("prmt.b32 %0, %0, %1, 0x0123;" : "+r"(x[i]) : "r"(y));
                if (OP == 3) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x[i]) : "r"(y), "r"(z));
                if (OP == 4) asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(x[i]) : "r"(y));
                if (OP == 5) { if (i & 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[i]) : "r"(y), "r"(z));
                               else asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x[i]) : "r"(y), "r"(z)); }
                if (OP == 6) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+r"(x[i]) : "r"(y), "r"(z));
            }
        }
    }
    const long long t1 = clock64();
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s ^= x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}
template <int OP>
static double pipe_rate(int n_sm, uint32_t *out, long long *cyc) {
    const int n = 2000;
    pipe_kernel<OP><<<n_sm, 512>>>(out, cyc, n, 0x9e3779b9u, 0x7f4a7c15u);
    cudaDeviceSynchronize();
    long long c0 = 1;
    cudaMemcpy(&c0, cyc, 8, cudaMemcpyDeviceToHost);
    return 512.0 * n * 32 / (double)c0;
}
static int pipes_main() {
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, 0) != cudaSuccess) { printf("{\"error\": \"no CUDA device\"}\n"); return 1; }
    const int n_sm = prop.multiProcessorCount;
    uint32_t *out; long long *cyc;
    cudaMalloc(&out, (size_t)n_sm * 512 * 4); cudaMalloc(&cyc, (size_t)n_sm * 8);
    printf("{\"gpu\": \"%s\", \"unit\": \"lane-ops per clock per SM\", \"LOP3\": %.1f, \"SHF\": %.1f, \"PRMT\": %.1f, \"IMAD\": %.1f, "
           "\"IMAD.HI\": %.1f, \"LOP3+IMAD 1:1\": %.1f, \"FFMA\": %.1f}\n", prop.name, pipe_rate<0>(n_sm, out, cyc), pipe_rate<1>(n_sm, out, cyc),
           pipe_rate<2>(n_sm, out, cyc), pipe_rate<3>(n_sm, out, cyc), pipe_rate<4>(n_sm, out, cyc), pipe_rate<5>(n_sm, out, cyc),
           pipe_rate<6>(n_sm, out, cyc));
    cudaFree(out); cudaFree(cyc);
    return cudaGetLastError() == cudaSuccess ? 0 : 1;
}

int main(int argc, char **argv) {
    if (argc > 1 && argv[1][0] == 'p') return pipes_main();
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
