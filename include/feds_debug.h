/*
 * feds_debug.h — host-side arithmetic self-checks of libfeds' device building blocks. NOT part of the data path and not
 * needed by users of the library: the functions run, on the host, the same __host__ __device__ code the kernels call, so that
 * the CPU-only test suite can pin it against outside libraries without a GPU.
 *   feds_debug_sha256_host   : SHA-256 of a host buffer through the kernels' compression function.
 *   feds_debug_aes128_host   : one AES-128 block through the kernels' T-table rounds.
 *   feds_debug_dct8x8_host   : forward (inverse=0) / inverse (inverse=1) 8x8 float32 transform, row-major; bit-identical to
 *                              what the kernels compute (every operation is an explicitly rounded IEEE-754 mul/add/fma).
 *   feds_debug_zigzag_host   : the kernels' zigzag table, out[z] = 8*row + col.
 *   feds_debug_launch_count  : number of kernels this library has launched from the calling thread so far (a diagnostic counter,
 *                              per thread like feds_last_cuda_error; bench.py reports its increase over the timed region).
 */
#ifndef FEDS_DEBUG_H
#define FEDS_DEBUG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

void feds_debug_sha256_host(const uint8_t *msg, size_t n, uint8_t out[32]);
void feds_debug_aes128_host(const uint8_t key[16], const uint8_t in[16], uint8_t out[16]);
void feds_debug_dct8x8_host(const float in[64], float out[64], int inverse);
void feds_debug_zigzag_host(int out[64]);
void feds_debug_strong_basis_host(int32_t out[64 * 64]); /* the strong level's fixed-point DCT basis B[z][p] */
unsigned long long feds_debug_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* FEDS_DEBUG_H */
