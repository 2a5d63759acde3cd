// feds_device.cuh — arithmetic building blocks of the CUDA path (sm_100a): SHA-256 compression, AES-128 T-table
// rounds, CTR counter arithmetic, factorised 8-point DCT/IDCT, zigzag table. All are __host__ __device__ so the
// -m "not gpu" tests can exercise exactly the code the kernels run (feds_debug_*_host in feds.h).
// Shares nothing with oracle/: tables are generated here at compile time from the standards' definitions.
#pragma once
#include <cmath>
#include <cstdint>
#include <cstddef>

#define FEDS_HD __host__ __device__ __forceinline__

namespace feds {

constexpr int G_BLOCKS = 8;        // blocks per DCT-path leaf
constexpr int FANOUT = 16;         // children per Merkle node
constexpr int DWT_LEAF_BYTES = 2048;

// ------------------------------------------------------------------------------------------------------------
// SHA-256 (FIPS 180-4 6.2). State and message words are native uint32; callers byte-swap little-endian data.
// ------------------------------------------------------------------------------------------------------------
FEDS_HD uint32_t rotr32(uint32_t x, int n) {
#ifdef __CUDA_ARCH__
    return __funnelshift_r(x, x, n);
#else
    return (x >> n) | (x << (32 - n));
#endif
}
FEDS_HD uint32_t bswap32(uint32_t x) {
#ifdef __CUDA_ARCH__
    return __byte_perm(x, 0, 0x0123);
#else
    return (x >> 24) | ((x >> 8) & 0xff00u) | ((x << 8) & 0xff0000u) | (x << 24);
#endif
}

#define FEDS_SHA256_K_LIST                                                                                          \
    0x428a2f98u, 0x71374491u, 0xb5c0fbcfu, 0xe9b5dba5u, 0x3956c25bu, 0x59f111f1u, 0x923f82a4u, 0xab1c5ed5u,         \
    0xd807aa98u, 0x12835b01u, 0x243185beu, 0x550c7dc3u, 0x72be5d74u, 0x80deb1feu, 0x9bdc06a7u, 0xc19bf174u,         \
    0xe49b69c1u, 0xefbe4786u, 0x0fc19dc6u, 0x240ca1ccu, 0x2de92c6fu, 0x4a7484aau, 0x5cb0a9dcu, 0x76f988dau,         \
    0x983e5152u, 0xa831c66du, 0xb00327c8u, 0xbf597fc7u, 0xc6e00bf3u, 0xd5a79147u, 0x06ca6351u, 0x14292967u,         \
    0x27b70a85u, 0x2e1b2138u, 0x4d2c6dfcu, 0x53380d13u, 0x650a7354u, 0x766a0abbu, 0x81c2c92eu, 0x92722c85u,         \
    0xa2bfe8a1u, 0xa81a664bu, 0xc24b8b70u, 0xc76c51a3u, 0xd192e819u, 0xd6990624u, 0xf40e3585u, 0x106aa070u,         \
    0x19a4c116u, 0x1e376c08u, 0x2748774cu, 0x34b0bcb5u, 0x391c0cb3u, 0x4ed8aa4au, 0x5b9cca4fu, 0x682e6ff3u,         \
    0x748f82eeu, 0x78a5636fu, 0x84c87814u, 0x8cc70208u, 0x90befffau, 0xa4506cebu, 0xbef9a3f7u, 0xc67178f2u

FEDS_HD void sha256_init(uint32_t (&H)[8]) {
    H[0] = 0x6a09e667u; H[1] = 0xbb67ae85u; H[2] = 0x3c6ef372u; H[3] = 0xa54ff53au;
    H[4] = 0x510e527fu; H[5] = 0x9b05688cu; H[6] = 0x1f83d9abu; H[7] = 0x5be0cd19u;
}

// One 512-bit block. w[16] holds the big-endian message words W_0..W_15 and is clobbered (rolling schedule).
// Fully unrolled: every K_t becomes an immediate, every register index is static.
FEDS_HD void sha256_compress(uint32_t (&H)[8], uint32_t (&w)[16]) {
    constexpr uint32_t K[64] = {FEDS_SHA256_K_LIST};
    uint32_t a = H[0], b = H[1], c = H[2], d = H[3], e = H[4], f = H[5], g = H[6], h = H[7];
#pragma unroll
    for (int t = 0; t < 64; ++t) {
        if (t >= 16) {
            const uint32_t w15 = w[(t - 15) & 15], w2 = w[(t - 2) & 15];
            const uint32_t s0 = rotr32(w15, 7) ^ rotr32(w15, 18) ^ (w15 >> 3);
            const uint32_t s1 = rotr32(w2, 17) ^ rotr32(w2, 19) ^ (w2 >> 10);
            w[t & 15] = w[t & 15] + s0 + w[(t - 7) & 15] + s1;
        }
        const uint32_t S1 = rotr32(e, 6) ^ rotr32(e, 11) ^ rotr32(e, 25);
        const uint32_t ch = (e & f) ^ (~e & g);
        const uint32_t T1 = h + S1 + ch + K[t] + w[t & 15];
        const uint32_t S0 = rotr32(a, 2) ^ rotr32(a, 13) ^ rotr32(a, 22);
        const uint32_t maj = (a & b) ^ (a & c) ^ (b & c);
        const uint32_t T2 = S0 + maj;
        h = g; g = f; f = e; e = d + T1; d = c; c = b; b = a; a = T1 + T2;
    }
    H[0] += a; H[1] += b; H[2] += c; H[3] += d; H[4] += e; H[5] += f; H[6] += g; H[7] += h;
}

// The same compression as a 4 x 16-round loop: 4x less code (the fused kernels are instruction-cache bound when fully
// unrolled), W indices still static, K_t read from constant memory with a warp-uniform index.
#ifdef __CUDACC__
static __constant__ uint32_t c_sha256_k[64] = {FEDS_SHA256_K_LIST};
#endif
FEDS_HD void sha256_compress_rolled(uint32_t (&H)[8], uint32_t (&w)[16]) {
#ifndef __CUDA_ARCH__
    constexpr uint32_t K[64] = {FEDS_SHA256_K_LIST};
#endif
    uint32_t a = H[0], b = H[1], c = H[2], d = H[3], e = H[4], f = H[5], g = H[6], h = H[7];
#pragma unroll 1
    for (int i = 0; i < 4; ++i) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            if (i > 0) {
                const uint32_t w15 = w[(j + 1) & 15], w2 = w[(j + 14) & 15];
                const uint32_t s0 = rotr32(w15, 7) ^ rotr32(w15, 18) ^ (w15 >> 3);
                const uint32_t s1 = rotr32(w2, 17) ^ rotr32(w2, 19) ^ (w2 >> 10);
                w[j] = w[j] + s0 + w[(j + 9) & 15] + s1;
            }
#ifdef __CUDA_ARCH__
            const uint32_t kt = c_sha256_k[16 * i + j];
#else
            const uint32_t kt = K[16 * i + j];
#endif
            const uint32_t S1 = rotr32(e, 6) ^ rotr32(e, 11) ^ rotr32(e, 25);
            const uint32_t ch = (e & f) ^ (~e & g);
            const uint32_t T1 = h + S1 + ch + kt + w[j];
            const uint32_t S0 = rotr32(a, 2) ^ rotr32(a, 13) ^ rotr32(a, 22);
            const uint32_t maj = (a & b) ^ (a & c) ^ (b & c);
            h = g; g = f; f = e; e = d + T1; d = c; c = b; b = a; a = T1 + S0 + maj;
        }
    }
    H[0] += a; H[1] += b; H[2] += c; H[3] += d; H[4] += e; H[5] += f; H[6] += g; H[7] += h;
}

// Variant whose 32-bit additions are issued as IMAD (x * one + y, `one` = 1 known only at run time) so that they
// execute on the FMA pipe and leave the ALU pipe (64 lanes/clk/SM, measured) to the shifts and logic ops that can run
// nowhere else. On the device the multiply-adds are inline PTX: the compiler cannot see through them, so it cannot fold
// the K_t additions back into ALU-pipe adds ((x + K) * one), which it does with the plain C++ form.
FEDS_HD uint32_t add_fma(uint32_t x, uint32_t y, uint32_t one) {
#ifdef __CUDA_ARCH__
    uint32_t d;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(x), "r"(one), "r"(y));
    return d;
#else
    return x * one + y;
#endif
}
FEDS_HD void sha256_round_fma(uint32_t &a, uint32_t &b, uint32_t &c, uint32_t &d, uint32_t &e, uint32_t &f, uint32_t &g, uint32_t &h,
                              const uint32_t kt, const uint32_t wj, const uint32_t one) {
    const uint32_t S1 = rotr32(e, 6) ^ rotr32(e, 11) ^ rotr32(e, 25);
    const uint32_t ch = (e & f) ^ (~e & g);
    const uint32_t hk = add_fma(add_fma(one, kt, h), wj, one);   // one * K_t + h: K_t stays a multiplicand
    const uint32_t T1 = add_fma(add_fma(S1, ch, one), hk, one);
    const uint32_t S0 = rotr32(a, 2) ^ rotr32(a, 13) ^ rotr32(a, 22);
    const uint32_t maj = (a & b) ^ (a & c) ^ (b & c);
    h = g; g = f; f = e; e = add_fma(d, T1, one); d = c; c = b; b = a; a = add_fma(add_fma(S0, maj, one), T1, one);
}
// Rounds 0..15 straight from W (no schedule, no per-round branch), then 3 x 16 rounds in a loop that extends the rolling
// schedule in place one word ahead of its round. Measured on B200 (register-resident, 16 warps/SM): 1.07 TB/s hashed
// = 94 % of the ALU-pipe bound, against 0.95 TB/s for the 4 x 16 form with a branch per round and 0.92 TB/s fully unrolled.
FEDS_HD void sha256_compress_rolled_fma(uint32_t (&H)[8], uint32_t (&w)[16], const uint32_t one) {
#ifndef __CUDA_ARCH__
    constexpr uint32_t K[64] = {FEDS_SHA256_K_LIST};
#define FEDS_KT(t) K[t]
#else
#define FEDS_KT(t) c_sha256_k[t]
#endif
    uint32_t a = H[0], b = H[1], c = H[2], d = H[3], e = H[4], f = H[5], g = H[6], h = H[7];
#pragma unroll
    for (int j = 0; j < 16; ++j) sha256_round_fma(a, b, c, d, e, f, g, h, FEDS_KT(j), w[j], one);
#pragma unroll 1
    for (int i = 1; i < 4; ++i) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const uint32_t w15 = w[(j + 1) & 15], w2 = w[(j + 14) & 15];
            const uint32_t s0 = rotr32(w15, 7) ^ rotr32(w15, 18) ^ (w15 >> 3);
            const uint32_t s1 = rotr32(w2, 17) ^ rotr32(w2, 19) ^ (w2 >> 10);
            w[j] = add_fma(add_fma(w[j], s0, one), add_fma(w[(j + 9) & 15], s1, one), one);
            sha256_round_fma(a, b, c, d, e, f, g, h, FEDS_KT(16 * i + j), w[j], one);
        }
    }
#undef FEDS_KT
    H[0] += a; H[1] += b; H[2] += c; H[3] += d; H[4] += e; H[5] += f; H[6] += g; H[7] += h;
}

// ------------------------------------------------------------------------------------------------------------
// AES-128 (FIPS-197) with one-lookup-per-byte round tables. State = 4 column words, byte r of a word = row r
// (little-endian view of the FIPS-197 input bytes in[r + 4c]).
//   T0[x] = (2S, S, S, 3S) as bytes 0..3, S = SubBytes(x); T1/T2/T3 = T0 rotated left by 8/16/24 bits.
// Tables are built at compile time from the definition (GF(2^8) inverse + affine map).
// ------------------------------------------------------------------------------------------------------------
struct AesTables {
    uint32_t T[4][256];
    uint8_t S[256];
};

constexpr uint8_t gf_xtime(uint8_t a) { return (uint8_t)((a << 1) ^ ((a & 0x80) ? 0x1b : 0)); }
constexpr uint8_t gf_mul(uint8_t a, uint8_t b) {
    uint8_t p = 0;
    for (int i = 0; i < 8; ++i) { if (b & 1) p ^= a; a = gf_xtime(a); b >>= 1; }
    return p;
}
constexpr AesTables make_aes_tables() {
    AesTables t{};
    // log/antilog over the generator 0x03 gives the inverse without 254 multiplications per entry
    uint8_t alog[256] = {}, lg[256] = {};
    uint8_t x = 1;
    for (int i = 0; i < 255; ++i) { alog[i] = x; lg[x] = (uint8_t)i; x = (uint8_t)(x ^ gf_xtime(x)); }
    for (int v = 0; v < 256; ++v) {
        uint8_t inv = (v == 0) ? 0 : alog[(255 - lg[v]) % 255];
        uint8_t s = 0;
        for (int i = 0; i < 8; ++i) {
            int bit = ((inv >> i) ^ (inv >> ((i + 4) & 7)) ^ (inv >> ((i + 5) & 7)) ^ (inv >> ((i + 6) & 7)) ^
                       (inv >> ((i + 7) & 7)) ^ (0x63 >> i)) & 1;
            s = (uint8_t)(s | (bit << i));
        }
        t.S[v] = s;
        const uint32_t s2 = gf_xtime(s), s3 = (uint32_t)(s2 ^ s);
        const uint32_t t0 = s2 | ((uint32_t)s << 8) | ((uint32_t)s << 16) | (s3 << 24);
        t.T[0][v] = t0;
        t.T[1][v] = (t0 << 8) | (t0 >> 24);
        t.T[2][v] = (t0 << 16) | (t0 >> 16);
        t.T[3][v] = (t0 << 24) | (t0 >> 8);
    }
    return t;
}

// FIPS-197 5.2 key expansion (host side, once per call): rk[4*round + c] = column word c of round key `round`.
inline void aes128_expand_key_host(const uint8_t key[16], uint32_t rk[44], const AesTables &tb) {
    for (int i = 0; i < 4; ++i)
        rk[i] = (uint32_t)key[4 * i] | ((uint32_t)key[4 * i + 1] << 8) | ((uint32_t)key[4 * i + 2] << 16) |
                ((uint32_t)key[4 * i + 3] << 24);
    uint8_t rcon = 1;
    for (int i = 4; i < 44; ++i) {
        uint32_t t = rk[i - 1];
        if ((i & 3) == 0) {
            t = (t >> 8) | (t << 24);  // RotWord on the little-endian column word
            t = (uint32_t)tb.S[t & 0xff] | ((uint32_t)tb.S[(t >> 8) & 0xff] << 8) | ((uint32_t)tb.S[(t >> 16) & 0xff] << 16) |
                ((uint32_t)tb.S[(t >> 24) & 0xff] << 24);
            t ^= rcon;
            rcon = gf_xtime(rcon);
        }
        rk[i] = rk[i - 4] ^ t;
    }
}

// 10 rounds on one block. `T` points at the 4x256 table (shared memory on the device), `rk` at 44 round-key words.
template <typename TabPtr, typename RkPtr>
FEDS_HD void aes128_encrypt(const TabPtr T, const RkPtr rk, uint32_t (&s)[4]) {
    uint32_t s0 = s[0] ^ rk[0], s1 = s[1] ^ rk[1], s2 = s[2] ^ rk[2], s3 = s[3] ^ rk[3];
#pragma unroll
    for (int r = 1; r < 10; ++r) {
        const uint32_t t0 = T[0 * 256 + (s0 & 0xff)] ^ T[1 * 256 + ((s1 >> 8) & 0xff)] ^ T[2 * 256 + ((s2 >> 16) & 0xff)] ^
                            T[3 * 256 + (s3 >> 24)] ^ rk[4 * r + 0];
        const uint32_t t1 = T[0 * 256 + (s1 & 0xff)] ^ T[1 * 256 + ((s2 >> 8) & 0xff)] ^ T[2 * 256 + ((s3 >> 16) & 0xff)] ^
                            T[3 * 256 + (s0 >> 24)] ^ rk[4 * r + 1];
        const uint32_t t2 = T[0 * 256 + (s2 & 0xff)] ^ T[1 * 256 + ((s3 >> 8) & 0xff)] ^ T[2 * 256 + ((s0 >> 16) & 0xff)] ^
                            T[3 * 256 + (s1 >> 24)] ^ rk[4 * r + 2];
        const uint32_t t3 = T[0 * 256 + (s3 & 0xff)] ^ T[1 * 256 + ((s0 >> 8) & 0xff)] ^ T[2 * 256 + ((s1 >> 16) & 0xff)] ^
                            T[3 * 256 + (s2 >> 24)] ^ rk[4 * r + 3];
        s0 = t0; s1 = t1; s2 = t2; s3 = t3;
    }
    // final round: SubBytes + ShiftRows only. S = byte 0 of T2 = byte 1,2 of T0 = byte 3 of T2 (see table layout).
    const uint32_t u0 = (T[2 * 256 + (s0 & 0xff)] & 0xffu) | (T[0 * 256 + ((s1 >> 8) & 0xff)] & 0xff00u) |
                        (T[0 * 256 + ((s2 >> 16) & 0xff)] & 0xff0000u) | (T[2 * 256 + (s3 >> 24)] & 0xff000000u);
    const uint32_t u1 = (T[2 * 256 + (s1 & 0xff)] & 0xffu) | (T[0 * 256 + ((s2 >> 8) & 0xff)] & 0xff00u) |
                        (T[0 * 256 + ((s3 >> 16) & 0xff)] & 0xff0000u) | (T[2 * 256 + (s0 >> 24)] & 0xff000000u);
    const uint32_t u2 = (T[2 * 256 + (s2 & 0xff)] & 0xffu) | (T[0 * 256 + ((s3 >> 8) & 0xff)] & 0xff00u) |
                        (T[0 * 256 + ((s0 >> 16) & 0xff)] & 0xff0000u) | (T[2 * 256 + (s1 >> 24)] & 0xff000000u);
    const uint32_t u3 = (T[2 * 256 + (s3 & 0xff)] & 0xffu) | (T[0 * 256 + ((s0 >> 8) & 0xff)] & 0xff00u) |
                        (T[0 * 256 + ((s1 >> 16) & 0xff)] & 0xff0000u) | (T[2 * 256 + (s2 >> 24)] & 0xff000000u);
    s[0] = u0 ^ rk[40]; s[1] = u1 ^ rk[41]; s[2] = u2 ^ rk[42]; s[3] = u3 ^ rk[43];
}

// CTR counter block T_i = (nonce + i) mod 2^128, nonce given as 4 big-endian 32-bit values n[0] (most significant)
// .. n[3]; result as the 4 little-endian column words of the AES input (SP 800-38A B.1, A6).
FEDS_HD void ctr_block(const uint32_t (&n)[4], uint64_t i, uint32_t (&col)[4]) {
    const uint32_t ilo = (uint32_t)i, ihi = (uint32_t)(i >> 32);
    const uint32_t c3 = n[3] + ilo;
    const uint32_t k3 = c3 < ilo ? 1u : 0u;
    const uint32_t t2 = n[2] + ihi;
    const uint32_t k2a = t2 < ihi ? 1u : 0u;
    const uint32_t c2 = t2 + k3;
    const uint32_t k2 = k2a | (c2 < k3 ? 1u : 0u);
    const uint32_t c1 = n[1] + k2;
    const uint32_t k1 = c1 < k2 ? 1u : 0u;
    const uint32_t c0 = n[0] + k1;
    col[0] = bswap32(c0); col[1] = bswap32(c1); col[2] = bswap32(c2); col[3] = bswap32(c3);
}

// ------------------------------------------------------------------------------------------------------------
// 8-point orthonormal DCT-II / DCT-III, even/odd factorisation, float32 (A18).
//   X[u] = c(u)/2 * sum_i x[i] cos((2i+1) u pi/16),  c(0) = 1/sqrt(2)
// ------------------------------------------------------------------------------------------------------------
#define FEDS_C1 0.490392640201615f /* cos(1 pi/16)/2 */
#define FEDS_C2 0.461939766255643f /* cos(2 pi/16)/2 */
#define FEDS_C3 0.415734806151273f /* cos(3 pi/16)/2 */
#define FEDS_C4 0.353553390593274f /* cos(4 pi/16)/2 = 1/(2 sqrt 2) */
#define FEDS_C5 0.277785116509801f /* cos(5 pi/16)/2 */
#define FEDS_C6 0.191341716182545f /* cos(6 pi/16)/2 */
#define FEDS_C7 0.097545161008064f /* cos(7 pi/16)/2 */

// Every operation is an explicitly rounded IEEE-754 single-precision mul / add / fma (no compiler contraction or
// reassociation), so every kernel that inlines these -- and the host build used by feds_debug_dct8x8_host -- produces the
// same bits: fragments and digests do not depend on which route or compiler version ran.
FEDS_HD float f_mul(float a, float b) {
#ifdef __CUDA_ARCH__
    return __fmul_rn(a, b);
#else
    return a * b;
#endif
}
FEDS_HD float f_add(float a, float b) {
#ifdef __CUDA_ARCH__
    return __fadd_rn(a, b);
#else
    return a + b;
#endif
}
FEDS_HD float f_sub(float a, float b) {
#ifdef __CUDA_ARCH__
    return __fsub_rn(a, b);
#else
    return a - b;
#endif
}
FEDS_HD float f_fma(float a, float b, float c) {
#ifdef __CUDA_ARCH__
    return __fmaf_rn(a, b, c);
#else
    return fmaf(a, b, c);
#endif
}

FEDS_HD void dct8(float &x0, float &x1, float &x2, float &x3, float &x4, float &x5, float &x6, float &x7) {
    const float a0 = f_add(x0, x7), a1 = f_add(x1, x6), a2 = f_add(x2, x5), a3 = f_add(x3, x4);
    const float b0 = f_sub(x0, x7), b1 = f_sub(x1, x6), b2 = f_sub(x2, x5), b3 = f_sub(x3, x4);
    const float e0 = f_add(a0, a3), e1 = f_add(a1, a2), e2 = f_sub(a0, a3), e3 = f_sub(a1, a2);
    x0 = f_mul(FEDS_C4, f_add(e0, e1));
    x4 = f_mul(FEDS_C4, f_sub(e0, e1));
    x2 = f_fma(FEDS_C2, e2, f_mul(FEDS_C6, e3));
    x6 = f_fma(FEDS_C6, e2, f_mul(-FEDS_C2, e3));
    x1 = f_fma(FEDS_C1, b0, f_fma(FEDS_C3, b1, f_fma(FEDS_C5, b2, f_mul(FEDS_C7, b3))));
    x3 = f_fma(FEDS_C3, b0, f_fma(-FEDS_C7, b1, f_fma(-FEDS_C1, b2, f_mul(-FEDS_C5, b3))));
    x5 = f_fma(FEDS_C5, b0, f_fma(-FEDS_C1, b1, f_fma(FEDS_C7, b2, f_mul(FEDS_C3, b3))));
    x7 = f_fma(FEDS_C7, b0, f_fma(-FEDS_C5, b1, f_fma(FEDS_C3, b2, f_mul(-FEDS_C1, b3))));
}

// inverse: x[i] = sum_u c(u)/2 X[u] cos((2i+1) u pi/16)
FEDS_HD void idct8(float &x0, float &x1, float &x2, float &x3, float &x4, float &x5, float &x6, float &x7) {
    const float p = f_mul(FEDS_C4, f_add(x0, x4)), q = f_mul(FEDS_C4, f_sub(x0, x4));
    const float r = f_fma(FEDS_C2, x2, f_mul(FEDS_C6, x6)), s = f_fma(FEDS_C6, x2, f_mul(-FEDS_C2, x6));
    const float e0 = f_add(p, r), e3 = f_sub(p, r), e1 = f_add(q, s), e2 = f_sub(q, s);  // even part at i = 0,1,2,3 (mirrored at 7,6,5,4)
    const float o0 = f_fma(FEDS_C1, x1, f_fma(FEDS_C3, x3, f_fma(FEDS_C5, x5, f_mul(FEDS_C7, x7))));
    const float o1 = f_fma(FEDS_C3, x1, f_fma(-FEDS_C7, x3, f_fma(-FEDS_C1, x5, f_mul(-FEDS_C5, x7))));
    const float o2 = f_fma(FEDS_C5, x1, f_fma(-FEDS_C1, x3, f_fma(FEDS_C7, x5, f_mul(FEDS_C3, x7))));
    const float o3 = f_fma(FEDS_C7, x1, f_fma(-FEDS_C5, x3, f_fma(FEDS_C3, x5, f_mul(-FEDS_C1, x7))));
    x0 = f_add(e0, o0); x7 = f_sub(e0, o0);
    x1 = f_add(e1, o1); x6 = f_sub(e1, o1);
    x2 = f_add(e2, o2); x5 = f_sub(e2, o2);
    x3 = f_add(e3, o3); x4 = f_sub(e3, o3);
}

// 2-D transform of a row-major block held in 64 registers: row pass then column pass (separable).
FEDS_HD void dct8x8(float (&v)[64]) {
#pragma unroll
    for (int r = 0; r < 8; ++r) dct8(v[8 * r], v[8 * r + 1], v[8 * r + 2], v[8 * r + 3], v[8 * r + 4], v[8 * r + 5], v[8 * r + 6], v[8 * r + 7]);
#pragma unroll
    for (int c = 0; c < 8; ++c) dct8(v[c], v[8 + c], v[16 + c], v[24 + c], v[32 + c], v[40 + c], v[48 + c], v[56 + c]);
}
FEDS_HD void idct8x8(float (&v)[64]) {
#pragma unroll
    for (int c = 0; c < 8; ++c) idct8(v[c], v[8 + c], v[16 + c], v[24 + c], v[32 + c], v[40 + c], v[48 + c], v[56 + c]);
#pragma unroll
    for (int r = 0; r < 8; ++r) idct8(v[8 * r], v[8 * r + 1], v[8 * r + 2], v[8 * r + 3], v[8 * r + 4], v[8 * r + 5], v[8 * r + 6], v[8 * r + 7]);
}

// Zigzag scan: z -> 8*row + col; anti-diagonals s = row + col, even s walks row downwards, odd s upwards.
struct ZigzagTable { int pos[64]; };
constexpr ZigzagTable make_zigzag() {
    ZigzagTable t{};
    int z = 0;
    for (int s = 0; s <= 14; ++s) {
        const int lo = s > 7 ? s - 7 : 0, hi = s < 7 ? s : 7;
        if ((s & 1) == 0) { for (int r = hi; r >= lo; --r) t.pos[z++] = 8 * r + (s - r); }
        else { for (int r = lo; r <= hi; ++r) t.pos[z++] = 8 * r + (s - r); }
    }
    return t;
}

}  // namespace feds
