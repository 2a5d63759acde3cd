// feds_dct_strong.cuh — the report's STRONG level of protection (PAPER.md 6.3.2, Figure 8), sm_100a.
//
// Part 1 (DC + first k zigzag AC of every 8x8 block) is encrypted with AES-128-CTR exactly as at the first level; the public part
// of a block is no longer its remaining coefficients but 64 pixel bytes -- "the reverse DCT result of the rest DCT coefficients
// padded with zero" -- XORed with SHA-512(Part 1 of that block), a 512-bit string: one hash per block.
// Byte format and the readings the report leaves open: DESIGN.md 2.3 (S1-S5). In short, with c_z the float32 coefficients of Part 1:
//   q_z = rne(8 c_z),  L[p] = floor((sum_z q_z B[z][p] + 2^14) / 2^15),  public[p] = ((x[p] - L[p]) mod 256) xor SHA-512(Part 1)[p]
// with B the orthonormal DCT basis in 12-bit fixed point: IDCT(rest) = x - IDCT(Part 1) by linearity, evaluated in integers so that
// both directions (and any other implementation) get the same bytes and the round trip is exact by construction.
//
// One thread per (block, channel), no staging: the work per block is one SHA-512 compression (~5,000 instructions on 64-bit words
// held as register pairs), an order of magnitude above the data movement, so the kernels are kept simple and take any image size.
#pragma once
#include "feds_dct.cuh"

namespace feds {

constexpr int STRONG_THREADS = 128;

// B[z][p] = rne(4096 * b_z(p)), b_z(8 i + j) = 1/4 C(u) C(v) cos((2i+1) u pi/16) cos((2j+1) v pi/16), (u, v) = zigzag(z): built at
// compile time from the definition (cosines of multiples of pi/16 by a Taylor series on the first octant: error < 1e-16, and no
// entry is anywhere near a rounding tie; a test compares all 4096 entries with a table computed from libm's cosines).
struct StrongBasis { int32_t B[64 * 64]; };
constexpr double cos_pi16(int m) {   // cos(m pi / 16)
    m = ((m % 32) + 32) % 32;
    if (m > 16) m = 32 - m;          // cos(2 pi - x) = cos x
    bool neg = false;
    if (m > 8) { m = 16 - m; neg = true; }   // cos(pi - x) = -cos x
    const double x = m * (3.14159265358979323846264338327950288 / 16.0), x2 = x * x;
    double term = 1.0, sum = 1.0;
    for (int n = 1; n <= 14; ++n) { term *= -x2 / ((2 * n - 1) * (2 * n)); sum += term; }
    return neg ? -sum : sum;
}
constexpr StrongBasis make_strong_basis() {
    StrongBasis t{};
    constexpr ZigzagTable ZZ = make_zigzag();
    for (int z = 0; z < 64; ++z) {
        const int u = ZZ.pos[z] / 8, v = ZZ.pos[z] % 8;
        const double cu = u ? 1.0 : 0.70710678118654752440, cv = v ? 1.0 : 0.70710678118654752440;
        for (int i = 0; i < 8; ++i)
            for (int j = 0; j < 8; ++j) {
                const double b = 4096.0 * 0.25 * cu * cv * cos_pi16((2 * i + 1) * u) * cos_pi16((2 * j + 1) * v);
                t.B[64 * z + 8 * i + j] = b >= 0.0 ? (int32_t)(b + 0.5) : -(int32_t)(-b + 0.5);
            }
    }
    return t;
}
#ifdef __CUDACC__
static __constant__ StrongBasis c_strong_basis_tab = make_strong_basis();
#endif

#define FEDS_SHA512_K_LIST                                                                                                       \
    0x428a2f98d728ae22ULL, 0x7137449123ef65cdULL, 0xb5c0fbcfec4d3b2fULL, 0xe9b5dba58189dbbcULL, 0x3956c25bf348b538ULL,           \
    0x59f111f1b605d019ULL, 0x923f82a4af194f9bULL, 0xab1c5ed5da6d8118ULL, 0xd807aa98a3030242ULL, 0x12835b0145706fbeULL,           \
    0x243185be4ee4b28cULL, 0x550c7dc3d5ffb4e2ULL, 0x72be5d74f27b896fULL, 0x80deb1fe3b1696b1ULL, 0x9bdc06a725c71235ULL,           \
    0xc19bf174cf692694ULL, 0xe49b69c19ef14ad2ULL, 0xefbe4786384f25e3ULL, 0x0fc19dc68b8cd5b5ULL, 0x240ca1cc77ac9c65ULL,           \
    0x2de92c6f592b0275ULL, 0x4a7484aa6ea6e483ULL, 0x5cb0a9dcbd41fbd4ULL, 0x76f988da831153b5ULL, 0x983e5152ee66dfabULL,           \
    0xa831c66d2db43210ULL, 0xb00327c898fb213fULL, 0xbf597fc7beef0ee4ULL, 0xc6e00bf33da88fc2ULL, 0xd5a79147930aa725ULL,           \
    0x06ca6351e003826fULL, 0x142929670a0e6e70ULL, 0x27b70a8546d22ffcULL, 0x2e1b21385c26c926ULL, 0x4d2c6dfc5ac42aedULL,           \
    0x53380d139d95b3dfULL, 0x650a73548baf63deULL, 0x766a0abb3c77b2a8ULL, 0x81c2c92e47edaee6ULL, 0x92722c851482353bULL,           \
    0xa2bfe8a14cf10364ULL, 0xa81a664bbc423001ULL, 0xc24b8b70d0f89791ULL, 0xc76c51a30654be30ULL, 0xd192e819d6ef5218ULL,           \
    0xd69906245565a910ULL, 0xf40e35855771202aULL, 0x106aa07032bbd1b8ULL, 0x19a4c116b8d2d0c8ULL, 0x1e376c085141ab53ULL,           \
    0x2748774cdf8eeb99ULL, 0x34b0bcb5e19b48a8ULL, 0x391c0cb3c5c95a63ULL, 0x4ed8aa4ae3418acbULL, 0x5b9cca4f7763e373ULL,           \
    0x682e6ff3d6b2b8a3ULL, 0x748f82ee5defb2fcULL, 0x78a5636f43172f60ULL, 0x84c87814a1f0ab72ULL, 0x8cc702081a6439ecULL,           \
    0x90befffa23631e28ULL, 0xa4506cebde82bde9ULL, 0xbef9a3f7b2c67915ULL, 0xc67178f2e372532bULL, 0xca273eceea26619cULL,           \
    0xd186b8c721c0c207ULL, 0xeada7dd6cde0eb1eULL, 0xf57d4f7fee6ed178ULL, 0x06f067aa72176fbaULL, 0x0a637dc5a2c898a6ULL,           \
    0x113f9804bef90daeULL, 0x1b710b35131c471bULL, 0x28db77f523047d84ULL, 0x32caab7b40c72493ULL, 0x3c9ebe0a15c9bebcULL,           \
    0x431d67c49c100d4cULL, 0x4cc5d4becb3e42b6ULL, 0x597f299cfc657e2aULL, 0x5fcb6fab3ad6faecULL, 0x6c44198c4a475817ULL
static __constant__ uint64_t c_sha512_k[80] = {FEDS_SHA512_K_LIST};

__device__ __forceinline__ uint64_t rotr64(uint64_t x, int n) { return (x >> n) | (x << (64 - n)); }

// FIPS 180-4 6.4.2, one 1024-bit block; w[16] = big-endian message words, clobbered (rolling schedule)
__device__ __forceinline__ void sha512_compress(uint64_t (&H)[8], uint64_t (&w)[16]) {
    uint64_t a = H[0], b = H[1], c = H[2], d = H[3], e = H[4], f = H[5], g = H[6], h = H[7];
#pragma unroll 1
    for (int i = 0; i < 5; ++i) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            if (i > 0) {
                const uint64_t w15 = w[(j + 1) & 15], w2 = w[(j + 14) & 15];
                const uint64_t s0 = rotr64(w15, 1) ^ rotr64(w15, 8) ^ (w15 >> 7);
                const uint64_t s1 = rotr64(w2, 19) ^ rotr64(w2, 61) ^ (w2 >> 6);
                w[j] = w[j] + s0 + w[(j + 9) & 15] + s1;
            }
            const uint64_t S1 = rotr64(e, 14) ^ rotr64(e, 18) ^ rotr64(e, 41);
            const uint64_t ch = (e & f) ^ (~e & g);
            const uint64_t T1 = h + S1 + ch + c_sha512_k[16 * i + j] + w[j];
            const uint64_t S0 = rotr64(a, 28) ^ rotr64(a, 34) ^ rotr64(a, 39);
            const uint64_t maj = (a & b) ^ (a & c) ^ (b & c);
            h = g; g = f; f = e; e = d + T1; d = c; c = b; b = a; a = T1 + S0 + maj;
        }
    }
    H[0] += a; H[1] += b; H[2] += c; H[3] += d; H[4] += e; H[5] += f; H[6] += g; H[7] += h;
}

// SHA-512 of the P little-endian 32-bit words part1[0], part1[stride], ... (a block's Part 1 in a shared-memory column);
// the 64 digest bytes come back as 16 words in memory order (ks[2 i], ks[2 i + 1] = bytes 8 i .. 8 i + 7 of the digest)
__device__ __forceinline__ void sha512_part1_keystream(const uint32_t *part1, int stride, int P, uint32_t (&ks)[16]) {
    uint64_t H[8] = {0x6a09e667f3bcc908ULL, 0xbb67ae8584caa73bULL, 0x3c6ef372fe94f82bULL, 0xa54ff53a5f1d36f1ULL,
                     0x510e527fade682d1ULL, 0x9b05688c2b3e6c1fULL, 0x1f83d9abfb41bd6bULL, 0x5be0cd19137e2179ULL};
    const int nblocks = (4 * P + 17 + 127) / 128;   // message + 0x80 + 128-bit length
    uint64_t w[16];
#pragma unroll 1
    for (int blk = 0; blk < nblocks; ++blk) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            uint32_t half[2];
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const int idx = 32 * blk + 2 * j + q;   // 32-bit word index in the padded message
                half[q] = idx < P ? bswap32(part1[idx * stride]) : (idx == P ? 0x80000000u : 0u);
            }
            w[j] = ((uint64_t)half[0] << 32) | half[1];
        }
        if (blk == nblocks - 1) w[15] = (uint64_t)P * 32ull;   // message length in bits
        sha512_compress(H, w);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        ks[2 * i] = bswap32((uint32_t)(H[i] >> 32));
        ks[2 * i + 1] = bswap32((uint32_t)H[i]);
    }
}

// L[p] (DESIGN.md 2.3 S1) of one block from the Part 1 column in shared memory; arithmetic modulo 2^32, of which only bits 15..22
// are used (a sum in 64 bits has the same bits there)
__device__ __forceinline__ void strong_low_pass(const uint32_t *part1, int stride, int P, int32_t (&acc)[64]) {
#pragma unroll
    for (int p = 0; p < 64; ++p) acc[p] = 16384;
#pragma unroll 1
    for (int z = 0; z < P; ++z) {
        const int32_t q = __float2int_rn(8.0f * __uint_as_float(part1[z * stride]));   // saturates; NaN -> 0
        const int32_t *Bz = c_strong_basis_tab.B + 64 * z;
#pragma unroll
        for (int p = 0; p < 64; ++p) acc[p] = (int32_t)((uint32_t)acc[p] + (uint32_t)q * (uint32_t)Bz[p]);
    }
}
// four remainder (fragment) or pixel (defragment) bytes: byte i = (in_i -/+ L_i) mod 256, L_i = acc_i >> 15
template <bool SUBTRACT>
__device__ __forceinline__ uint32_t strong_apply4(uint32_t in, int32_t a0, int32_t a1, int32_t a2, int32_t a3) {
    const uint32_t L = ((uint32_t)(a0 >> 15) & 255u) | (((uint32_t)(a1 >> 15) & 255u) << 8) | (((uint32_t)(a2 >> 15) & 255u) << 16) |
                       (((uint32_t)(a3 >> 15) & 255u) << 24);
    return SUBTRACT ? __vsub4(in, L) : __vadd4(in, L);   // per-byte, modulo 256
}

// AES-128-CTR keystream for the P words [w0, w0 + P) of the image's private stream, XORed into the column part1[z * stride] and
// written to / read from global memory by the caller; every counter block that overlaps the run is computed by this thread
template <typename Tab>
__device__ __forceinline__ void strong_ctr_xor(const DctParams &p, const Tab sT, const uint32_t (&nonce)[4], unsigned long long w0, int P,
                                               uint32_t *part1, int stride) {
    unsigned long long blk = w0 >> 2;
    int z = -(int)(w0 & 3);   // run-relative index of the counter block's first word
#pragma unroll 1
    for (; z < P; z += 4, ++blk) {
        uint32_t ks[4];
        ctr_block(nonce, blk, ks);
        aes128_encrypt(sT, p.rk, ks);
#pragma unroll
        for (int t = 0; t < 4; ++t)
            if (z + t >= 0 && z + t < P) part1[(z + t) * stride] ^= ks[t];
    }
}

struct StrongCoord {
    int n, ch, br, bc;
    size_t b;   // linear block index in the image
};
template <int C>
__device__ __forceinline__ bool strong_decode(const DctParams &p, unsigned long long gid, StrongCoord &S) {
    const unsigned long long per_image = (unsigned long long)C * p.nbr * p.nbc;
    if (gid >= per_image * p.n_images) return false;
    S.n = (int)(gid / per_image);
    unsigned rem = (unsigned)(gid % per_image);
    S.ch = (int)(rem % C);   // channel fastest: the C lanes of one pixel strip are adjacent (store_block_packed)
    rem /= C;
    S.bc = (int)(rem % (unsigned)p.nbc);
    S.br = (int)(rem / (unsigned)p.nbc);
    S.b = ((size_t)S.ch * p.nbr + S.br) * p.nbc + S.bc;
    return true;
}

// The same bytes without unpacking (small k). x - floor((S + 2^14) / 2^15) = floor((x 2^15 + 2^14 - 1 - S) / 2^15), and with
// everything doubled the low byte of that quotient is byte 2 of acc = (x << 16 | 0x7ffe) - sum (2 q_z) B_z; the inverse is byte 2
// of (r << 16 | 0x8000) + sum (2 q_z) B_z. One PRMT drops the byte into the accumulator over the constant BIAS, one IMAD per
// coefficient against the table in constant memory (immediate offsets), one PRMT per two results. m[z] = -/+ 2 q_z (arithmetic
// modulo 2^32 throughout, as in strong_low_pass). Rows 4 HALF .. 4 HALF + 3 of the block (words x[8 HALF ..]) -> r[0..7].
template <int HALF, int PMAX, uint32_t BIAS>
__device__ __forceinline__ void strong_bytes_half(const uint32_t (&x)[16], const int32_t (&m)[PMAX], int P, uint32_t (&r)[8]) {
    int32_t acc[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) acc[i] = (int32_t)__byte_perm(x[8 * HALF + (i >> 2)], BIAS, 0x7054u + ((uint32_t)(i & 3) << 8));
#pragma unroll
    for (int z = 0; z < PMAX; ++z) {
        if (z < P) {   // warp-uniform
#pragma unroll
            for (int i = 0; i < 32; ++i)
                acc[i] = (int32_t)((uint32_t)acc[i] + (uint32_t)m[z] * (uint32_t)c_strong_basis_tab.B[64 * z + 32 * HALF + i]);
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i)
        r[i] = __byte_perm(__byte_perm((uint32_t)acc[4 * i], (uint32_t)acc[4 * i + 1], 0x0062u), __byte_perm((uint32_t)acc[4 * i + 2], (uint32_t)acc[4 * i + 3], 0x0062u), 0x5410u);
}
// m[z] = sign * 2 * rne(8 c_z) from the Part 1 column
template <int PMAX>
__device__ __forceinline__ void strong_scaled_q(const uint32_t *part1, int stride, int P, int sign, int32_t (&m)[PMAX]) {
#pragma unroll
    for (int z = 0; z < PMAX; ++z)
        m[z] = z < P ? (int32_t)((uint32_t)__float2int_rn(8.0f * __uint_as_float(part1[z * stride])) * (uint32_t)(2 * sign)) : 0;
}

// the channel's 8 pixel bytes of row r of the block as two packed words (global memory, read-only path)
template <int C>
__device__ __forceinline__ uint2 strong_load_row(const uint8_t *row, int c) {
    if (C == 1) return __ldg(reinterpret_cast<const uint2 *>(row));
    if (C == 3) {
        const uint2 q0 = __ldg(reinterpret_cast<const uint2 *>(row)), q1 = __ldg(reinterpret_cast<const uint2 *>(row) + 1),
                    q2 = __ldg(reinterpret_cast<const uint2 *>(row) + 2);
        const uint32_t wd[7] = {q0.x, q0.y, q1.x, q1.y, q2.x, q2.y, 0u};
        uint32_t ws[6];
#pragma unroll
        for (int j = 0; j < 6; ++j) ws[j] = __funnelshift_r(wd[j], wd[j + 1], 8 * c);   // channel c now sits at bytes 0, 3, 6, ...
        uint2 o;
        o.x = __byte_perm(__byte_perm(ws[0], ws[1], 0x0630), __byte_perm(ws[1], ws[2], 0x0052), 0x5410);   // bytes 0, 3, 6, 9
        o.y = __byte_perm(__byte_perm(ws[3], ws[4], 0x0630), __byte_perm(ws[4], ws[5], 0x0052), 0x5410);   // bytes 12, 15, 18, 21
        return o;
    }
    const uint4 a = __ldg(reinterpret_cast<const uint4 *>(row)), b = __ldg(reinterpret_cast<const uint4 *>(row) + 1);
    const uint32_t s = 0x4440u + (uint32_t)c;
    uint2 o;
    o.x = __byte_perm(a.x, 0, s) | (__byte_perm(a.y, 0, s) << 8) | (__byte_perm(a.z, 0, s) << 16) | (__byte_perm(a.w, 0, s) << 24);
    o.y = __byte_perm(b.x, 0, s) | (__byte_perm(b.y, 0, s) << 8) | (__byte_perm(b.z, 0, s) << 16) | (__byte_perm(b.w, 0, s) << 24);
    return o;
}

// Store packed rows (two words per row) of the block of channel c: as store_block, after its rounding and packing.
template <int C>
__device__ __forceinline__ void store_block_packed(uint8_t *__restrict__ img, int w, int y0, int x0, int c, bool act, const uint32_t (&rows)[16]) {
    const int lane = threadIdx.x & 31;
    bool complete = true;
    if (C > 1) {
        const int l0 = lane - c;
        complete = (l0 >= 0) && (l0 + C - 1 <= 31);
        const unsigned actmask = __ballot_sync(0xffffffffu, act);
        if (complete) complete = ((actmask >> l0) & ((1u << C) - 1u)) == ((1u << C) - 1u);
    }
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const uint32_t lo = rows[2 * r], hi = rows[2 * r + 1];
        uint8_t *row = img + ((size_t)(y0 + r) * w + x0) * C;
        if (C == 1) {
            if (act) *reinterpret_cast<uint2 *>(row) = make_uint2(lo, hi);
        } else if (C == 3) {
            const uint32_t glo = __shfl_down_sync(0xffffffffu, lo, 1), ghi = __shfl_down_sync(0xffffffffu, hi, 1);
            const uint32_t blo = __shfl_down_sync(0xffffffffu, lo, 2), bhi = __shfl_down_sync(0xffffffffu, hi, 2);
            if (complete) {
                if (c == 0) {
                    const uint32_t rg0 = __byte_perm(lo, glo, 0x5140), rg1 = __byte_perm(lo, glo, 0x7362);
                    const uint32_t rg2 = __byte_perm(hi, ghi, 0x5140), rg3 = __byte_perm(hi, ghi, 0x7362);
                    uint2 *o = reinterpret_cast<uint2 *>(row);
                    o[0] = make_uint2(__byte_perm(rg0, blo, 0x2410), __byte_perm(__byte_perm(rg0, blo, 0x0053), rg1, 0x5410));
                    o[1] = make_uint2(__byte_perm(rg1, blo, 0x7326), __byte_perm(rg2, bhi, 0x2410));
                    o[2] = make_uint2(__byte_perm(__byte_perm(rg2, bhi, 0x0053), rg3, 0x5410), __byte_perm(rg3, bhi, 0x7326));
                }
            } else if (act) {
#pragma unroll
                for (int i = 0; i < 8; ++i) row[i * 3 + c] = (uint8_t)((i < 4 ? lo : hi) >> (8 * (i & 3)));
            }
        } else {
            const uint32_t glo = __shfl_down_sync(0xffffffffu, lo, 1), ghi = __shfl_down_sync(0xffffffffu, hi, 1);
            const uint32_t blo = __shfl_down_sync(0xffffffffu, lo, 2), bhi = __shfl_down_sync(0xffffffffu, hi, 2);
            const uint32_t alo = __shfl_down_sync(0xffffffffu, lo, 3), ahi = __shfl_down_sync(0xffffffffu, hi, 3);
            if (complete) {
                if (c == 0) {
                    const uint32_t rg0 = __byte_perm(lo, glo, 0x5140), rg1 = __byte_perm(lo, glo, 0x7362);
                    const uint32_t ba0 = __byte_perm(blo, alo, 0x5140), ba1 = __byte_perm(blo, alo, 0x7362);
                    const uint32_t rg2 = __byte_perm(hi, ghi, 0x5140), rg3 = __byte_perm(hi, ghi, 0x7362);
                    const uint32_t ba2 = __byte_perm(bhi, ahi, 0x5140), ba3 = __byte_perm(bhi, ahi, 0x7362);
                    uint4 *o = reinterpret_cast<uint4 *>(row);
                    o[0] = make_uint4(__byte_perm(rg0, ba0, 0x5410), __byte_perm(rg0, ba0, 0x7632), __byte_perm(rg1, ba1, 0x5410), __byte_perm(rg1, ba1, 0x7632));
                    o[1] = make_uint4(__byte_perm(rg2, ba2, 0x5410), __byte_perm(rg2, ba2, 0x7632), __byte_perm(rg3, ba3, 0x5410), __byte_perm(rg3, ba3, 0x7632));
                }
            } else if (act) {
#pragma unroll
                for (int i = 0; i < 8; ++i) row[i * 4 + c] = (uint8_t)((i < 4 ? lo : hi) >> (8 * (i & 3)));
            }
        }
    }
}

// Shared memory: the AES round tables (1024 words), then one column of 64 words per thread (word z of thread t at z * THREADS + t).
// PMAX = 4 or 8 >= k + 1: only the first PMAX zigzag coefficients are computed (the rest of the transform is dead code) and
// the remainder comes from strong_bytes_half; PMAX = 64: any k.
template <int C, int PMAX = 64>
__global__ void __launch_bounds__(STRONG_THREADS) fragment_dct_strong_kernel(const __grid_constant__ DctParams p) {
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *sT = smem;
    load_aes_tables(sT);
    uint32_t *col = smem + AES_TABLE_WORDS + threadIdx.x;
    constexpr ZigzagTable ZZ = make_zigzag();
    StrongCoord S;
    if (!strong_decode<C>(p, (unsigned long long)blockIdx.x * STRONG_THREADS + threadIdx.x, S)) return;
    const int P = p.k + 1;
    const uint8_t *img = p.images + (size_t)S.n * p.image_stride;
    {   // steps 1-3: pixels -> DCT -> Part 1 (plaintext) into this thread's column, in zigzag order
        float v[64];
        load_block<C>(img, p.w, 8 * S.br, 8 * S.bc, S.ch, v);
        dct8x8(v);
#pragma unroll
        for (int z = 0; z < PMAX; ++z) col[z * STRONG_THREADS] = __float_as_uint(v[ZZ.pos[z]]);
    }
    uint32_t rows[16];
    if constexpr (PMAX < 64) {   // the remainder x - L, modulo 256
        uint32_t x[16];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const uint2 xr = strong_load_row<C>(img + ((size_t)(8 * S.br + r) * p.w + 8 * S.bc) * C, S.ch);
            x[2 * r] = xr.x; x[2 * r + 1] = xr.y;
        }
        int32_t m[PMAX];
        strong_scaled_q<PMAX>(col, STRONG_THREADS, P, -1, m);
        strong_bytes_half<0, PMAX, 0x00007ffeu>(x, m, P, reinterpret_cast<uint32_t(&)[8]>(rows[0]));
        strong_bytes_half<1, PMAX, 0x00007ffeu>(x, m, P, reinterpret_cast<uint32_t(&)[8]>(rows[8]));
    } else {
        int32_t acc[64];
        strong_low_pass(col, STRONG_THREADS, P, acc);
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const uint2 x = strong_load_row<C>(img + ((size_t)(8 * S.br + r) * p.w + 8 * S.bc) * C, S.ch);
            rows[2 * r] = strong_apply4<true>(x.x, acc[8 * r], acc[8 * r + 1], acc[8 * r + 2], acc[8 * r + 3]);
            rows[2 * r + 1] = strong_apply4<true>(x.y, acc[8 * r + 4], acc[8 * r + 5], acc[8 * r + 6], acc[8 * r + 7]);
        }
    }
    {   // XOR with SHA-512(Part 1), store the 64 public bytes of the block
        uint32_t ks[16];
        sha512_part1_keystream(col, STRONG_THREADS, P, ks);
        uint4 *dst = reinterpret_cast<uint4 *>(p.pub + (size_t)S.n * p.pub_stride + 64 * S.b);
#pragma unroll
        for (int i = 0; i < 4; ++i)
            dst[i] = make_uint4(rows[4 * i] ^ ks[4 * i], rows[4 * i + 1] ^ ks[4 * i + 1], rows[4 * i + 2] ^ ks[4 * i + 2], rows[4 * i + 3] ^ ks[4 * i + 3]);
    }
    {   // step 4: AES-128-CTR on Part 1, store
        uint32_t nonce[4];
        load_nonce(p, S.n, nonce);
        const unsigned long long w0 = (unsigned long long)S.b * P;
        strong_ctr_xor(p, sT, nonce, w0, P, col, STRONG_THREADS);
        uint32_t *dst = reinterpret_cast<uint32_t *>(p.priv + (size_t)S.n * p.priv_stride) + w0;
#pragma unroll 1
        for (int z = 0; z < P; ++z) dst[z] = col[z * STRONG_THREADS];
    }
}

template <int C, int PMAX = 64>
__global__ void __launch_bounds__(STRONG_THREADS) defragment_dct_strong_kernel(const __grid_constant__ DctParams p) {
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *sT = smem;
    load_aes_tables(sT);
    uint32_t *col = smem + AES_TABLE_WORDS + threadIdx.x;
    StrongCoord S;
    const bool act = strong_decode<C>(p, (unsigned long long)blockIdx.x * STRONG_THREADS + threadIdx.x, S);
    uint32_t rows[16];
    if (act) {
        const int P = p.k + 1;
        const unsigned long long w0 = (unsigned long long)S.b * P;
        const uint32_t *src = reinterpret_cast<const uint32_t *>(p.priv + (size_t)S.n * p.priv_stride) + w0;
#pragma unroll 1
        for (int z = 0; z < P; ++z) col[z * STRONG_THREADS] = __ldg(src + z);
        uint32_t nonce[4];
        load_nonce(p, S.n, nonce);
        strong_ctr_xor(p, sT, nonce, w0, P, col, STRONG_THREADS);   // Part 1 in plaintext
        uint32_t ks[16];
        sha512_part1_keystream(col, STRONG_THREADS, P, ks);
        const uint4 *q = reinterpret_cast<const uint4 *>(p.pub + (size_t)S.n * p.pub_stride + 64 * S.b);
        if constexpr (PMAX < 64) {
            uint32_t x[16];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const uint4 v = __ldg(q + i);
                x[4 * i] = v.x ^ ks[4 * i]; x[4 * i + 1] = v.y ^ ks[4 * i + 1]; x[4 * i + 2] = v.z ^ ks[4 * i + 2]; x[4 * i + 3] = v.w ^ ks[4 * i + 3];
            }
            int32_t m[PMAX];
            strong_scaled_q<PMAX>(col, STRONG_THREADS, P, 1, m);
            strong_bytes_half<0, PMAX, 0x00008000u>(x, m, P, reinterpret_cast<uint32_t(&)[8]>(rows[0]));
            strong_bytes_half<1, PMAX, 0x00008000u>(x, m, P, reinterpret_cast<uint32_t(&)[8]>(rows[8]));
        } else {
        int32_t acc[64];
        strong_low_pass(col, STRONG_THREADS, P, acc);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const uint4 x = __ldg(q + i);
            rows[4 * i] = strong_apply4<false>(x.x ^ ks[4 * i], acc[16 * i], acc[16 * i + 1], acc[16 * i + 2], acc[16 * i + 3]);
            rows[4 * i + 1] = strong_apply4<false>(x.y ^ ks[4 * i + 1], acc[16 * i + 4], acc[16 * i + 5], acc[16 * i + 6], acc[16 * i + 7]);
            rows[4 * i + 2] = strong_apply4<false>(x.z ^ ks[4 * i + 2], acc[16 * i + 8], acc[16 * i + 9], acc[16 * i + 10], acc[16 * i + 11]);
            rows[4 * i + 3] = strong_apply4<false>(x.w ^ ks[4 * i + 3], acc[16 * i + 12], acc[16 * i + 13], acc[16 * i + 14], acc[16 * i + 15]);
        }
        }
    }
    if (!act) { S.n = 0; S.ch = 0; S.br = 0; S.bc = 0; }
    store_block_packed<C>(p.images_out + (size_t)S.n * p.image_stride, p.w, 8 * S.br, 8 * S.bc, S.ch, act, rows);
}

}  // namespace feds
