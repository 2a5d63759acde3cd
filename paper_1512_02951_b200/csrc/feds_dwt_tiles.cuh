// feds_dwt_tiles.cuh — the report's own DWT design (PAPER.md 6.9.3-6.9.4, Figure 18), sm_100a:
// selective encryption of 8x8 tiles with two levels of the integer 5/3 transform. Level 1 (the four LL2 coefficients) goes under
// AES-128-CTR, level 2 (HL2, LH2, HH2) under SHA-256(level 1 || key || IV), level 3 (HL1, LH1, HH1) under SHA-512(level 2 || key ||
// IV); 10-bit two's complement fields, 11 for HH2: 5 + 16 + 60 bytes per tile. Byte format: DESIGN.md 2.5 (readings T1-T7).
//
// One thread per (tile, channel): the whole tile -- 64 coefficients, both hashes, the packing -- lives in its registers; the two
// hash compressions (one SHA-256 block, one SHA-512 block) are what a tile costs. Pixels move as in the strong-level kernels.
#pragma once
#include "feds_dct_strong.cuh"

namespace feds {

constexpr int TILES_THREADS = 128;

// 1-D 5/3 analysis / synthesis of 8 and of 4 samples in place, whole-sample symmetric extension: out = [s | d]
__device__ __forceinline__ void lift8_fwd(int &x0, int &x1, int &x2, int &x3, int &x4, int &x5, int &x6, int &x7) {
    const int d0 = x1 - ((x0 + x2) >> 1), d1 = x3 - ((x2 + x4) >> 1), d2 = x5 - ((x4 + x6) >> 1), d3 = x7 - ((x6 + x6) >> 1);
    const int s0 = x0 + ((d0 + d0 + 2) >> 2), s1 = x2 + ((d0 + d1 + 2) >> 2), s2 = x4 + ((d1 + d2 + 2) >> 2), s3 = x6 + ((d2 + d3 + 2) >> 2);
    x0 = s0; x1 = s1; x2 = s2; x3 = s3; x4 = d0; x5 = d1; x6 = d2; x7 = d3;
}
__device__ __forceinline__ void lift8_inv(int &y0, int &y1, int &y2, int &y3, int &y4, int &y5, int &y6, int &y7) {
    const int e0 = y0 - ((y4 + y4 + 2) >> 2), e1 = y1 - ((y4 + y5 + 2) >> 2), e2 = y2 - ((y5 + y6 + 2) >> 2), e3 = y3 - ((y6 + y7 + 2) >> 2);
    const int o0 = y4 + ((e0 + e1) >> 1), o1 = y5 + ((e1 + e2) >> 1), o2 = y6 + ((e2 + e3) >> 1), o3 = y7 + ((e3 + e3) >> 1);
    y0 = e0; y1 = o0; y2 = e1; y3 = o1; y4 = e2; y5 = o2; y6 = e3; y7 = o3;
}
__device__ __forceinline__ void lift4_fwd(int &x0, int &x1, int &x2, int &x3) {
    const int d0 = x1 - ((x0 + x2) >> 1), d1 = x3 - ((x2 + x2) >> 1);
    const int s0 = x0 + ((d0 + d0 + 2) >> 2), s1 = x2 + ((d0 + d1 + 2) >> 2);
    x0 = s0; x1 = s1; x2 = d0; x3 = d1;
}
__device__ __forceinline__ void lift4_inv(int &y0, int &y1, int &y2, int &y3) {
    const int e0 = y0 - ((y2 + y2 + 2) >> 2), e1 = y1 - ((y2 + y3 + 2) >> 2);
    const int o0 = y2 + ((e0 + e1) >> 1), o1 = y3 + ((e1 + e1) >> 1);
    y0 = e0; y1 = o0; y2 = e1; y3 = o1;
}
// two levels on an 8x8 tile held row-major in t[64]: rows then columns (T1)
__device__ __forceinline__ void tile_dwt_fwd(int (&t)[64]) {
#pragma unroll
    for (int r = 0; r < 8; ++r) lift8_fwd(t[8 * r], t[8 * r + 1], t[8 * r + 2], t[8 * r + 3], t[8 * r + 4], t[8 * r + 5], t[8 * r + 6], t[8 * r + 7]);
#pragma unroll
    for (int c = 0; c < 8; ++c) lift8_fwd(t[c], t[8 + c], t[16 + c], t[24 + c], t[32 + c], t[40 + c], t[48 + c], t[56 + c]);
#pragma unroll
    for (int r = 0; r < 4; ++r) lift4_fwd(t[8 * r], t[8 * r + 1], t[8 * r + 2], t[8 * r + 3]);
#pragma unroll
    for (int c = 0; c < 4; ++c) lift4_fwd(t[c], t[8 + c], t[16 + c], t[24 + c]);
}
__device__ __forceinline__ void tile_dwt_inv(int (&t)[64]) {
#pragma unroll
    for (int c = 0; c < 4; ++c) lift4_inv(t[c], t[8 + c], t[16 + c], t[24 + c]);
#pragma unroll
    for (int r = 0; r < 4; ++r) lift4_inv(t[8 * r], t[8 * r + 1], t[8 * r + 2], t[8 * r + 3]);
#pragma unroll
    for (int c = 0; c < 8; ++c) lift8_inv(t[c], t[8 + c], t[16 + c], t[24 + c], t[32 + c], t[40 + c], t[48 + c], t[56 + c]);
#pragma unroll
    for (int r = 0; r < 8; ++r) lift8_inv(t[8 * r], t[8 * r + 1], t[8 * r + 2], t[8 * r + 3], t[8 * r + 4], t[8 * r + 5], t[8 * r + 6], t[8 * r + 7]);
}

// position in the row-major tile of coefficient i in level order (T2), and its field width (T3)
__host__ __device__ constexpr int tiles_pos(int i) {
    return i < 4 ? 8 * (i / 2) + i % 2                       // LL2
         : i < 8 ? 8 * ((i - 4) / 2) + 2 + (i - 4) % 2       // HL2
         : i < 12 ? 8 * (2 + (i - 8) / 2) + (i - 8) % 2      // LH2
         : i < 16 ? 8 * (2 + (i - 12) / 2) + 2 + (i - 12) % 2   // HH2
         : i < 32 ? 8 * ((i - 16) / 4) + 4 + (i - 16) % 4    // HL1
         : i < 48 ? 8 * (4 + (i - 32) / 4) + (i - 32) % 4    // LH1
         : 8 * (4 + (i - 48) / 4) + 4 + (i - 48) % 4;        // HH1
}
__host__ __device__ constexpr int tiles_bits(int i) { return (i >= 12 && i < 16) ? 11 : 10; }

// fields of coefficients [LO, HI) <-> a little-endian bit stream held in N 32-bit words (all positions are compile-time constants)
template <int LO, int HI, int N>
__device__ __forceinline__ void tiles_pack(const int (&t)[64], uint32_t (&w)[N]) {
#pragma unroll
    for (int i = 0; i < N; ++i) w[i] = 0u;
    int pos = 0;
#pragma unroll
    for (int i = LO; i < HI; ++i) {
        const int b = tiles_bits(i);
        const uint32_t f = (uint32_t)t[tiles_pos(i)] & ((1u << b) - 1u);
        w[pos >> 5] |= f << (pos & 31);
        if ((pos & 31) + b > 32) w[(pos >> 5) + 1] |= f >> (32 - (pos & 31));
        pos += b;
    }
}
template <int LO, int HI, int N>
__device__ __forceinline__ void tiles_unpack(const uint32_t (&w)[N], int (&t)[64]) {
    int pos = 0;
#pragma unroll
    for (int i = LO; i < HI; ++i) {
        const int b = tiles_bits(i);
        uint32_t f = w[pos >> 5] >> (pos & 31);
        if ((pos & 31) + b > 32) f |= w[(pos >> 5) + 1] << (32 - (pos & 31));
        t[tiles_pos(i)] = (int)(f << (32 - b)) >> (32 - b);   // sign-extend the two's complement field
        pos += b;
    }
}

struct TilesSecrets {
    uint32_t key[4], iv[4];   // little-endian words of the 16 key / nonce bytes
};
// K2 = SHA-256(level-1 bytes[5] || key || IV): one block; the first 16 digest bytes as 4 words in memory order (T4)
__device__ __forceinline__ void tiles_k2(uint32_t l1lo, uint32_t l1hi, const TilesSecrets &S, uint32_t one, uint32_t (&k2)[4]) {
    const uint32_t K[4] = {S.key[0], S.key[1], S.key[2], S.key[3]}, V[4] = {S.iv[0], S.iv[1], S.iv[2], S.iv[3]};
    uint32_t le[10];   // the 37 message bytes + the 0x80 marker as little-endian words
    le[0] = l1lo;
    le[1] = (l1hi & 0xffu) | (K[0] << 8);
    le[2] = (K[0] >> 24) | (K[1] << 8);
    le[3] = (K[1] >> 24) | (K[2] << 8);
    le[4] = (K[2] >> 24) | (K[3] << 8);
    le[5] = (K[3] >> 24) | (V[0] << 8);
    le[6] = (V[0] >> 24) | (V[1] << 8);
    le[7] = (V[1] >> 24) | (V[2] << 8);
    le[8] = (V[2] >> 24) | (V[3] << 8);
    le[9] = (V[3] >> 24) | (0x80u << 8);
    uint32_t w[16], H[8];
#pragma unroll
    for (int i = 0; i < 10; ++i) w[i] = bswap32(le[i]);
#pragma unroll
    for (int i = 10; i < 15; ++i) w[i] = 0u;
    w[15] = 37u * 8u;
    sha256_init(H);
    sha256_compress_rolled_fma(H, w, one);
#pragma unroll
    for (int i = 0; i < 4; ++i) k2[i] = bswap32(H[i]);
}
// K3 = SHA-512(level-2 bytes[16] || key || IV): one block; the first 60 digest bytes as 15 words in memory order
__device__ __forceinline__ void tiles_k3(const uint32_t (&l2)[4], const TilesSecrets &S, uint32_t (&k3)[15]) {
    const uint32_t le[12] = {l2[0], l2[1], l2[2], l2[3], S.key[0], S.key[1], S.key[2], S.key[3], S.iv[0], S.iv[1], S.iv[2], S.iv[3]};
    uint64_t H[8] = {0x6a09e667f3bcc908ULL, 0xbb67ae8584caa73bULL, 0x3c6ef372fe94f82bULL, 0xa54ff53a5f1d36f1ULL,
                     0x510e527fade682d1ULL, 0x9b05688c2b3e6c1fULL, 0x1f83d9abfb41bd6bULL, 0x5be0cd19137e2179ULL};
    uint64_t w[16];
#pragma unroll
    for (int j = 0; j < 6; ++j) w[j] = ((uint64_t)bswap32(le[2 * j]) << 32) | bswap32(le[2 * j + 1]);
    w[6] = 0x8000000000000000ULL;
#pragma unroll
    for (int j = 7; j < 15; ++j) w[j] = 0ULL;
    w[15] = 48ull * 8ull;
    sha512_compress(H, w);
#pragma unroll
    for (int i = 0; i < 7; ++i) { k3[2 * i] = bswap32((uint32_t)(H[i] >> 32)); k3[2 * i + 1] = bswap32((uint32_t)H[i]); }
    k3[14] = bswap32((uint32_t)(H[7] >> 32));
}
__device__ __forceinline__ void tiles_secrets(const DctParams &p, int n, TilesSecrets &S) {
#pragma unroll
    for (int i = 0; i < 4; ++i) S.key[i] = p.rk[i];   // round key 0 is the key itself, as little-endian column words
    if (p.d_nonces) {
        const uint4 q = __ldg(reinterpret_cast<const uint4 *>(p.d_nonces) + n);
        S.iv[0] = q.x; S.iv[1] = q.y; S.iv[2] = q.z; S.iv[3] = q.w;
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) S.iv[i] = bswap32(p.nonce_be[i]);
    }
}
// AES-128-CTR keystream bytes [off, off + 5) of the image's level-1 section, as (low 4 bytes, 5th byte)
template <typename Tab>
__device__ __forceinline__ void tiles_ctr5(const DctParams &p, const Tab sT, int n, unsigned long long off, uint32_t &lo, uint32_t &hi) {
    uint32_t nonce[4];
    load_nonce(p, n, nonce);
    const unsigned long long blk = off >> 4;
    const int r = (int)(off & 15);
    uint32_t a[4], b[4] = {0u, 0u, 0u, 0u};
    ctr_block(nonce, blk, a);
    aes128_encrypt(sT, p.rk, a);
    if (r > 11) { ctr_block(nonce, blk + 1, b); aes128_encrypt(sT, p.rk, b); }   // the five bytes straddle two counter blocks
    // bytes r .. r + 4 of the 32-byte window a || b: three consecutive words, funnel-shifted by the byte offset
    const int wi = r >> 2, sh = 8 * (r & 3);
    uint32_t w0, w1, w2;
    if (wi == 0) { w0 = a[0]; w1 = a[1]; w2 = a[2]; }
    else if (wi == 1) { w0 = a[1]; w1 = a[2]; w2 = a[3]; }
    else if (wi == 2) { w0 = a[2]; w1 = a[3]; w2 = b[0]; }
    else { w0 = a[3]; w1 = b[0]; w2 = b[1]; }
    lo = __funnelshift_r(w0, w1, sh);
    hi = __funnelshift_r(w1, w2, sh) & 0xffu;
}

struct TilesCoord {
    int n, ch, tr, tc;
    unsigned long long t;   // tile index in fragment order
    unsigned long long T;   // tiles per image
};
template <int C>
__device__ __forceinline__ bool tiles_decode(const DctParams &p, unsigned long long gid, TilesCoord &S) {
    S.T = (unsigned long long)C * p.nbr * p.nbc;
    if (gid >= S.T * p.n_images) return false;
    S.n = (int)(gid / S.T);
    unsigned rem = (unsigned)(gid % S.T);
    S.ch = (int)(rem % C);   // channel fastest: the C lanes of one pixel strip are adjacent (store_block_packed)
    rem /= C;
    S.tc = (int)(rem % (unsigned)p.nbc);
    S.tr = (int)(rem / (unsigned)p.nbc);
    S.t = ((unsigned long long)S.ch * p.nbr + S.tr) * p.nbc + S.tc;
    return true;
}

template <int C>
__global__ void __launch_bounds__(TILES_THREADS) fragment_dwt_tiles_kernel(const __grid_constant__ DctParams p) {
    __shared__ uint32_t sT[AES_TABLE_WORDS];
    load_aes_tables(sT);
    TilesCoord S;
    if (!tiles_decode<C>(p, (unsigned long long)blockIdx.x * TILES_THREADS + threadIdx.x, S)) return;
    const uint8_t *img = p.images + (size_t)S.n * p.image_stride;
    int t[64];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const uint2 x = strong_load_row<C>(img + ((size_t)(8 * S.tr + r) * p.w + 8 * S.tc) * C, S.ch);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            t[8 * r + i] = (int)((x.x >> (8 * i)) & 255u) - 128;
            t[8 * r + 4 + i] = (int)((x.y >> (8 * i)) & 255u) - 128;
        }
    }
    tile_dwt_fwd(t);
    uint32_t l1[2], l2[4], l3[15];
    tiles_pack<0, 4, 2>(t, l1);
    tiles_pack<4, 16, 4>(t, l2);
    tiles_pack<16, 64, 15>(t, l3);
    TilesSecrets K;
    tiles_secrets(p, S.n, K);
    uint32_t k2[4], k3[15];
    tiles_k2(l1[0], l1[1], K, p.one, k2);
    tiles_k3(l2, K, k3);
    uint8_t *priv = p.priv + (size_t)S.n * p.priv_stride;
    *reinterpret_cast<uint4 *>(priv + 16 * S.t) = make_uint4(l2[0] ^ k2[0], l2[1] ^ k2[1], l2[2] ^ k2[2], l2[3] ^ k2[3]);
    uint32_t *pub = reinterpret_cast<uint32_t *>(p.pub + (size_t)S.n * p.pub_stride + 60 * S.t);
#pragma unroll
    for (int i = 0; i < 15; ++i) pub[i] = l3[i] ^ k3[i];
    uint32_t klo, khi;
    tiles_ctr5(p, sT, S.n, 5ull * S.t, klo, khi);
    const uint32_t clo = l1[0] ^ klo, chi = (l1[1] ^ khi) & 0xffu;
    uint8_t *a = priv + 16 * S.T + 5 * S.t;
    a[0] = (uint8_t)clo; a[1] = (uint8_t)(clo >> 8); a[2] = (uint8_t)(clo >> 16); a[3] = (uint8_t)(clo >> 24); a[4] = (uint8_t)chi;
}

template <int C>
__global__ void __launch_bounds__(TILES_THREADS) defragment_dwt_tiles_kernel(const __grid_constant__ DctParams p) {
    __shared__ uint32_t sT[AES_TABLE_WORDS];
    load_aes_tables(sT);
    TilesCoord S;
    const bool act = tiles_decode<C>(p, (unsigned long long)blockIdx.x * TILES_THREADS + threadIdx.x, S);
    uint32_t rows[16];
    if (act) {
        const uint8_t *priv = p.priv + (size_t)S.n * p.priv_stride;
        const uint8_t *a = priv + 16 * S.T + 5 * S.t;
        uint32_t l1[2], l2[4], l3[15];
        uint32_t klo, khi;
        tiles_ctr5(p, sT, S.n, 5ull * S.t, klo, khi);
        l1[0] = ((uint32_t)a[0] | ((uint32_t)a[1] << 8) | ((uint32_t)a[2] << 16) | ((uint32_t)a[3] << 24)) ^ klo;
        l1[1] = ((uint32_t)a[4] ^ khi) & 0xffu;
        TilesSecrets K;
        tiles_secrets(p, S.n, K);
        uint32_t k2[4], k3[15];
        tiles_k2(l1[0], l1[1], K, p.one, k2);
        const uint4 q = __ldg(reinterpret_cast<const uint4 *>(priv + 16 * S.t));
        l2[0] = q.x ^ k2[0]; l2[1] = q.y ^ k2[1]; l2[2] = q.z ^ k2[2];
        l2[3] = (q.w ^ k2[3]) & 0x0fffffffu;   // the four pad bits of the 124-bit stream are zero in the plaintext (T3)
        tiles_k3(l2, K, k3);
        const uint32_t *pub = reinterpret_cast<const uint32_t *>(p.pub + (size_t)S.n * p.pub_stride + 60 * S.t);
#pragma unroll
        for (int i = 0; i < 15; ++i) l3[i] = __ldg(pub + i) ^ k3[i];
        int t[64];
        tiles_unpack<0, 4, 2>(l1, t);
        tiles_unpack<4, 16, 4>(l2, t);
        tiles_unpack<16, 64, 15>(l3, t);
        tile_dwt_inv(t);
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            uint32_t lo = 0u, hi = 0u;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                lo |= (uint32_t)min(max(t[8 * r + i] + 128, 0), 255) << (8 * i);
                hi |= (uint32_t)min(max(t[8 * r + 4 + i] + 128, 0), 255) << (8 * i);
            }
            rows[2 * r] = lo; rows[2 * r + 1] = hi;
        }
    }
    if (!act) { S.n = 0; S.ch = 0; S.tr = 0; S.tc = 0; }
    store_block_packed<C>(p.images_out + (size_t)S.n * p.image_stride, p.w, 8 * S.tr, 8 * S.tc, S.ch, act, rows);
}

}  // namespace feds
