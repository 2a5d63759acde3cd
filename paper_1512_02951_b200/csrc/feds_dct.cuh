// feds_dct.cuh — what the DCT-path kernels share (sm_100a): the parameter block, vector run access, pixel <-> float32 block load /
// store for the generic tile kernels, leaf geometry, per-image nonces, digest store. The kernels themselves live in
// feds_dct_tile.cuh (generic tile kernels, leaf-hash kernel), feds_dct_tma.cuh (bulk-copy tile kernels) and feds_dct_fused.cuh
// (warp-specialised fused kernels with digests).
#pragma once
#include "feds_device.cuh"

namespace feds {

static __device__ const AesTables g_aes = make_aes_tables();   // one copy per translation unit

constexpr int AES_TABLE_WORDS = 1024;

struct DctParams {
    const uint8_t *images;  // fragment: input images; defragment: unused
    uint8_t *images_out;    // defragment: output images
    size_t image_stride;
    uint8_t *priv;          // fragment: out; defragment: in
    size_t priv_stride;
    uint8_t *pub;
    size_t pub_stride;
    uint8_t *leaves;        // level-0 digests [n][2][nl][32] (or the final digest buffer when nl == 1)
    const uint8_t *d_nonces;  // device uint8[n][16], or nullptr: use nonce_be
    uint32_t nonce_be[4];
    uint32_t rk[44];
    int n_images, w, h, k;
    int nbr, nbc, nlr;
    unsigned leaves_per_image;  // C * nbr * nlr
    unsigned long long total_leaves;
    uint32_t one;     // = 1, opaque to the compiler (see sha256_compress_rolled_fma)
    uint32_t c128;    // = 128, opaque to the compiler (rep_lookup, feds_aes_rep.cuh)
    int pub_words;      // 32-bit words per block in the public fragment: 63 - k (first level) or 16 (strong level: 64 pixel bytes)
    int priv_words;     // 32-bit words per block in the private fragment for the leaf-hash kernels: k + 1, or 0 = skip (packed storage)
    // packed integer storage (feds_dct_packed.cuh)
    int ac_bits;                  // 11 or 8
    unsigned packed_group_bytes;  // 11 + k * ac_bits: bits per block = bytes per full group of 8 blocks
    size_t packed_row_bytes;      // private bytes per block row of one channel
    int generic_tiles;  // 1: digest-free path on the generic tile kernels even where the bulk-copy kernels apply (FEDS_FLAG_GENERIC_TILES)
};

// words per vector access of a coefficient run: the largest of {4, 2, 1} dividing P = k + 1 (then it divides Q = 64 - P too, and
// every run starts 4V-byte aligned)
__host__ __device__ inline int dct_vec_width(int k) { return ((k + 1) % 4 == 0) ? 4 : ((k + 1) % 2 == 0) ? 2 : 1; }

template <int V> struct VecT;
template <> struct VecT<1> { using type = uint32_t; };
template <> struct VecT<2> { using type = uint2; };
template <> struct VecT<4> { using type = uint4; };

template <int V>
__device__ __forceinline__ void vec_store(uint32_t *dst, const uint32_t (&x)[V]) {
    if (V == 1) dst[0] = x[0];
    else if (V == 2) *reinterpret_cast<uint2 *>(dst) = make_uint2(x[0], x[1]);
    else *reinterpret_cast<uint4 *>(dst) = make_uint4(x[0], x[1 % V], x[2 % V], x[3 % V]);
}
template <int V>
__device__ __forceinline__ void vec_load(const uint32_t *src, uint32_t (&x)[V]) {
    if (V == 1) x[0] = src[0];
    else if (V == 2) { const uint2 t = *reinterpret_cast<const uint2 *>(src); x[0] = t.x; x[1 % V] = t.y; }
    else { const uint4 t = *reinterpret_cast<const uint4 *>(src); x[0] = t.x; x[1 % V] = t.y; x[2 % V] = t.z; x[3 % V] = t.w; }
}
template <int V>
__device__ __forceinline__ void vec_load_global(const uint32_t *src, uint32_t (&x)[V]) {
    if (V == 1) x[0] = __ldg(src);
    else if (V == 2) { const uint2 t = __ldg(reinterpret_cast<const uint2 *>(src)); x[0] = t.x; x[1 % V] = t.y; }
    else { const uint4 t = __ldg(reinterpret_cast<const uint4 *>(src)); x[0] = t.x; x[1 % V] = t.y; x[2 % V] = t.z; x[3 % V] = t.w; }
}

template <typename T, bool GLOBAL>
__device__ __forceinline__ T ld_ro(const T *q) { return GLOBAL ? __ldg(q) : *q; }
// uint8 -> float32, exact: byte `pos` of `word` becomes the low mantissa byte of 2^23 (one PRMT), minus 2^23 (one FADD on the
// FMA pipe) -- instead of shift, mask and I2F on the ALU pipe.
__device__ __forceinline__ float byte_to_float(uint32_t word, int pos) {
    return __uint_as_float(__byte_perm(word, 0x4B000000u, 0x7540 + pos)) - 8388608.0f;
}
// four float32 -> four uint8 packed little-endian: round to nearest even, saturate to [0,255] (A5). ptxas fuses each
// pair of conversions with its cvt.pack into one F2IP.U8.F32: two instructions for four pixels.
__device__ __forceinline__ uint32_t pack4_u8(float a, float b, float c, float d) {
    int ia, ib, ic, id;
    asm("cvt.rni.s32.f32 %0, %1;" : "=r"(ia) : "f"(a));
    asm("cvt.rni.s32.f32 %0, %1;" : "=r"(ib) : "f"(b));
    asm("cvt.rni.s32.f32 %0, %1;" : "=r"(ic) : "f"(c));
    asm("cvt.rni.s32.f32 %0, %1;" : "=r"(id) : "f"(d));
    uint32_t hi, r;
    asm("cvt.pack.sat.u8.s32.b32 %0, %1, %2, %3;" : "=r"(hi) : "r"(id), "r"(ic), "r"(0));
    asm("cvt.pack.sat.u8.s32.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(ib), "r"(ia), "r"(hi));
    return r;
}
// GLOBAL = false: `img` is a tile of pixel rows staged in shared memory (same interleaved layout, pitch w pixels)
template <int C, bool GLOBAL = true>
__device__ __forceinline__ void load_block(const uint8_t *__restrict__ img, int w, int y0, int x0, int c, float (&v)[64]) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const uint8_t *row = img + ((size_t)(y0 + r) * w + x0) * C;
        if (C == 1) {
            const uint2 q = ld_ro<uint2, GLOBAL>(reinterpret_cast<const uint2 *>(row));
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                v[8 * r + i] = byte_to_float(q.x, i);
                v[8 * r + 4 + i] = byte_to_float(q.y, i);
            }
        } else if (C == 3) {
            const uint2 q0 = ld_ro<uint2, GLOBAL>(reinterpret_cast<const uint2 *>(row));
            const uint2 q1 = ld_ro<uint2, GLOBAL>(reinterpret_cast<const uint2 *>(row) + 1);
            const uint2 q2 = ld_ro<uint2, GLOBAL>(reinterpret_cast<const uint2 *>(row) + 2);
            // shift the 24-byte row right by c bytes (c is fixed per thread), then the wanted bytes sit at 3*i
            const uint32_t wd[7] = {q0.x, q0.y, q1.x, q1.y, q2.x, q2.y, 0u};
            uint32_t ws[6];
#pragma unroll
            for (int j = 0; j < 6; ++j) ws[j] = __funnelshift_r(wd[j], wd[j + 1], 8 * c);
#pragma unroll
            for (int i = 0; i < 8; ++i) v[8 * r + i] = byte_to_float(ws[(3 * i) >> 2], (3 * i) & 3);
        } else {
            const uint4 a = ld_ro<uint4, GLOBAL>(reinterpret_cast<const uint4 *>(row));
            const uint4 b = ld_ro<uint4, GLOBAL>(reinterpret_cast<const uint4 *>(row) + 1);
            const uint32_t wd[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
            for (int i = 0; i < 8; ++i) v[8 * r + i] = __uint_as_float(__byte_perm(wd[i], 0x4B000000u, 0x7540u + (uint32_t)c)) - 8388608.0f;
        }
    }
}

// Round to nearest even, clamp to [0,255] (A5) and store the 8x8 block of channel c.
// C == 1: one 8-byte store per row. C == 3 / 4: the C lanes holding the channels of one pixel strip are adjacent
// (channel-fastest leaf order); lane c == 0 gathers its partners' rows with shuffles, interleaves them with byte
// permutes and stores whole 8*C-byte row segments. Strips whose C lanes straddle a warp fall back to byte stores.
template <int C>
__device__ __forceinline__ void store_block(uint8_t *__restrict__ img, int w, int y0, int x0, int c, bool act, const float (&v)[64]) {
    const int lane = threadIdx.x & 31;
    bool complete = true;
    if (C > 1) {
        // all C lanes of my strip are in this warp, and all are active
        const int l0 = lane - c;
        complete = (l0 >= 0) && (l0 + C - 1 <= 31);
        const unsigned actmask = __ballot_sync(0xffffffffu, act);
        if (complete) complete = ((actmask >> l0) & ((1u << C) - 1u)) == ((1u << C) - 1u);
    }
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const uint32_t lo = pack4_u8(v[8 * r], v[8 * r + 1], v[8 * r + 2], v[8 * r + 3]);
        const uint32_t hi = pack4_u8(v[8 * r + 4], v[8 * r + 5], v[8 * r + 6], v[8 * r + 7]);
        uint8_t *row = img + ((size_t)(y0 + r) * w + x0) * C;  // start of the strip's 8*C-byte row segment
        if (C == 1) {
            if (act) *reinterpret_cast<uint2 *>(row) = make_uint2(lo, hi);
        } else if (C == 3) {
            const uint32_t glo = __shfl_down_sync(0xffffffffu, lo, 1), ghi = __shfl_down_sync(0xffffffffu, hi, 1);
            const uint32_t blo = __shfl_down_sync(0xffffffffu, lo, 2), bhi = __shfl_down_sync(0xffffffffu, hi, 2);
            if (complete) {
                if (c == 0) {
                    // bytes: R = lo/hi, G = glo/ghi, B = blo/bhi; output RGB RGB ...
                    const uint32_t rg0 = __byte_perm(lo, glo, 0x5140);   // R0 G0 R1 G1
                    const uint32_t rg1 = __byte_perm(lo, glo, 0x7362);   // R2 G2 R3 G3
                    const uint32_t rg2 = __byte_perm(hi, ghi, 0x5140);   // R4 G4 R5 G5
                    const uint32_t rg3 = __byte_perm(hi, ghi, 0x7362);   // R6 G6 R7 G7
                    const uint32_t w0 = __byte_perm(rg0, blo, 0x2410);   // R0 G0 B0 R1
                    const uint32_t w1 = __byte_perm(__byte_perm(rg0, blo, 0x0053), rg1, 0x5410);  // G1 B1 R2 G2
                    const uint32_t w2 = __byte_perm(rg1, blo, 0x7326);   // B2 R3 G3 B3
                    const uint32_t w3 = __byte_perm(rg2, bhi, 0x2410);
                    const uint32_t w4 = __byte_perm(__byte_perm(rg2, bhi, 0x0053), rg3, 0x5410);
                    const uint32_t w5 = __byte_perm(rg3, bhi, 0x7326);
                    uint2 *o = reinterpret_cast<uint2 *>(row);
                    o[0] = make_uint2(w0, w1);
                    o[1] = make_uint2(w2, w3);
                    o[2] = make_uint2(w4, w5);
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
                    o[0] = make_uint4(__byte_perm(rg0, ba0, 0x5410), __byte_perm(rg0, ba0, 0x7632), __byte_perm(rg1, ba1, 0x5410),
                                      __byte_perm(rg1, ba1, 0x7632));
                    o[1] = make_uint4(__byte_perm(rg2, ba2, 0x5410), __byte_perm(rg2, ba2, 0x7632), __byte_perm(rg3, ba3, 0x5410),
                                      __byte_perm(rg3, ba3, 0x7632));
                }
            } else if (act) {
#pragma unroll
                for (int i = 0; i < 8; ++i) row[i * 4 + c] = (uint8_t)((i < 4 ? lo : hi) >> (8 * (i & 3)));
            }
        }
    }
}

struct LeafCoord {
    bool valid;
    int n, c, br, g, nblk;
    unsigned li;           // leaf index in fragment order
    unsigned b0;           // linear block index of the leaf's first block
};

template <int C>
__device__ __forceinline__ LeafCoord decode_leaf(const DctParams &p, unsigned long long gid) {
    LeafCoord L;
    L.valid = gid < p.total_leaves;
    const unsigned long long g2 = L.valid ? gid : 0;
    L.n = (int)(g2 / p.leaves_per_image);
    unsigned rem = (unsigned)(g2 % p.leaves_per_image);
    L.c = (int)(rem % C);            // channel fastest: the C leaves of one pixel strip sit in adjacent lanes
    rem /= C;
    L.g = (int)(rem % (unsigned)p.nlr);
    L.br = (int)(rem / (unsigned)p.nlr);
    L.li = (unsigned)((L.c * p.nbr + L.br) * p.nlr + L.g);
    L.b0 = (unsigned)((L.c * p.nbr + L.br) * p.nbc + L.g * G_BLOCKS);
    const int left = p.nbc - L.g * G_BLOCKS;
    L.nblk = L.valid ? (left < G_BLOCKS ? left : G_BLOCKS) : 0;
    return L;
}

__device__ __forceinline__ void load_nonce(const DctParams &p, int n, uint32_t (&nonce)[4]) {
    if (p.d_nonces) {
        const uint4 q = __ldg(reinterpret_cast<const uint4 *>(p.d_nonces) + n);
        nonce[0] = bswap32(q.x); nonce[1] = bswap32(q.y); nonce[2] = bswap32(q.z); nonce[3] = bswap32(q.w);
    } else {
        nonce[0] = p.nonce_be[0]; nonce[1] = p.nonce_be[1]; nonce[2] = p.nonce_be[2]; nonce[3] = p.nonce_be[3];
    }
}

__device__ __forceinline__ void store_digest(uint8_t *dst, const uint32_t (&H)[8]) {
    uint4 a, b;
    a.x = bswap32(H[0]); a.y = bswap32(H[1]); a.z = bswap32(H[2]); a.w = bswap32(H[3]);
    b.x = bswap32(H[4]); b.y = bswap32(H[5]); b.z = bswap32(H[6]); b.w = bswap32(H[7]);
    reinterpret_cast<uint4 *>(dst)[0] = a;
    reinterpret_cast<uint4 *>(dst)[1] = b;
}

__device__ __forceinline__ void load_aes_tables(uint32_t *sT) {
    const uint32_t *src = &g_aes.T[0][0];
    for (int i = threadIdx.x; i < AES_TABLE_WORDS; i += blockDim.x) sT[i] = src[i];
    __syncthreads();
}

}  // namespace feds
