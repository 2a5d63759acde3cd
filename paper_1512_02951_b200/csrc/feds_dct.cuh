// feds_dct.cuh — the fused fragment kernel of the DCT path and the block load / store /
// slot helpers the other DCT kernels share (feds_dct_tile.cuh: digest-free kernels, leaf-hash kernel), sm_100a.
//
// One thread owns one Merkle leaf = up to G consecutive 8x8 blocks of one block row of one channel
// (DESIGN.md 2.1). For each block it: loads the 8x8 pixels, runs the separable FP32 DCT in 64 registers,
// splits the coefficients in zigzag order into its private / public words, AES-128-CTR-encrypts the private
// words (shared-memory T-tables, sequential keystream along the leaf), writes both runs to HBM, and absorbs the
// stored bytes of both fragments into two running SHA-256 states fed from a per-lane shared-memory slot (one
// inlined compression site). Pixels are read once; coefficients are written once; only 2 x 32 B of leaf digest
// per leaf go to the workspace.
//
// Template parameter V = words per vector access of a coefficient run, the largest of {4, 2, 1} dividing
// P = k+1 (then it divides Q = 64-P too, and every run starts 4V-byte aligned):
//   V = 4 / 2 : each lane moves its own runs with 128 / 64-bit accesses straight from / to registers; no warp
//               cooperation, no barrier in the block loop.
//   k + 1 odd : 4-byte runs would scatter 64 stores per block over 32 lines each; the host routes those k to the tile
//               kernel followed by the leaf-hash kernel (feds_dct_tile.cuh), which measured 2-4 % faster than a
//               warp-cooperative copy inside this kernel did.
#pragma once
#include "feds_device.cuh"

namespace feds {

static __device__ const AesTables g_aes = make_aes_tables();   // one copy per translation unit

constexpr int DCT_THREADS = 512;     // one persistent CTA per SM: 16 warps, 4 per scheduler (8 warps when the slots of 16 do not fit)
constexpr int DCT_CTAS_PER_SM = 1;
constexpr size_t DCT_SMEM_MAX = 227 * 1024;
constexpr int AES_TABLE_WORDS = 1024;
constexpr int CA = 16;  // carry area: a SHA-256 block is 16 words, at most 15 (16 - V) words wait between blocks

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
    int slot_stride;  // words per lane slot
    uint32_t one;     // = 1, opaque to the compiler (see sha256_compress_rolled_fma)
    unsigned n_groups;  // ceil(total_leaves / 32): one group = the 32 leaves one warp owns at a time
    // warp-specialised kernels (feds_dct_ws.cuh)
    unsigned ws_n_sg;   // strip groups: ceil(n_images * nbr * nlr / 32)
    int ws_ahead;       // slabs a worker may run in front of its slowest hash warp
    uint32_t c128;      // = 128, opaque to the compiler (ws_lookup)
    int generic_tiles;  // 1: digest-free path on the generic tile kernels even where the bulk-copy kernels apply (FEDS_FLAG_GENERIC_TILES)
};

// Slot layout (word offsets in a lane's slot), P private and Q = 64 - P public words per block:
//   [0, 16)        private carry        [16, 16+P)       private words of the current block, index z
//   [16+P, 32+P)   public carry         [32+P, 96)       public words of the current block, index z (address 32 + z)
// plus slack so that the <= 32 padding words of the final phase fit behind the public carry area.
// The stride makes per-lane V-word accesses conflict-free: odd (V=1), 2 mod 4 (V=2), 4 mod 8 (V=4).
__host__ __device__ inline int dct_vec_width(int k) { return ((k + 1) % 4 == 0) ? 4 : ((k + 1) % 2 == 0) ? 2 : 1; }
__host__ __device__ inline int dct_slot_words(int k) {
    const int Q = 63 - k, V = dct_vec_width(k);
    int wds = 2 * CA + 64 + (Q < 32 ? 32 - Q : 0) + 8;  // + 8: the waiting stream's chaining value (dct_stash_offset)
    while (wds % (2 * V) != V) ++wds;
    return wds;
}

__host__ __device__ inline int dct_stash_offset(int k) { const int Q = 63 - k; return 2 * CA + 64 + (Q < 32 ? 32 - Q : 0); }

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

// One SHA-256 stream living in a lane's slot: `carry` words wait at [base+16-carry, base+16), `fresh` new words
// were just written at [base+16, base+16+fresh). Compress every full 16-word block, slide the rest down.
struct ShaMeta {
    int base;
    int carry;
    int fresh;
    unsigned total_words;
};
struct ShaStream {
    uint32_t H[8];
    int base;
    int carry;
    int fresh;
    unsigned total_words;  // message length of the whole leaf in 32-bit words (0: stream unused)
};

// Only the stream being absorbed keeps its chaining value in registers; the other one's waits in the lane's slot at
// word offset `hoff` (8 words). 16 fewer live registers across the compression loop than a register swap.
template <int V>
__device__ __forceinline__ void swap_streams(uint32_t *my, int hoff, ShaStream &a, ShaMeta &b) {
#pragma unroll
    for (int i = 0; i < 8; i += V) {
        uint32_t t[V], u[V];
        vec_load<V>(my + hoff + i, t);
#pragma unroll
        for (int j = 0; j < V; ++j) u[j] = a.H[i + j];
        vec_store<V>(my + hoff + i, u);
#pragma unroll
        for (int j = 0; j < V; ++j) a.H[i + j] = t[j];
    }
    int t;
    t = a.base; a.base = b.base; b.base = t;
    t = a.carry; a.carry = b.carry; b.carry = t;
    t = a.fresh; a.fresh = b.fresh; b.fresh = t;
    const unsigned u = a.total_words; a.total_words = b.total_words; b.total_words = u;
}
template <int V>
__device__ __forceinline__ void stash_init(uint32_t *my, int hoff) {
    uint32_t H[8];
    sha256_init(H);
#pragma unroll
    for (int i = 0; i < 8; i += V) {
        uint32_t u[V];
#pragma unroll
        for (int j = 0; j < V; ++j) u[j] = H[i + j];
        vec_store<V>(my + hoff + i, u);
    }
}
template <int V>
__device__ __forceinline__ void stash_read(const uint32_t *my, int hoff, uint32_t (&H)[8]) {
#pragma unroll
    for (int i = 0; i < 8; i += V) {
        uint32_t t[V];
        vec_load<V>(my + hoff + i, t);
#pragma unroll
        for (int j = 0; j < V; ++j) H[i + j] = t[j];
    }
}

// Append the FIPS 180-4 5.1.1 padding for a message of `total_words` 32-bit words after the carried words.
// Slot words are little-endian data words (byte-swapped when loaded into W), so the padding is written pre-swapped.
__device__ __forceinline__ void write_padding(uint32_t *my, ShaStream &s) {
    const int n = s.carry;
    int tot = n + 3;                      // 0x80 word + 64-bit length
    tot = (tot + 15) & ~15;               // 16 or 32
    const int fresh = tot - n;
    uint32_t *dst = my + s.base + CA;
    dst[0] = 0x00000080u;
    for (int i = 1; i < fresh - 2; ++i) dst[i] = 0u;
    const unsigned long long bits = (unsigned long long)s.total_words * 32ull;
    dst[fresh - 2] = bswap32((uint32_t)(bits >> 32));
    dst[fresh - 1] = bswap32((uint32_t)bits);
    s.fresh = fresh;
}

// `VA` = alignment (in words) every quantity of this stream is a multiple of: the window start, carry and fresh.
template <int VA>
__device__ __forceinline__ void absorb(uint32_t *my, ShaStream &s, const uint32_t one) {
    int cnt = s.carry + s.fresh;
    int ptr = s.base + CA - s.carry;
    while (cnt >= 16) {
        uint32_t w[16];
#pragma unroll
        for (int i = 0; i < 16; i += VA) {
            uint32_t x[VA];
            vec_load<VA>(my + ptr + i, x);
#pragma unroll
            for (int t = 0; t < VA; ++t) w[i + t] = bswap32(x[t]);
        }
        sha256_compress_rolled_fma(s.H, w, one);
        ptr += 16;
        cnt -= 16;
    }
    const int dst = s.base + CA - cnt;
    if (dst != ptr)
        for (int i = 0; i < cnt; ++i) my[dst + i] = my[ptr + i];  // dst <= ptr: ascending copy is safe
    s.carry = cnt;
    s.fresh = 0;
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

// Sequential CTR keystream along one private run: V words starting at word `wi` (absolute 32-bit word index in
// the image's private stream, a multiple of V); a new AES block is computed only when a 16-byte boundary is crossed.
struct Keystream {
    uint32_t ks[4];
    unsigned long long blk;
};
template <int V, typename Tab>
__device__ __forceinline__ void keystream_words(Keystream &K, const Tab sT, const uint32_t *rk, const uint32_t (&nonce)[4],
                                                unsigned long long wi, uint32_t (&out)[V]) {
    const unsigned long long blk = wi >> 2;
    if (V == 4 || blk != K.blk) {
        ctr_block(nonce, blk, K.ks);
        aes128_encrypt(sT, rk, K.ks);
        K.blk = blk;
    }
    if (V == 4) {
#pragma unroll
        for (int t = 0; t < V; ++t) out[t] = K.ks[t];
    } else if (V == 2) {
        const bool up = (wi & 2) != 0;
        out[0] = up ? K.ks[2] : K.ks[0];
        out[1 % V] = up ? K.ks[3] : K.ks[1];
    } else {
        const int sel = (int)(wi & 3);
        out[0] = sel == 0 ? K.ks[0] : sel == 1 ? K.ks[1] : sel == 2 ? K.ks[2] : K.ks[3];
    }
}

// ------------------------------------------------------------------------------------------------------------
// fragment: steps 1-5. V = 2 or 4 (when k + 1 is odd the host takes the tile kernel + leaf-hash kernel route instead).
// ------------------------------------------------------------------------------------------------------------
template <int C, int V>
__global__ void __launch_bounds__(DCT_THREADS, DCT_CTAS_PER_SM) fragment_dct_kernel(const __grid_constant__ DctParams p) {
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *sT = smem;
    load_aes_tables(sT);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *wslots = smem + AES_TABLE_WORDS + warp * 32 * p.slot_stride;
    uint32_t *my = wslots + lane * p.slot_stride;
    constexpr ZigzagTable ZZ = make_zigzag();

    const int k = p.k, P = k + 1, Q = 63 - k;
    uint32_t *mp = my + CA;      // private words of the current block, indexed by z
    uint32_t *mq = my + 2 * CA;  // public words of the current block, indexed by z (z >= P)
#pragma unroll 1
    for (unsigned grp = (unsigned)warp * gridDim.x + blockIdx.x; grp < p.n_groups; grp += (blockDim.x >> 5) * gridDim.x) {
    const LeafCoord L = decode_leaf<C>(p, (unsigned long long)grp * 32 + lane);
    const uint8_t *img = p.images + (size_t)L.n * p.image_stride;
    uint32_t *pub_dst = reinterpret_cast<uint32_t *>(p.pub + (size_t)L.n * p.pub_stride) + (size_t)L.b0 * Q;
    uint32_t *priv_dst = reinterpret_cast<uint32_t *>(p.priv + (size_t)L.n * p.priv_stride) + (size_t)L.b0 * P;
    uint32_t nonce[4];
    load_nonce(p, L.n, nonce);

    // cur = public stream, oth = private stream (swapped twice per phase). The public stream goes first so that in the
    // final phase the private stream's padding may spill into the (then finished) public region.
    ShaStream cur;
    ShaMeta oth;
    const int hoff = dct_stash_offset(k);
    sha256_init(cur.H);
    stash_init<V>(my, hoff);
    cur.base = CA + P; cur.carry = 0; cur.fresh = 0; cur.total_words = (unsigned)(L.nblk * Q);
    oth.base = 0; oth.carry = 0; oth.fresh = 0; oth.total_words = (unsigned)(L.nblk * P);
    Keystream K;
    K.blk = ~0ull;
    const unsigned long long priv_word0 = (unsigned long long)L.b0 * P;

#pragma unroll 1
    for (int s = 0; s <= G_BLOCKS; ++s) {
        if (s < G_BLOCKS) {
            const bool act = s < L.nblk;
            uint32_t *pq = pub_dst + (size_t)s * Q - P;  // public run of this block, indexed by z
            uint32_t *pv = priv_dst + (size_t)s * P;      // private run of this block, indexed by z
            if (act) {
                float v[64];
                load_block<C>(img, p.w, 8 * L.br, 8 * (L.g * G_BLOCKS + s), L.c, v);
                dct8x8(v);
#pragma unroll
                for (int g = 0; g < 64; g += V) {
                    uint32_t x[V];
#pragma unroll
                    for (int t = 0; t < V; ++t) x[t] = __float_as_uint(v[ZZ.pos[g + t]]);
                    if (g < P) {
                        vec_store<V>(mp + g, x);   // plaintext; encrypted in place below
                    } else {
                        vec_store<V>(mq + g, x);
                        vec_store<V>(pq + g, x);
                    }
                }
                const unsigned long long w0 = priv_word0 + (unsigned long long)s * P;
#pragma unroll 1
                for (int j = 0; j < P; j += V) {
                    uint32_t ks[V], x[V];
                    keystream_words<V>(K, sT, p.rk, nonce, w0 + j, ks);
                    vec_load<V>(mp + j, x);
#pragma unroll
                    for (int t = 0; t < V; ++t) x[t] ^= ks[t];
                    vec_store<V>(mp + j, x);
                    vec_store<V>(pv + j, x);
                }
            }
            cur.fresh = act ? Q : 0; oth.fresh = act ? P : 0;
        }
#pragma unroll 1
        for (int it = 0; it < 2; ++it) {
            if (s == G_BLOCKS && cur.total_words != 0u) write_padding(my, cur);
            absorb<V>(my, cur, p.one);
            swap_streams<V>(my, hoff, cur, oth);
        }
    }
    if (L.valid) {
        const size_t nl = p.leaves_per_image;
        if (Q > 0) store_digest(p.leaves + (((size_t)L.n * 2 + 1) * nl + L.li) * 32, cur.H);
        stash_read<V>(my, hoff, cur.H);  // after an even number of swaps the private stream is the stashed one
        store_digest(p.leaves + (((size_t)L.n * 2 + 0) * nl + L.li) * 32, cur.H);
    }
    }
}

}  // namespace feds
