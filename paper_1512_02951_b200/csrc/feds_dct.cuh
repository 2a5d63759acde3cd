// feds_dct.cuh — fused DCT-path kernels, sm_100a.
//
// One thread owns one Merkle leaf = up to G consecutive 8x8 blocks of one block row of one channel
// (DESIGN.md 2.1). For each block it: loads the 8x8 pixels, runs the separable FP32 DCT in 64 registers,
// splits the coefficients in zigzag order into its private / public words in a per-lane shared-memory slot,
// AES-128-CTR-encrypts the private words (shared-memory T-tables, sequential keystream along the leaf),
// lets the warp copy both runs out to HBM coalesced, and absorbs the stored bytes of both fragments into two
// running SHA-256 states (one inlined compression site). Pixels are read once; coefficients are written once;
// only 2 x 32 B of leaf digest per leaf go to the workspace.
#pragma once
#include "feds_device.cuh"

namespace feds {

__device__ const AesTables g_aes = make_aes_tables();
__device__ const ZigzagTable g_zigzag_unused = make_zigzag();  // (kept for cuobjdump inspection; kernels use the constexpr)

constexpr int DCT_THREADS = 128;
constexpr int AES_TABLE_WORDS = 1024;
constexpr int CARRY = 15;  // a SHA-256 block is 16 words: at most 15 words are carried between blocks

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
    int slot_stride;  // words per lane slot (odd)
};

// slot layout (word offsets in a lane's slot): private region [0, 15+P), public region [15+P, 30+64) (+ slack so
// that the 32 padding words of the final phase fit after the public carry area)
__host__ __device__ inline int dct_slot_words(int k, bool digest) {
    const int Q = 63 - k;
    int wds = digest ? (2 * CARRY + 64 + (Q < 32 ? 32 - Q : 0)) : 64 + 2 * CARRY;
    return wds | 1;
}

template <int C>
__device__ __forceinline__ void load_block(const uint8_t *__restrict__ img, int w, int y0, int x0, int c, float (&v)[64]) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const uint8_t *row = img + ((size_t)(y0 + r) * w + x0) * C;
        if (C == 1) {
            const uint2 q = __ldg(reinterpret_cast<const uint2 *>(row));
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                v[8 * r + i] = (float)((q.x >> (8 * i)) & 0xffu);
                v[8 * r + 4 + i] = (float)((q.y >> (8 * i)) & 0xffu);
            }
        } else if (C == 3) {
            const uint2 q0 = __ldg(reinterpret_cast<const uint2 *>(row));
            const uint2 q1 = __ldg(reinterpret_cast<const uint2 *>(row) + 1);
            const uint2 q2 = __ldg(reinterpret_cast<const uint2 *>(row) + 2);
            // shift the 24-byte row right by c bytes (c is fixed per thread), then the wanted bytes sit at 3*i
            const uint32_t wd[7] = {q0.x, q0.y, q1.x, q1.y, q2.x, q2.y, 0u};
            uint32_t ws[6];
#pragma unroll
            for (int j = 0; j < 6; ++j) ws[j] = __funnelshift_r(wd[j], wd[j + 1], 8 * c);
#pragma unroll
            for (int i = 0; i < 8; ++i) v[8 * r + i] = (float)((ws[(3 * i) >> 2] >> (8 * ((3 * i) & 3))) & 0xffu);
        } else {
            const uint4 a = __ldg(reinterpret_cast<const uint4 *>(row));
            const uint4 b = __ldg(reinterpret_cast<const uint4 *>(row) + 1);
            const uint32_t wd[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
            const int sh = 8 * c;
#pragma unroll
            for (int i = 0; i < 8; ++i) v[8 * r + i] = (float)((wd[i] >> sh) & 0xffu);
        }
    }
}

template <int C>
__device__ __forceinline__ void store_block(uint8_t *__restrict__ img, int w, int y0, int x0, int c, const float (&v)[64]) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        uint32_t px[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            int q = __float2int_rn(v[8 * r + i]);  // round to nearest even (A5)
            q = min(max(q, 0), 255);
            px[i] = (uint32_t)q;
        }
        uint8_t *row = img + ((size_t)(y0 + r) * w + x0) * C;
        if (C == 1) {
            uint2 q;
            q.x = px[0] | (px[1] << 8) | (px[2] << 16) | (px[3] << 24);
            q.y = px[4] | (px[5] << 8) | (px[6] << 16) | (px[7] << 24);
            *reinterpret_cast<uint2 *>(row) = q;
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i) row[i * C + c] = (uint8_t)px[i];
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

// One SHA-256 stream living in a lane's slot: `carry` words wait at [base+15-carry, base+15), `fresh` new words
// were just written at [base+15, base+15+fresh). Compress every full 16-word block, slide the rest down.
struct ShaStream {
    uint32_t H[8];
    int base;
    int carry;
    int fresh;
    unsigned total_words;  // message length of the whole leaf in 32-bit words (0: stream unused)
};

__device__ __forceinline__ void swap_streams(ShaStream &a, ShaStream &b) {
#pragma unroll
    for (int i = 0; i < 8; ++i) { const uint32_t t = a.H[i]; a.H[i] = b.H[i]; b.H[i] = t; }
    int t;
    t = a.base; a.base = b.base; b.base = t;
    t = a.carry; a.carry = b.carry; b.carry = t;
    t = a.fresh; a.fresh = b.fresh; b.fresh = t;
    const unsigned u = a.total_words; a.total_words = b.total_words; b.total_words = u;
}

// Append the FIPS 180-4 5.1.1 padding for a message of `total_words` 32-bit words after the carried words.
// Slot words are little-endian data words (byte-swapped when loaded into W), so the padding is written pre-swapped.
__device__ __forceinline__ void write_padding(uint32_t *my, ShaStream &s) {
    const int n = s.carry;
    int tot = n + 3;                      // 0x80 word + 64-bit length
    tot = (tot + 15) & ~15;               // 16 or 32
    const int fresh = tot - n;
    uint32_t *dst = my + s.base + CARRY;
    dst[0] = 0x00000080u;
    for (int i = 1; i < fresh - 2; ++i) dst[i] = 0u;
    const unsigned long long bits = (unsigned long long)s.total_words * 32ull;
    dst[fresh - 2] = bswap32((uint32_t)(bits >> 32));
    dst[fresh - 1] = bswap32((uint32_t)bits);
    s.fresh = fresh;
}

__device__ __forceinline__ void absorb(uint32_t *my, ShaStream &s) {
    int cnt = s.carry + s.fresh;
    int ptr = s.base + CARRY - s.carry;
    while (cnt >= 16) {
        uint32_t w[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) w[i] = bswap32(my[ptr + i]);
        sha256_compress(s.H, w);
        ptr += 16;
        cnt -= 16;
    }
    const int dst = s.base + CARRY - cnt;
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

// Sequential CTR keystream along one private run: word `wi` (absolute 32-bit word index in the image's private
// stream) -> keystream word; a new AES block is computed only when wi crosses a 16-byte boundary.
struct Keystream {
    uint32_t ks[4];
    unsigned long long blk;
};
__device__ __forceinline__ uint32_t keystream_word(Keystream &K, const uint32_t *sT, const uint32_t *rk, const uint32_t (&nonce)[4],
                                                   unsigned long long wi) {
    const unsigned long long blk = wi >> 2;
    if (blk != K.blk) {
        ctr_block(nonce, blk, K.ks);
        aes128_encrypt(sT, rk, K.ks);
        K.blk = blk;
    }
    const int sel = (int)(wi & 3);
    return sel == 0 ? K.ks[0] : sel == 1 ? K.ks[1] : sel == 2 ? K.ks[2] : K.ks[3];
}

// ------------------------------------------------------------------------------------------------------------
// fragment: steps 1-5
// ------------------------------------------------------------------------------------------------------------
template <int C, bool DIGEST>
__global__ void __launch_bounds__(DCT_THREADS, 4) fragment_dct_kernel(const __grid_constant__ DctParams p) {
    extern __shared__ uint32_t smem[];
    uint32_t *sT = smem;
    load_aes_tables(sT);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *wslots = smem + AES_TABLE_WORDS + warp * 32 * p.slot_stride;
    uint32_t *my = wslots + lane * p.slot_stride;
    constexpr ZigzagTable ZZ = make_zigzag();

    const int k = p.k, P = k + 1, Q = 63 - k;
    const LeafCoord L = decode_leaf<C>(p, (unsigned long long)blockIdx.x * DCT_THREADS + threadIdx.x);
    const uint8_t *img = p.images + (size_t)L.n * p.image_stride;
    uint32_t *pub_dst = reinterpret_cast<uint32_t *>(p.pub + (size_t)L.n * p.pub_stride) + (size_t)L.b0 * Q;
    uint32_t *priv_dst = reinterpret_cast<uint32_t *>(p.priv + (size_t)L.n * p.priv_stride) + (size_t)L.b0 * P;
    uint32_t nonce[4];
    load_nonce(p, L.n, nonce);

    // cur = public stream, oth = private stream (swapped twice per phase). The public stream goes first so that in the
    // final phase the private stream's padding may spill into the (then finished) public region.
    ShaStream cur, oth;
    sha256_init(cur.H); sha256_init(oth.H);
    cur.base = CARRY + P; cur.carry = 0; cur.fresh = 0; cur.total_words = (unsigned)(L.nblk * Q);
    oth.base = 0; oth.carry = 0; oth.fresh = 0; oth.total_words = (unsigned)(L.nblk * P);
    Keystream K;
    K.blk = ~0ull;
    const unsigned long long priv_word0 = (unsigned long long)L.b0 * P;

    for (int s = 0; s <= G_BLOCKS; ++s) {
        if (s < G_BLOCKS) {
            const bool act = s < L.nblk;
            if (act) {
                float v[64];
                load_block<C>(img, p.w, 8 * L.br, 8 * (L.g * G_BLOCKS + s), L.c, v);
                dct8x8(v);
                uint32_t *mp = my + CARRY;      // private words: [15, 15+P), indexed by z
                uint32_t *mq = my + 2 * CARRY;  // public words: region base (15+P) + 15 + (z-P) = 30 + z, indexed by z
#pragma unroll
                for (int z = 0; z < 64; ++z) {
                    const uint32_t bits = __float_as_uint(v[ZZ.pos[z]]);
                    if (z <= k) mp[z] = bits; else mq[z] = bits;
                }
                const unsigned long long w0 = priv_word0 + (unsigned long long)s * P;
                for (int j = 0; j < P; ++j) mp[j] ^= keystream_word(K, sT, p.rk, nonce, w0 + j);
            }
            __syncwarp();
            // the warp copies every lane's two runs out, coalesced
            const unsigned long long pd = act ? reinterpret_cast<unsigned long long>(pub_dst + (size_t)s * Q) : 0ull;
            const unsigned long long vd = act ? reinterpret_cast<unsigned long long>(priv_dst + (size_t)s * P) : 0ull;
            for (int l = 0; l < 32; ++l) {
                const unsigned long long pdl = __shfl_sync(0xffffffffu, pd, l);
                const unsigned long long vdl = __shfl_sync(0xffffffffu, vd, l);
                if (pdl == 0ull) continue;
                const uint32_t *src = wslots + l * p.slot_stride;
                uint32_t *dq = reinterpret_cast<uint32_t *>(pdl);
                uint32_t *dp = reinterpret_cast<uint32_t *>(vdl);
                if (lane < Q) dq[lane] = src[2 * CARRY + P + lane];
                if (lane + 32 < Q) dq[lane + 32] = src[2 * CARRY + P + lane + 32];
                if (lane < P) dp[lane] = src[CARRY + lane];
                if (lane + 32 < P) dp[lane + 32] = src[CARRY + lane + 32];
            }
            __syncwarp();
            if (DIGEST) { cur.fresh = act ? Q : 0; oth.fresh = act ? P : 0; }
        }
        if (DIGEST) {
#pragma unroll 1
            for (int it = 0; it < 2; ++it) {
                if (s == G_BLOCKS && cur.total_words != 0u) write_padding(my, cur);
                absorb(my, cur);
                swap_streams(cur, oth);
            }
        }
    }
    if (DIGEST && L.valid) {
        const size_t nl = p.leaves_per_image;
        store_digest(p.leaves + (((size_t)L.n * 2 + 0) * nl + L.li) * 32, oth.H);
        if (Q > 0) store_digest(p.leaves + (((size_t)L.n * 2 + 1) * nl + L.li) * 32, cur.H);
    }
}

// ------------------------------------------------------------------------------------------------------------
// defragment: steps 6-8 (+ recomputation of the leaf digests of the fragments as received when VERIFY)
// ------------------------------------------------------------------------------------------------------------
template <int C, bool VERIFY>
__global__ void __launch_bounds__(DCT_THREADS, 4) defragment_dct_kernel(const __grid_constant__ DctParams p) {
    extern __shared__ uint32_t smem[];
    uint32_t *sT = smem;
    load_aes_tables(sT);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *wslots = smem + AES_TABLE_WORDS + warp * 32 * p.slot_stride;
    uint32_t *my = wslots + lane * p.slot_stride;
    constexpr ZigzagTable ZZ = make_zigzag();

    const int k = p.k, P = k + 1, Q = 63 - k;
    const LeafCoord L = decode_leaf<C>(p, (unsigned long long)blockIdx.x * DCT_THREADS + threadIdx.x);
    uint8_t *img = p.images_out + (size_t)L.n * p.image_stride;
    const uint32_t *pub_src = reinterpret_cast<const uint32_t *>(p.pub + (size_t)L.n * p.pub_stride) + (size_t)L.b0 * Q;
    const uint32_t *priv_src = reinterpret_cast<const uint32_t *>(p.priv + (size_t)L.n * p.priv_stride) + (size_t)L.b0 * P;
    uint32_t nonce[4];
    load_nonce(p, L.n, nonce);

    // cur = public stream, oth = private stream (swapped twice per phase). The public stream goes first so that in the
    // final phase the private stream's padding may spill into the (then finished) public region.
    ShaStream cur, oth;
    sha256_init(cur.H); sha256_init(oth.H);
    cur.base = CARRY + P; cur.carry = 0; cur.fresh = 0; cur.total_words = (unsigned)(L.nblk * Q);
    oth.base = 0; oth.carry = 0; oth.fresh = 0; oth.total_words = (unsigned)(L.nblk * P);
    Keystream K;
    K.blk = ~0ull;
    const unsigned long long priv_word0 = (unsigned long long)L.b0 * P;

    for (int s = 0; s <= G_BLOCKS; ++s) {
        const bool act = s < L.nblk;
        if (s < G_BLOCKS) {
            // the warp copies every lane's two runs in, coalesced
            const unsigned long long pd = act ? reinterpret_cast<unsigned long long>(pub_src + (size_t)s * Q) : 0ull;
            const unsigned long long vd = act ? reinterpret_cast<unsigned long long>(priv_src + (size_t)s * P) : 0ull;
            for (int l = 0; l < 32; ++l) {
                const unsigned long long pdl = __shfl_sync(0xffffffffu, pd, l);
                const unsigned long long vdl = __shfl_sync(0xffffffffu, vd, l);
                if (vdl == 0ull) continue;
                uint32_t *dst = wslots + l * p.slot_stride;
                const uint32_t *sq = reinterpret_cast<const uint32_t *>(pdl);
                const uint32_t *sp = reinterpret_cast<const uint32_t *>(vdl);
                if (lane < Q) dst[2 * CARRY + P + lane] = __ldg(sq + lane);
                if (lane + 32 < Q) dst[2 * CARRY + P + lane + 32] = __ldg(sq + lane + 32);
                if (lane < P) dst[CARRY + lane] = __ldg(sp + lane);
                if (lane + 32 < P) dst[CARRY + lane + 32] = __ldg(sp + lane + 32);
            }
            __syncwarp();
            if (VERIFY) { cur.fresh = act ? Q : 0; oth.fresh = act ? P : 0; }
        }
        if (VERIFY) {
#pragma unroll 1
            for (int it = 0; it < 2; ++it) {
                if (s == G_BLOCKS && cur.total_words != 0u) write_padding(my, cur);
                absorb(my, cur);  // hashes the bytes as received (ciphertext / public coefficients); keeps [base+15, ..) intact
                swap_streams(cur, oth);
            }
        }
        if (s < G_BLOCKS) {
            if (act) {
                uint32_t *mp = my + CARRY;
                const uint32_t *mq = my + 2 * CARRY;
                const unsigned long long w0 = priv_word0 + (unsigned long long)s * P;
                for (int j = 0; j < P; ++j) mp[j] ^= keystream_word(K, sT, p.rk, nonce, w0 + j);
                float v[64];
#pragma unroll
                for (int z = 0; z < 64; ++z) v[ZZ.pos[z]] = __uint_as_float(z <= k ? mp[z] : mq[z]);
                idct8x8(v);
                store_block<C>(img, p.w, 8 * L.br, 8 * (L.g * G_BLOCKS + s), L.c, v);
            }
            __syncwarp();  // the next phase's copy-in overwrites the slots
        }
    }
    if (VERIFY && L.valid) {
        const size_t nl = p.leaves_per_image;
        store_digest(p.leaves + (((size_t)L.n * 2 + 0) * nl + L.li) * 32, oth.H);
        if (Q > 0) store_digest(p.leaves + (((size_t)L.n * 2 + 1) * nl + L.li) * 32, cur.H);
    }
}

}  // namespace feds
