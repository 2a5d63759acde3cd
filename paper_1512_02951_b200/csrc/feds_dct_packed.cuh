// feds_dct_packed.cuh — the report's packed integer coefficient storage (PAPER.md 6.4.3, Table 5; SURVEY.md 8(f)
// NEXT-4), sm_100a. Byte format: DESIGN.md 2.4 (readings K1-K4). Part 1 of a block is stored as integers -- DC in 11 bits, each AC in
// an 11- or 8-bit sign-magnitude field -- bit-tight per leaf group of 8 blocks (12.9 % / 9.96 % of the image at k = 5), under
// AES-128-CTR; the public part is the image-sized remainder x - L ("IDCT of the rest"), taken against the QUANTISED Part 1 in
// the fixed-point arithmetic of the strong level, so that every pixel comes back exactly with either storage.
//
// These are the general kernels (any shape, any k); feds_dct_packed_tile.cuh has the tile-group kernels the host prefers where the
// shape allows (w % 64 == 0, k <= 15). One thread per (leaf group, channel): it walks the group's blocks, appends their fields to a bit buffer and writes the group's
// bytes. The channels of one pixel strip sit in adjacent lanes (store_block_packed). Encryption is the stream kernel's, in place.
#pragma once
#include "feds_dct_strong.cuh"

namespace feds {

constexpr int PACKED_THREADS = 128;

// four bytes: (in_i -/+ L_i) mod 256, L_i = acc_i >> 12 (DESIGN.md 2.4 K3: the integers are not scaled by 8 here)
template <bool SUBTRACT>
__device__ __forceinline__ uint32_t packed_apply4(uint32_t in, int32_t a0, int32_t a1, int32_t a2, int32_t a3) {
    const uint32_t L = ((uint32_t)(a0 >> 12) & 255u) | (((uint32_t)(a1 >> 12) & 255u) << 8) | (((uint32_t)(a2 >> 12) & 255u) << 16) |
                       (((uint32_t)(a3 >> 12) & 255u) << 24);
    return SUBTRACT ? __vsub4(in, L) : __vadd4(in, L);
}
// acc[p] = 2^11 + sum_z q_z B[z][p], q_z = the integers in the thread's shared-memory column
__device__ __forceinline__ void packed_low_pass(const uint32_t *col, int stride, int P, int32_t (&acc)[64]) {
#pragma unroll
    for (int p = 0; p < 64; ++p) acc[p] = 2048;
#pragma unroll 1
    for (int z = 0; z < P; ++z) {
        const int32_t q = (int32_t)col[z * stride];
        const int32_t *Bz = c_strong_basis_tab.B + 64 * z;
#pragma unroll
        for (int p = 0; p < 64; ++p) acc[p] = (int32_t)((uint32_t)acc[p] + (uint32_t)q * (uint32_t)Bz[p]);
    }
}
// K1: float32 coefficient -> stored integer (round to nearest even; NaN -> 0; DC 0..2047, AC +-M)
__device__ __forceinline__ int32_t packed_quantise(float c, bool dc, int M) {
    const int32_t q = __float2int_rn(c);   // saturates, NaN -> 0
    return dc ? min(max(q, 0), 2047) : min(max(q, -M), M);
}

struct PackedCoord {
    bool valid;
    int n, ch, br, g, nblk;
    size_t row;       // ch * nbr + br
    size_t byte_off;  // of the group inside the image's private fragment
    unsigned nbytes;  // of the group
};
template <int C>
__device__ __forceinline__ PackedCoord packed_decode(const DctParams &p, unsigned long long gid) {
    PackedCoord S;
    const unsigned long long per_image = (unsigned long long)C * p.nbr * p.nlr;
    S.valid = gid < per_image * p.n_images;
    const unsigned long long g2 = S.valid ? gid : 0;
    S.n = (int)(g2 / per_image);
    unsigned rem = (unsigned)(g2 % per_image);
    S.ch = (int)(rem % C);
    rem /= C;
    S.g = (int)(rem % (unsigned)p.nlr);
    S.br = (int)(rem / (unsigned)p.nlr);
    const int left = p.nbc - S.g * G_BLOCKS;
    S.nblk = S.valid ? (left < G_BLOCKS ? left : G_BLOCKS) : 0;
    S.row = (size_t)S.ch * p.nbr + S.br;
    S.byte_off = S.row * p.packed_row_bytes + (size_t)S.g * p.packed_group_bytes;
    S.nbytes = (unsigned)(((unsigned)S.nblk * p.packed_group_bytes + 7u) / 8u);
    return S;
}

// shared memory: one column of 64 words per thread (word z of thread t at z * THREADS + t)
template <int C>
__global__ void __launch_bounds__(PACKED_THREADS) fragment_dct_packed_kernel(const __grid_constant__ DctParams p) {
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *col = smem + threadIdx.x;
    constexpr ZigzagTable ZZ = make_zigzag();
    const PackedCoord S = packed_decode<C>(p, (unsigned long long)blockIdx.x * PACKED_THREADS + threadIdx.x);
    if (!S.valid) return;
    const int P = p.k + 1, bits = p.ac_bits, M = (1 << (bits - 1)) - 1;
    const uint8_t *img = p.images + (size_t)S.n * p.image_stride;
    uint8_t *out = p.priv + (size_t)S.n * p.priv_stride + S.byte_off;
    unsigned long long buf = 0ull;   // little-endian bit stream of the group (K2)
    int nbuf = 0;
#pragma unroll 1
    for (int j = 0; j < S.nblk; ++j) {
        const int bc = S.g * G_BLOCKS + j;
        {
            float v[64];
            load_block<C>(img, p.w, 8 * S.br, 8 * bc, S.ch, v);
            dct8x8(v);
#pragma unroll
            for (int z = 0; z < 64; ++z) col[z * PACKED_THREADS] = __float_as_uint(v[ZZ.pos[z]]);
        }
#pragma unroll 1
        for (int z = 0; z < P; ++z) {
            const int32_t q = packed_quantise(__uint_as_float(col[z * PACKED_THREADS]), z == 0, M);
            col[z * PACKED_THREADS] = (uint32_t)q;
            const uint32_t field = z == 0 ? (uint32_t)q : ((uint32_t)abs(q) | (q < 0 ? 1u << (bits - 1) : 0u));
            buf |= (unsigned long long)field << nbuf;
            nbuf += z == 0 ? 11 : bits;
            while (nbuf >= 8) { *out++ = (uint8_t)buf; buf >>= 8; nbuf -= 8; }
        }
        int32_t acc[64];
        packed_low_pass(col, PACKED_THREADS, P, acc);
        const size_t b = S.row * p.nbc + bc;
        uint4 *dst = reinterpret_cast<uint4 *>(p.pub + (size_t)S.n * p.pub_stride + 64 * b);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const uint2 x0 = strong_load_row<C>(img + ((size_t)(8 * S.br + 2 * i) * p.w + 8 * bc) * C, S.ch);
            const uint2 x1 = strong_load_row<C>(img + ((size_t)(8 * S.br + 2 * i + 1) * p.w + 8 * bc) * C, S.ch);
            dst[i] = make_uint4(packed_apply4<true>(x0.x, acc[16 * i], acc[16 * i + 1], acc[16 * i + 2], acc[16 * i + 3]),
                                packed_apply4<true>(x0.y, acc[16 * i + 4], acc[16 * i + 5], acc[16 * i + 6], acc[16 * i + 7]),
                                packed_apply4<true>(x1.x, acc[16 * i + 8], acc[16 * i + 9], acc[16 * i + 10], acc[16 * i + 11]),
                                packed_apply4<true>(x1.y, acc[16 * i + 12], acc[16 * i + 13], acc[16 * i + 14], acc[16 * i + 15]));
        }
    }
    if (nbuf > 0) *out++ = (uint8_t)buf;   // zero bits up to the byte boundary
}

// `plain` = the decrypted private fragments of the batch (workspace), image n at plain + n * plain_stride
template <int C>
__global__ void __launch_bounds__(PACKED_THREADS) defragment_dct_packed_kernel(const __grid_constant__ DctParams p, const uint8_t *plain,
                                                                               size_t plain_stride) {
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *col = smem + threadIdx.x;
    const PackedCoord S = packed_decode<C>(p, (unsigned long long)blockIdx.x * PACKED_THREADS + threadIdx.x);
    const int P = p.k + 1, bits = p.ac_bits;
    const uint8_t *in = plain + (size_t)S.n * plain_stride + S.byte_off;
    const uint8_t *const in_end = in + S.nbytes;
    unsigned long long buf = 0ull;
    int nbuf = 0;
#pragma unroll 1
    for (int j = 0; j < G_BLOCKS; ++j) {   // every lane walks all eight steps: store_block_packed shuffles across the warp
        const bool act = j < S.nblk;
        const int bc = S.g * G_BLOCKS + (act ? j : 0);
        uint32_t rows[16];
        if (act) {
#pragma unroll 1
            for (int z = 0; z < P; ++z) {
                const int nb = z == 0 ? 11 : bits;
                while (nbuf < nb) { buf |= (unsigned long long)(in < in_end ? *in : 0) << nbuf; ++in; nbuf += 8; }
                const uint32_t field = (uint32_t)buf & ((1u << nb) - 1u);
                buf >>= nb;
                nbuf -= nb;
                int32_t q = (int32_t)field;
                if (z > 0) {
                    const int32_t mag = (int32_t)(field & ((1u << (bits - 1)) - 1u));
                    q = (field >> (bits - 1)) ? -mag : mag;
                }
                col[z * PACKED_THREADS] = (uint32_t)q;
            }
            int32_t acc[64];
            packed_low_pass(col, PACKED_THREADS, P, acc);
            const size_t b = S.row * p.nbc + bc;
            const uint4 *src = reinterpret_cast<const uint4 *>(p.pub + (size_t)S.n * p.pub_stride + 64 * b);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const uint4 x = __ldg(src + i);
                rows[4 * i] = packed_apply4<false>(x.x, acc[16 * i], acc[16 * i + 1], acc[16 * i + 2], acc[16 * i + 3]);
                rows[4 * i + 1] = packed_apply4<false>(x.y, acc[16 * i + 4], acc[16 * i + 5], acc[16 * i + 6], acc[16 * i + 7]);
                rows[4 * i + 2] = packed_apply4<false>(x.z, acc[16 * i + 8], acc[16 * i + 9], acc[16 * i + 10], acc[16 * i + 11]);
                rows[4 * i + 3] = packed_apply4<false>(x.w, acc[16 * i + 12], acc[16 * i + 13], acc[16 * i + 14], acc[16 * i + 15]);
            }
        }
        store_block_packed<C>(p.images_out + (size_t)S.n * p.image_stride, p.w, 8 * S.br, 8 * bc, S.ch, act, rows);
    }
}

// SHA-256 of the packed private leaves (the bytes of one leaf group, any length and alignment): one thread per leaf
__global__ void __launch_bounds__(PACKED_THREADS) packed_private_leaves_kernel(const __grid_constant__ DctParams p, int channels) {
    const unsigned long long gid = (unsigned long long)blockIdx.x * PACKED_THREADS + threadIdx.x;
    const unsigned long long per_image = (unsigned long long)channels * p.nbr * p.nlr;
    if (gid >= per_image * p.n_images) return;
    const int n = (int)(gid / per_image);
    const unsigned li = (unsigned)(gid % per_image);   // leaf index in fragment order: row * nlr + g
    const unsigned row = li / (unsigned)p.nlr, g = li % (unsigned)p.nlr;
    const int left = p.nbc - (int)g * G_BLOCKS, nblk = left < G_BLOCKS ? left : G_BLOCKS;
    const unsigned nbytes = ((unsigned)nblk * p.packed_group_bytes + 7u) / 8u;
    const uint8_t *msg = p.priv + (size_t)n * p.priv_stride + (size_t)row * p.packed_row_bytes + (size_t)g * p.packed_group_bytes;
    const unsigned nblocks = (nbytes + 9u + 63u) / 64u;
    uint32_t H[8], w[16];
    sha256_init(H);
    // message words from aligned 32-bit loads joined by a funnel shift; never past the last whole word of the image's fragment
    const uintptr_t addr = reinterpret_cast<uintptr_t>(msg);
    const uint32_t *aligned = reinterpret_cast<const uint32_t *>(addr & ~(uintptr_t)3);
    const unsigned shift = 8u * (unsigned)(addr & 3u);
    const uintptr_t safe_end = reinterpret_cast<uintptr_t>(p.priv + (size_t)n * p.priv_stride) + ((size_t)channels * p.nbr * p.packed_row_bytes & ~(size_t)3);
#pragma unroll 1
    for (unsigned b = 0; b < nblocks; ++b) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const unsigned pos0 = 64u * b + 4u * j;
            uint32_t word = 0u;
            if (pos0 + 4u <= nbytes && addr + pos0 + 4u <= safe_end) {
                const uint32_t lo = __ldg(aligned + (pos0 >> 2)), hi = shift ? __ldg(aligned + (pos0 >> 2) + 1) : 0u;
                word = bswap32(__funnelshift_r(lo, hi, shift));
            } else {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const unsigned pos = pos0 + q;
                    word = (word << 8) | (pos < nbytes ? (uint32_t)msg[pos] : (pos == nbytes ? 0x80u : 0u));
                }
            }
            w[j] = word;
        }
        if (b == nblocks - 1) { w[14] = 0u; w[15] = nbytes * 8u; }
        sha256_compress_rolled_fma(H, w, p.one);
    }
    store_digest(p.leaves + (((size_t)n * 2 + 0) * p.leaves_per_image + li) * 32, H);
}

}  // namespace feds
