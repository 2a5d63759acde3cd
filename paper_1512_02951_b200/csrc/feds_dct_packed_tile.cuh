// feds_dct_packed_tile.cuh — the packed-storage kernels (feds_dct_packed.cuh) on the bulk-copy tile groups of
// feds_dct_tma.cuh, sm_100a. Same bytes; what changes is how the work is laid out:
//   * tiles of 32 (gray: 64) blocks in linear block order, pixel rows brought in by cp.async.bulk into a double buffer; one thread
//     per (block, channel), the channel warp-uniform -- no strided per-thread pixel loads, no 64-word shared-memory column per thread;
//   * only the coefficients z <= k that are stored get computed: the transform is inlined and every output the zigzag prefix never
//     reads is dead code (k <= 15 here; larger k take the thread-per-group kernels);
//   * the low-pass prediction L = floor((sum q_z B_z + 2^11) / 2^12) runs over the table in constant memory with immediate
//     offsets (one IMAD per pixel and coefficient, no loads), four pixel rows at a time;
//   * a warp owns the four leaf groups of its 32 blocks: exactly b 32-bit words of shared memory, which its lanes fill with
//     atomicOr at their bit offsets and then copy out -- no barrier besides the one that hands the pixel buffer back.
// Shapes: w % 64 == 0 (leaf groups never straddle a tile, every group is full: b bytes) and at least one tile per block row.
#pragma once
#include "feds_dct_packed.cuh"
#include "feds_dct_tma.cuh"

namespace feds {

constexpr int PT_MAX_P = 16;          // stored coefficients per block these kernels handle (k <= 15)
constexpr int PT_MAX_B = 11 + 15 * 11;  // bits per block = bytes per group = words per warp region
template <int C> struct PackedTileShape {
    using S = TmaShape<C>;
    static constexpr int GROUPS = C == 1 ? 12 : (C == 3 ? 8 : 6);   // tile groups per CTA: 768 threads of <= 80 registers (measured at C = 3: 5 groups 1.12 ms, 8 groups 0.92 ms for the inverse)
    static constexpr int CTA = GROUPS * S::THREADS;
    static constexpr int WARPS = CTA / 32;
};
template <int C> __host__ __device__ inline size_t packed_tile_smem_bytes() {
    return TMA_BAR_BYTES + (size_t)PackedTileShape<C>::GROUPS * 2 * TmaShape<C>::PIX_BYTES + (size_t)PackedTileShape<C>::WARPS * PT_MAX_B * 4;
}
template <int C> __host__ __device__ inline bool packed_tile_ok(int w, int k) { return (w % 64) == 0 && (w / 8) >= TmaShape<C>::TB && k < PT_MAX_P; }

// bytes 4i .. 4i+3 of channel CH of one pixel row of a block (row = its 8 * C bytes as words), i = 0, 1
template <int C, int CH>
__device__ __forceinline__ void row_bytes_of_channel(const uint32_t (&wd)[2 * C], uint32_t &lo, uint32_t &hi) {
    if (C == 1) { lo = wd[0]; hi = wd[1]; return; }
    uint32_t out[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        // pixel p = 4h + q sits at byte C * p + CH of the row
        const int o0 = C * (4 * h + 0) + CH, o1 = C * (4 * h + 1) + CH, o2 = C * (4 * h + 2) + CH, o3 = C * (4 * h + 3) + CH;
        const uint32_t a = __byte_perm(wd[o0 >> 2], wd[o1 >> 2], (uint32_t)((o0 & 3) | (((o1 & 3) + 4) << 4)));
        const uint32_t b = __byte_perm(wd[o2 >> 2], wd[o3 >> 2], (uint32_t)((o2 & 3) | (((o3 & 3) + 4) << 4)));
        out[h] = __byte_perm(a, b, 0x5410);
    }
    lo = out[0]; hi = out[1];
}
template <int C, int CH>
__device__ __forceinline__ void load_row_bytes(uint32_t row, uint32_t &lo, uint32_t &hi) {
    uint32_t wd[2 * C];
    if (C == 1) {
        const uint2 q = lds64(row);
        wd[0] = q.x; wd[1 % (2 * C)] = q.y;
    } else if (C == 3) {
        const uint2 q0 = lds64(row), q1 = lds64(row + 8), q2 = lds64(row + 16);
        wd[0] = q0.x; wd[1] = q0.y; wd[2 % (2 * C)] = q1.x; wd[3 % (2 * C)] = q1.y; wd[4 % (2 * C)] = q2.x; wd[5 % (2 * C)] = q2.y;
    } else {
        const uint4 a = lds128(row), b = lds128(row + 16);
        wd[0] = a.x; wd[1] = a.y; wd[2 % (2 * C)] = a.z; wd[3 % (2 * C)] = a.w; wd[4 % (2 * C)] = b.x; wd[5 % (2 * C)] = b.y; wd[6 % (2 * C)] = b.z; wd[7 % (2 * C)] = b.w;
    }
    row_bytes_of_channel<C, CH>(wd, lo, hi);
}

// Remainder bytes without unpacking: x - floor((S + 2^11) / 2^12) = floor((x * 2^12 + 2^11 - 1 - S) / 2^12), S = sum q_z B_z, and
// with everything scaled by 16 the quotient's low byte is byte 2 of the accumulator: acc = (x << 16 | 0x7ff0) - sum (16 q_z) B_z.
// One PRMT drops pixel byte x into byte 2 over the constant, one IMAD per coefficient, one PRMT per two results to collect them.
// nq[z] = -16 q_z. Pixel rows 4 * HALF .. 4 * HALF + 3 of the block (words x[8 * HALF ..]) -> 32 remainder bytes r[0..7].
template <int HALF, int PMAX>
__device__ __forceinline__ void packed_remainder_words(const uint32_t (&x)[16], const int32_t (&nq)[PMAX], int P, uint32_t (&r)[8]) {
    int32_t acc[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) acc[i] = (int32_t)__byte_perm(x[8 * HALF + (i >> 2)], 0x00007ff0u, 0x7054u + ((uint32_t)(i & 3) << 8));
#pragma unroll
    for (int z = 0; z < PMAX; ++z) {
        if (z < P) {   // warp-uniform
#pragma unroll
            for (int i = 0; i < 32; ++i)
                acc[i] = (int32_t)((uint32_t)acc[i] + (uint32_t)nq[z] * (uint32_t)c_strong_basis_tab.B[64 * z + 32 * HALF + i]);
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i)
        r[i] = __byte_perm(__byte_perm((uint32_t)acc[4 * i], (uint32_t)acc[4 * i + 1], 0x0062u), __byte_perm((uint32_t)acc[4 * i + 2], (uint32_t)acc[4 * i + 3], 0x0062u), 0x5410u);
}

// The inverse: x = pub + floor((S + 2^11) / 2^12) mod 256 = byte 2 of (pub << 16 | 0x8000) + sum (16 q_z) B_z. q16[z] = 16 q_z.
template <int HALF, int PMAX>
__device__ __forceinline__ void packed_restore_words(const uint32_t (&x)[16], const int32_t (&q16)[PMAX], int P, uint32_t (&r)[8]) {
    int32_t acc[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) acc[i] = (int32_t)__byte_perm(x[8 * HALF + (i >> 2)], 0x00008000u, 0x7054u + ((uint32_t)(i & 3) << 8));
#pragma unroll
    for (int z = 0; z < PMAX; ++z) {
        if (z < P) {   // warp-uniform
#pragma unroll
            for (int i = 0; i < 32; ++i)
                acc[i] = (int32_t)((uint32_t)acc[i] + (uint32_t)q16[z] * (uint32_t)c_strong_basis_tab.B[64 * z + 32 * HALF + i]);
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i)
        r[i] = __byte_perm(__byte_perm((uint32_t)acc[4 * i], (uint32_t)acc[4 * i + 1], 0x0062u), __byte_perm((uint32_t)acc[4 * i + 2], (uint32_t)acc[4 * i + 3], 0x0062u), 0x5410u);
}

// ------------------------------------------------------------------------------------------------------------ fragment
// the 64 bytes of block (j, ch) of the pixel tile, row-major, 16 words. Only this gather depends on the channel (immediate byte
// selectors); everything after it is one copy of code for all warps.
template <int C>
__device__ __forceinline__ void packed_block_bytes(const uint8_t *s_pix, const TmaTile &T, int j, int ch, uint32_t (&x)[16]) {
    uint32_t off, pitch;
    tma_pixel_slot<C>(T, j, off, pitch);
    const uint32_t blk = smem_u32(s_pix) + off;
#define FEDS_ROWS(CH)                                                                        \
    _Pragma("unroll") for (int r = 0; r < 8; ++r) load_row_bytes<C, CH>(blk + r * pitch, x[2 * r], x[2 * r + 1]);
    if (C == 1) { FEDS_ROWS(0) }
    else if (ch == 0) { FEDS_ROWS(0) }   // warp-uniform
    else if (ch == 1) { FEDS_ROWS(1) }
    else if (ch == 2) { FEDS_ROWS(2) }
    else { FEDS_ROWS((C == 4 ? 3 : 0)) }
#undef FEDS_ROWS
}
// remainder of pixel rows 4 * HALF .. + 3 of one block: (x - L) mod 256, 32 bytes -> two 16-byte stores
template <int HALF, int PMAX>
__device__ __forceinline__ void packed_remainder_half(const uint32_t (&x)[16], const int32_t (&nq)[PMAX], int P, uint4 *dst) {
    uint32_t r[8];
    packed_remainder_words<HALF, PMAX>(x, nq, P, r);
    dst[2 * HALF] = make_uint4(r[0], r[1], r[2], r[3]);
    dst[2 * HALF + 1] = make_uint4(r[4], r[5], r[6], r[7]);
}
template <int PMAX>
__device__ __forceinline__ void packed_fragment_block(const DctParams &p, const uint32_t (&x)[16], uint32_t *region, int lane, uint4 *dst) {
    constexpr ZigzagTable ZZ = make_zigzag();
    const int P = p.k + 1, bits = p.ac_bits, M = (1 << (bits - 1)) - 1;
    int32_t q[PMAX];
    {
        float v[64];
#pragma unroll
        for (int i = 0; i < 64; ++i) v[i] = byte_to_biased_float(x[i >> 2], i & 3);
        dct8x8_biased(v);
#pragma unroll
        for (int z = 0; z < PMAX; ++z) q[z] = z < P ? packed_quantise(v[ZZ.pos[z]], z == 0, M) : 0;
    }
    // the block's b bits at bit (lane & 7) * b of group lane >> 3, i.e. at bit lane * b of the warp's region (K2)
    {
        const unsigned bitpos = (unsigned)lane * p.packed_group_bytes;
        uint32_t *word = region + (bitpos >> 5);
        unsigned long long buf = 0ull;
        int nbuf = (int)(bitpos & 31u);
#pragma unroll
        for (int z = 0; z < PMAX; ++z) {
            if (z < P) {
                const uint32_t field = z == 0 ? (uint32_t)q[0] : ((uint32_t)abs(q[z]) | (q[z] < 0 ? 1u << (bits - 1) : 0u));
                buf |= (unsigned long long)field << nbuf;
                nbuf += z == 0 ? 11 : bits;
                if (nbuf >= 32) { atomicOr(word++, (uint32_t)buf); buf >>= 32; nbuf -= 32; }
            }
        }
        if (nbuf > 0) atomicOr(word, (uint32_t)buf);
    }
#pragma unroll
    for (int z = 0; z < PMAX; ++z) q[z] *= -16;
    packed_remainder_half<0, PMAX>(x, q, P, dst);
    packed_remainder_half<1, PMAX>(x, q, P, dst);
}

// PMAX (4, 6, 8 or 16) >= k + 1: the unrolled per-coefficient code the kernel carries
template <int C, int PMAX>
__global__ void __launch_bounds__(PackedTileShape<C>::CTA, 1) fragment_dct_packed_tile_kernel(const __grid_constant__ DctParams p) {
    using S = TmaShape<C>;
    using PS = PackedTileShape<C>;
    extern __shared__ __align__(128) uint32_t smem[];
    const int gid = threadIdx.x / S::THREADS, tid = threadIdx.x % S::THREADS, lane = threadIdx.x & 31;
    const int ch = (tid >> 5) % C, j = ((tid >> 5) / C) * 32 + lane;
    uint8_t *base = reinterpret_cast<uint8_t *>(smem) + TMA_BAR_BYTES;
    uint8_t *pix[2] = {base + (size_t)gid * 2 * S::PIX_BYTES, base + (size_t)gid * 2 * S::PIX_BYTES + S::PIX_BYTES};
    uint32_t *region = reinterpret_cast<uint32_t *>(base + (size_t)PS::GROUPS * 2 * S::PIX_BYTES) + (threadIdx.x >> 5) * PT_MAX_B;
    const uint32_t bar[2] = {smem_u32(smem) + 16u * gid, smem_u32(smem) + 16u * gid + 8u};
    if (tid == 0) { mbar_init(bar[0], 1); mbar_init(bar[1], 1); mbar_init_fence(); }
    const int b = (int)p.packed_group_bytes;   // bits per block = bytes per group = words per warp region
    for (int i = lane; i < b; i += 32) region[i] = 0u;
    __syncthreads();
    const unsigned tiles_per_plane = ((unsigned)p.nbr * p.nbc + S::TB - 1) / S::TB;
    const unsigned total = (unsigned)p.n_images * tiles_per_plane, step = gridDim.x * PS::GROUPS;
    const size_t plane = (size_t)p.nbr * p.nbc;
    unsigned t = blockIdx.x * PS::GROUPS + gid;
    if (t < total && tid == S::LOADER) tma_move_pixels<C, false>(p, tma_decode_tile<C>(p, t, tiles_per_plane), smem_u32(pix[0]), bar[0]);
#pragma unroll 1
    for (unsigned it = 0; t < total; t += step, ++it) {
        const int s = it & 1;
        const TmaTile T = tma_decode_tile<C>(p, t, tiles_per_plane);
        // the other pixel tile was last read one iteration ago, before that iteration's barrier: refill it now
        if (tid == S::LOADER && t + step < total)
            tma_move_pixels<C, false>(p, tma_decode_tile<C>(p, t + step, tiles_per_plane), smem_u32(s ? pix[0] : pix[1]), s ? bar[0] : bar[1]);
        mbar_wait(s ? bar[1] : bar[0], (it >> 1) & 1);
        const uint8_t *s_pix = s ? pix[1] : pix[0];
        const size_t blk0 = (size_t)ch * plane + T.B0;   // fragment-order index of the tile's first block of this channel
        if (j < T.nb) {
            uint4 *dst = reinterpret_cast<uint4 *>(p.pub + (size_t)T.n * p.pub_stride + 64 * (blk0 + j));
            uint32_t x[16];
            packed_block_bytes<C>(s_pix, T, j, ch, x);
            packed_fragment_block<PMAX>(p, x, region, lane, dst);
        }
        __syncwarp();
        // the warp's groups leave (nb is a multiple of 8: whole groups) and the region is cleared for the next tile
        const int j0 = j - lane, ngroups = min(4, (T.nb - j0) / 8);
        if (ngroups > 0) {
            uint8_t *out = p.priv + (size_t)T.n * p.priv_stride + ((blk0 + j0) >> 3) * (size_t)b;
            const int nbytes = ngroups * b;
            if ((reinterpret_cast<uintptr_t>(out) & 3u) == 0 && (nbytes & 3) == 0) {
                for (int i = lane; i < (nbytes >> 2); i += 32) reinterpret_cast<uint32_t *>(out)[i] = region[i];
            } else {
                const uint8_t *rb = reinterpret_cast<const uint8_t *>(region);
                for (int i = lane; i < nbytes; i += 32) out[i] = rb[i];
            }
            __syncwarp();
            for (int i = lane; i < b; i += 32) region[i] = 0u;
        }
        group_sync(gid, S::THREADS);
    }
}

// ------------------------------------------------------------------------------------------------------------ defragment
// Shared memory per group as in the fragment kernel, used differently: [0] planar rows of the finished blocks, [1] the interleaved
// out tile the bulk stores read (feds_dct_tma.cuh's defragment). `plain` = the decrypted private fragments (workspace).
template <int C, int PMAX>
__global__ void __launch_bounds__(PackedTileShape<C>::CTA, 1) defragment_dct_packed_tile_kernel(const __grid_constant__ DctParams p, const uint8_t *plain,
                                                                                                size_t plain_stride) {
    using S = TmaShape<C>;
    using PS = PackedTileShape<C>;
    constexpr int TB = S::TB;
    extern __shared__ __align__(128) uint32_t smem[];
    const int gid = threadIdx.x / S::THREADS, tid = threadIdx.x % S::THREADS, lane = threadIdx.x & 31;
    const int ch = (tid >> 5) % C, j = ((tid >> 5) / C) * 32 + lane;
    uint8_t *base = reinterpret_cast<uint8_t *>(smem) + TMA_BAR_BYTES;
    uint8_t *planar = base + (size_t)gid * 2 * S::PIX_BYTES, *out_tile = planar + S::PIX_BYTES;
    uint32_t *region = reinterpret_cast<uint32_t *>(base + (size_t)PS::GROUPS * 2 * S::PIX_BYTES) + (threadIdx.x >> 5) * PT_MAX_B;
    const int b = (int)p.packed_group_bytes, P = p.k + 1, bits = p.ac_bits;
    const unsigned tiles_per_plane = ((unsigned)p.nbr * p.nbc + TB - 1) / TB;
    const unsigned total = (unsigned)p.n_images * tiles_per_plane, step = gridDim.x * PS::GROUPS;
    const size_t plane = (size_t)p.nbr * p.nbc;
    unsigned t = blockIdx.x * PS::GROUPS + gid;
    // the block's 64 public bytes, one tile ahead
    uint4 xn[4];
    auto load_pub = [&](unsigned tt, uint4 (&x)[4]) {
        const TmaTile T = tma_decode_tile<C>(p, tt, tiles_per_plane);
        if (j < T.nb) {
            const uint4 *src = reinterpret_cast<const uint4 *>(p.pub + (size_t)T.n * p.pub_stride + 64 * ((size_t)ch * plane + T.B0 + j));
#pragma unroll
            for (int i = 0; i < 4; ++i) x[i] = __ldg(src + i);
        }
    };
    if (t < total) load_pub(t, xn);
#pragma unroll 1
    for (; t < total; t += step) {
        const TmaTile T = tma_decode_tile<C>(p, t, tiles_per_plane);
        const size_t blk0 = (size_t)ch * plane + T.B0;
        const int j0 = j - lane, ngroups = min(4, (T.nb - j0) / 8);
        if (ngroups > 0) {   // the warp's groups: ngroups * b bytes of the decrypted stream
            const uint8_t *in = plain + (size_t)T.n * plain_stride + ((blk0 + j0) >> 3) * (size_t)b;
            const int nbytes = ngroups * b;
            if ((reinterpret_cast<uintptr_t>(in) & 3u) == 0 && (nbytes & 3) == 0) {
                for (int i = lane; i < (nbytes >> 2); i += 32) region[i] = __ldg(reinterpret_cast<const uint32_t *>(in) + i);
            } else {
                uint8_t *rb = reinterpret_cast<uint8_t *>(region);
                for (int i = lane; i < nbytes; i += 32) rb[i] = __ldg(in + i);
            }
        }
        uint32_t x[16];
#pragma unroll
        for (int i = 0; i < 4; ++i) { x[4 * i] = xn[i].x; x[4 * i + 1] = xn[i].y; x[4 * i + 2] = xn[i].z; x[4 * i + 3] = xn[i].w; }
        if (t + step < total) load_pub(t + step, xn);
        __syncwarp();
        uint32_t rows[16];
        if (j < T.nb) {
            int32_t q[PMAX];
            const unsigned bitpos = (unsigned)lane * (unsigned)b;
            const uint32_t *word = region + (bitpos >> 5);
            unsigned long long buf = (unsigned long long)(*word >> (bitpos & 31u));
            int nbuf = 32 - (int)(bitpos & 31u);
#pragma unroll
            for (int z = 0; z < PMAX; ++z) {
                q[z] = 0;
                if (z < P) {
                    const int nb = z == 0 ? 11 : bits;
                    if (nbuf < nb) { buf |= (unsigned long long)*++word << nbuf; nbuf += 32; }
                    const uint32_t field = (uint32_t)buf & ((1u << nb) - 1u);
                    buf >>= nb;
                    nbuf -= nb;
                    int32_t v = (int32_t)field;
                    if (z > 0) {
                        const int32_t mag = (int32_t)(field & ((1u << (bits - 1)) - 1u));
                        v = (field >> (bits - 1)) ? -mag : mag;
                    }
                    q[z] = 16 * v;
                }
            }
            packed_restore_words<0, PMAX>(x, q, P, reinterpret_cast<uint32_t(&)[8]>(rows[0]));
            packed_restore_words<1, PMAX>(x, q, P, reinterpret_cast<uint32_t(&)[8]>(rows[8]));
        }
        if (tid == 0) bulk_wait_read0();   // the previous tile's pixel stores have read the out tile
        group_sync(gid, S::THREADS);
        if constexpr (C == 1) {
            if (j < T.nb) {
                uint32_t off, pitch;
                tma_pixel_slot<C>(T, j, off, pitch);
#pragma unroll
                for (int r = 0; r < 8; ++r) *reinterpret_cast<uint2 *>(out_tile + off + r * pitch) = make_uint2(rows[2 * r], rows[2 * r + 1]);
            }
        } else {
            if (j < T.nb) {
#pragma unroll
                for (int r = 0; r < 8; ++r) *reinterpret_cast<uint2 *>(planar + (ch * 8 + r) * (TB * 8) + j * 8) = make_uint2(rows[2 * r], rows[2 * r + 1]);
            }
            group_sync(gid, S::THREADS);
            tma_interleave<C>(T, planar, out_tile, tid);
        }
        fence_proxy_async();
        group_sync(gid, S::THREADS);
        if (tid == 0) tma_move_pixels<C, true>(p, T, smem_u32(out_tile), 0u);
    }
    if (tid == 0) bulk_wait0();
}

}  // namespace feds
