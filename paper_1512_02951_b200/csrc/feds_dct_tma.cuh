// feds_dct_tma.cuh — the digest-free DCT path on bulk asynchronous copies (TMA, cp.async.bulk; SASS UBLKCP), sm_100a:
// steps 1-4 and 6-8 of SURVEY.md 8(a), i.e. the report's own selective encryption (DCT + select + AES).
// The same tile groups are the producers / reconstruction groups of the fused digest kernels (feds_dct_fused.cuh).
//
//   A tile = TB consecutive 8x8 blocks of ONE image plane in linear block order (block row, block column), all C channels.
//   Because blocks are linear in the fragments too, the tile's public words of one channel are ONE contiguous
//   run of the public fragment, and likewise its private words: a tile touches HBM as 2 C flat runs plus 8 (or 16, when it
//   wraps into the next block row) pixel-row segments. Every one of those moves as one cp.async.bulk between global and
//   shared memory, issued by one elected thread of the group: no per-thread address arithmetic, no copy loops, nothing in the
//   issue stream (the round-1 tile kernels spent a third of their instructions on exactly that).
//   A group = WARPS warps; warp w transforms channel w % C, lane l block (w / C) * 32 + l of the tile, 64 coefficients in
//   registers. The channel is warp-uniform, so the byte selectors that pull a channel out of the interleaved pixels are
//   immediates (one PRMT per pixel, no funnel shifts).
//   uint8 -> float32: PRMT drops the byte into mantissa bits 8..15 of 2^15, giving 32768 + x exactly; the row pass of the DCT
//   starts with sums and differences only, which stay exact integers, the differences lose the bias by themselves and the one
//   sum of all eight (the DC term) is corrected with a single exact subtraction of 2^18: one FADD per row instead of eight, and
//   bit-identical results (every intermediate value is the same real number, exactly representable, as without the bias).
//   One persistent CTA per SM holds GROUPS such groups on named barriers; pixel tiles are double-buffered (fragment) and the
//   fragment stage is refilled as soon as it has been read (defragment), so copies overlap arithmetic without holding warps.
//   AES-128-CTR: as in feds_dct_tile.cuh (T0 replicated 32-fold, conflict-free).
//
// Requirements (the host routes everything else to the generic tile kernels of feds_dct_tile.cuh): w % 32 == 0 (all runs and
// row segments are 16-byte multiples at 16-byte aligned addresses) and w / 8 >= TB (a tile spans at most two block rows).
#pragma once
#include "feds_dct_tile.cuh"
#include "feds_aes_rep.cuh"

namespace feds {

template <int C> struct TmaShape {
    static constexpr int WARPS = (C == 1) ? 2 : C;       // per group
    static constexpr int THREADS = 32 * WARPS;
    static constexpr int TB = THREADS / C;               // blocks per tile and channel: 64 / 32 / 32
    static constexpr int GROUPS = (C == 1) ? 7 : (C == 3) ? 5 : 3;
    static constexpr int CTA = THREADS * GROUPS;
    static constexpr int BLOCK_ROW_BYTES = 8 * C;        // one pixel row of one block, all channels
    static constexpr int PIX_BYTES = TB * 8 * BLOCK_ROW_BYTES;   // one pixel tile
    // bulk loads are issued by lane 0 of the group's last warp, bulk stores by lane 0 of its first: the issuing warp runs ~150
    // instructions per tile that the others do not, and every barrier waits for the slowest warp
    static constexpr int LOADER = THREADS - 32;
};
constexpr int TMA_BAR_BYTES = 256;   // mbarriers of all groups (2 x 8 bytes each), behind the AES table

template <int C> __host__ __device__ inline int tma_stage_words(int k) {
    return C * (tile_run_stride(TmaShape<C>::TB * (63 - k)) + tile_run_stride(TmaShape<C>::TB * (k + 1)));
}
template <int C> __host__ __device__ inline size_t tma_group_bytes(int k) { return (size_t)2 * TmaShape<C>::PIX_BYTES + (size_t)tma_stage_words<C>(k) * 4; }
// `table_bytes`: the AES tables in front of everything else (T0 32-fold: 32 KB; the four-table layout of feds_aes_rep.cuh: 128 KB)
template <int C> __host__ __device__ inline size_t tma_smem_bytes(int k, int groups, size_t table_bytes = (size_t)T0_WORDS * 4) {
    return table_bytes + TMA_BAR_BYTES + (size_t)groups * tma_group_bytes<C>(k);
}
// one AES block on whichever table layout the kernel holds
template <bool SMALL, typename RkPtr> __device__ __forceinline__ void tile_aes(const T0Lane &T, const RkPtr rk, uint32_t (&s)[4]) { aes128_encrypt<SMALL>(T, rk, s); }
template <bool SMALL, typename RkPtr> __device__ __forceinline__ void tile_aes(const RepAes &A, const RkPtr rk, uint32_t (&s)[4]) { aes128_encrypt_rep32<SMALL>(A, rk, s); }
template <int C> __host__ __device__ inline bool tma_shape_ok(int w) { return (w % 32) == 0 && (w / 8) >= TmaShape<C>::TB; }

// ------------------------------------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
// global -> shared, completion counted in bytes on an mbarrier
__device__ __forceinline__ void bulk_load(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// shared -> global, completion tracked by the issuing thread's bulk groups
__device__ __forceinline__ void bulk_store(void *dst, uint32_t src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
// generic-proxy writes to shared memory (st.shared) before async-proxy reads of it (bulk store): by every writer, then a barrier
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ------------------------------------------------------------------------------------------------------------ tiles
struct TmaTile {
    int n;          // image
    unsigned B0;    // first block of the tile, linear in the plane (block row * nbc + block column)
    int nb;         // blocks in the tile (a multiple of 4)
    int br0, bc0;   // block row / column of the first block
    int n0;         // blocks in the first block row; the other nb - n0 start the next block row
};
template <int C>
__device__ __forceinline__ TmaTile tma_decode_tile(const DctParams &p, unsigned t, unsigned tiles_per_plane) {
    constexpr int TB = TmaShape<C>::TB;
    TmaTile T;
    T.n = (int)(t / tiles_per_plane);
    T.B0 = (t % tiles_per_plane) * TB;
    const unsigned plane = (unsigned)p.nbr * p.nbc;
    T.nb = (int)min((unsigned)TB, plane - T.B0);
    T.br0 = (int)(T.B0 / (unsigned)p.nbc);
    T.bc0 = (int)(T.B0 % (unsigned)p.nbc);
    T.n0 = min(T.nb, p.nbc - T.bc0);
    return T;
}
// Pixel tile in shared memory: segment 0 = 8 rows of n0 blocks (pitch n0 * 8C bytes), then segment 1 = 8 rows of nb - n0
// blocks. Byte offset of block j's first row and its row pitch:
template <int C>
__device__ __forceinline__ void tma_pixel_slot(const TmaTile &T, int j, uint32_t &off, uint32_t &pitch) {
    constexpr uint32_t BRB = TmaShape<C>::BLOCK_ROW_BYTES;
    if (j < T.n0) { off = (uint32_t)j * BRB; pitch = (uint32_t)T.n0 * BRB; }
    else { off = 8u * T.n0 * BRB + (uint32_t)(j - T.n0) * BRB; pitch = (uint32_t)(T.nb - T.n0) * BRB; }
}
// elected thread: the tile's pixel rows, global <-> shared (TO_GLOBAL: bulk stores, committed as one group)
template <int C, bool TO_GLOBAL>
__device__ __forceinline__ void tma_move_pixels(const DctParams &p, const TmaTile &T, uint32_t s_pix, uint32_t bar) {
    constexpr uint32_t BRB = TmaShape<C>::BLOCK_ROW_BYTES;
    const size_t row_bytes = (size_t)p.w * C;
    uint8_t *img = (TO_GLOBAL ? p.images_out : const_cast<uint8_t *>(p.images)) + (size_t)T.n * p.image_stride;
    if (!TO_GLOBAL) mbar_expect_tx(bar, (uint32_t)T.nb * 8u * BRB);
    const uint32_t b0 = (uint32_t)T.n0 * BRB, b1 = (uint32_t)(T.nb - T.n0) * BRB;
    uint8_t *g0 = img + (size_t)(8 * T.br0) * row_bytes + (size_t)(8 * T.bc0) * C;
    uint8_t *g1 = img + (size_t)(8 * (T.br0 + 1)) * row_bytes;
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        if (TO_GLOBAL) bulk_store(g0 + r * row_bytes, s_pix + r * b0, b0); else bulk_load(s_pix + r * b0, g0 + r * row_bytes, b0, bar);
    }
    if (b1) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            if (TO_GLOBAL) bulk_store(g1 + r * row_bytes, s_pix + 8 * b0 + r * b1, b1); else bulk_load(s_pix + 8 * b0 + r * b1, g1 + r * row_bytes, b1, bar);
        }
    }
    if (TO_GLOBAL) bulk_commit();
}
// elected thread: the tile's 2 C fragment runs, global <-> shared stage (public runs RSQ words apart, then private runs RSP apart)
template <int C, bool TO_GLOBAL>
__device__ __forceinline__ void tma_move_runs(const DctParams &p, const TmaTile &T, uint32_t s_pub, int RSQ, int RSP, uint32_t bar) {
    const int P = p.k + 1, Q = 63 - p.k;
    const uint32_t s_priv = s_pub + 4u * C * RSQ;
    const size_t plane = (size_t)p.nbr * p.nbc;
    uint8_t *pub = p.pub + (size_t)T.n * p.pub_stride, *priv = p.priv + (size_t)T.n * p.priv_stride;
    const uint32_t qb = (uint32_t)T.nb * Q * 4u, pb = (uint32_t)T.nb * P * 4u;
    if (!TO_GLOBAL) mbar_expect_tx(bar, (uint32_t)C * (qb + pb));
#pragma unroll
    for (int c = 0; c < C; ++c) {
        const size_t b0 = c * plane + T.B0;
        if (qb) { if (TO_GLOBAL) bulk_store(pub + b0 * Q * 4, s_pub + 4u * c * RSQ, qb); else bulk_load(s_pub + 4u * c * RSQ, pub + b0 * Q * 4, qb, bar); }
        if (TO_GLOBAL) bulk_store(priv + b0 * P * 4, s_priv + 4u * c * RSP, pb); else bulk_load(s_priv + 4u * c * RSP, priv + b0 * P * 4, pb, bar);
    }
    if (TO_GLOBAL) bulk_commit();
}

// ------------------------------------------------------------------------------------------------------------ pixels <-> registers
// 32768 + x, exactly: the byte goes to mantissa bits 8..15 of 2^15
__device__ __forceinline__ float byte_to_biased_float(uint32_t word, int pos) { return __uint_as_float(__byte_perm(word, 0x47000000u, 0x7404u + ((uint32_t)pos << 4))); }
__device__ __forceinline__ uint2 lds64(uint32_t a) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ uint4 lds128(uint32_t a) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
    return v;
}
// `blk` = shared-memory address of the block's first pixel row
template <int C, int CH>
__device__ __forceinline__ void load_block_biased(uint32_t blk, uint32_t pitch, float (&v)[64]) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const uint32_t row = blk + r * pitch;
        if (C == 1) {
            const uint2 q = lds64(row);
#pragma unroll
            for (int i = 0; i < 4; ++i) { v[8 * r + i] = byte_to_biased_float(q.x, i); v[8 * r + 4 + i] = byte_to_biased_float(q.y, i); }
        } else if (C == 3) {
            const uint2 q0 = lds64(row), q1 = lds64(row + 8), q2 = lds64(row + 16);
            const uint32_t wd[6] = {q0.x, q0.y, q1.x, q1.y, q2.x, q2.y};
#pragma unroll
            for (int i = 0; i < 8; ++i) v[8 * r + i] = byte_to_biased_float(wd[(3 * i + CH) >> 2], (3 * i + CH) & 3);
        } else {
            const uint4 a = lds128(row), b = lds128(row + 16);
            const uint32_t wd[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
            for (int i = 0; i < 8; ++i) v[8 * r + i] = byte_to_biased_float(wd[i], CH);
        }
    }
}
// dct8 of eight values that each carry a bias of 32768: same operations as dct8, the DC sum loses 8 * 32768 first (exact)
__device__ __forceinline__ void dct8_biased(float &x0, float &x1, float &x2, float &x3, float &x4, float &x5, float &x6, float &x7) {
    const float a0 = f_add(x0, x7), a1 = f_add(x1, x6), a2 = f_add(x2, x5), a3 = f_add(x3, x4);
    const float b0 = f_sub(x0, x7), b1 = f_sub(x1, x6), b2 = f_sub(x2, x5), b3 = f_sub(x3, x4);
    const float e0 = f_add(a0, a3), e1 = f_add(a1, a2), e2 = f_sub(a0, a3), e3 = f_sub(a1, a2);
    x0 = f_mul(FEDS_C4, f_sub(f_add(e0, e1), 262144.0f));
    x4 = f_mul(FEDS_C4, f_sub(e0, e1));
    x2 = f_fma(FEDS_C2, e2, f_mul(FEDS_C6, e3));
    x6 = f_fma(FEDS_C6, e2, f_mul(-FEDS_C2, e3));
    x1 = f_fma(FEDS_C1, b0, f_fma(FEDS_C3, b1, f_fma(FEDS_C5, b2, f_mul(FEDS_C7, b3))));
    x3 = f_fma(FEDS_C3, b0, f_fma(-FEDS_C7, b1, f_fma(-FEDS_C1, b2, f_mul(-FEDS_C5, b3))));
    x5 = f_fma(FEDS_C5, b0, f_fma(-FEDS_C1, b1, f_fma(FEDS_C7, b2, f_mul(FEDS_C3, b3))));
    x7 = f_fma(FEDS_C7, b0, f_fma(-FEDS_C5, b1, f_fma(FEDS_C3, b2, f_mul(-FEDS_C1, b3))));
}
__device__ __forceinline__ void dct8x8_biased(float (&v)[64]) {
#pragma unroll
    for (int r = 0; r < 8; ++r) dct8_biased(v[8 * r], v[8 * r + 1], v[8 * r + 2], v[8 * r + 3], v[8 * r + 4], v[8 * r + 5], v[8 * r + 6], v[8 * r + 7]);
#pragma unroll
    for (int c = 0; c < 8; ++c) dct8(v[c], v[8 + c], v[16 + c], v[24 + c], v[32 + c], v[40 + c], v[48 + c], v[56 + c]);
}
// pixels of block (ch, j) of the tile staged at s_pix -> 64 DCT coefficients
template <int C>
__device__ __forceinline__ void tma_block_dct(const uint8_t *s_pix, const TmaTile &T, int j, int ch, float (&v)[64]) {
    uint32_t off, pitch;
    tma_pixel_slot<C>(T, j, off, pitch);
    const uint32_t blk = smem_u32(s_pix) + off;
    if (C == 1) load_block_biased<1, 0>(blk, pitch, v);
    else if (ch == 0) load_block_biased<C, 0>(blk, pitch, v);   // warp-uniform branches: the channel selects immediates
    else if (ch == 1) load_block_biased<C, 1>(blk, pitch, v);
    else if (ch == 2) load_block_biased<C, 2>(blk, pitch, v);
    else load_block_biased<C, (C == 4 ? 3 : 0)>(blk, pitch, v);
    dct8x8_biased(v);
}

// AES-128-CTR over the staged private runs of a tile by the whole group (k + 1 not a multiple of 4): every counter block that
// overlaps a run is computed once. Run c holds words [W0_c, W0_c + nb * P) of the image's private stream.
template <int C, bool SMALL = false, typename Tab>
__device__ __forceinline__ void tma_aes_ctr_runs(const DctParams &p, const Tab &sT, const TmaTile &T, uint32_t *s_priv, int RSP, int P, int tid) {
    constexpr int THREADS = TmaShape<C>::THREADS, TB = TmaShape<C>::TB;
    uint32_t nonce[4];
    load_nonce(p, T.n, nonce);
    const int nw = T.nb * P;
    const int per = (TB * P + 3) / 4 + 1;   // >= counter blocks overlapping one run
    const unsigned long long plane = (unsigned long long)p.nbr * p.nbc;
    for (int idx = tid; idx < C * per; idx += THREADS) {
        const int c = idx / per, i = idx % per;
        const unsigned long long W0 = (c * plane + T.B0) * P;
        const unsigned long long blk = (W0 >> 2) + i;
        const long long first = (long long)(blk << 2) - (long long)W0;   // run-relative index of the block's first word
        if (first >= nw) continue;
        uint32_t ks[4];
        ctr_block(nonce, blk, ks);
        tile_aes<SMALL>(sT, p.rk, ks);
        uint32_t *run = s_priv + c * RSP;
        if (first >= 0 && first + 4 <= nw && (first & 3) == 0) {
            uint4 x = *reinterpret_cast<uint4 *>(run + first);
            x.x ^= ks[0]; x.y ^= ks[1]; x.z ^= ks[2]; x.w ^= ks[3];
            *reinterpret_cast<uint4 *>(run + first) = x;
        } else {
#pragma unroll
            for (int w = 0; w < 4; ++w) {
                const long long r = first + w;
                if (r >= 0 && r < nw) run[r] ^= ks[w];
            }
        }
    }
}
// AES-128-CTR of one block's own private words in the stage (4 | k + 1: they are whole counter blocks)
template <bool SMALL = false, typename Tab>
__device__ __forceinline__ void tma_aes_ctr_own(const DctParams &p, const Tab &sT, int n, unsigned long long w0, int P, uint32_t *my_priv) {
    uint32_t nonce[4];
    load_nonce(p, n, nonce);
#pragma unroll 1
    for (int g = 0; g < P; g += 4) {
        uint32_t ks[4];
        ctr_block(nonce, (w0 + g) >> 2, ks);
        tile_aes<SMALL>(sT, p.rk, ks);
        uint4 x = *reinterpret_cast<uint4 *>(my_priv + g);
        x.x ^= ks[0]; x.y ^= ks[1]; x.z ^= ks[2]; x.w ^= ks[3];
        *reinterpret_cast<uint4 *>(my_priv + g) = x;
    }
}

// ------------------------------------------------------------------------------------------------------------ one group's context
template <int C> struct TmaGroup {
    int gid, tid, ch, j;          // group in the CTA, thread in the group, channel and block-in-tile of this thread
    uint8_t *pix[2];              // fragment: two pixel tiles (double buffer); defragment: [0] planar rows, [1] interleaved out tile
    uint32_t *s_pub, *s_priv;     // fragment stage
    int RSQ, RSP;
    uint32_t bar[2];              // mbarriers (shared addresses)
};
template <int C>
__device__ __forceinline__ TmaGroup<C> tma_group_setup(uint32_t *smem, int k, int gid, int tid, size_t table_bytes = (size_t)T0_WORDS * 4) {
    using S = TmaShape<C>;
    TmaGroup<C> G;
    G.gid = gid; G.tid = tid;
    const int warp = tid >> 5, lane = tid & 31;
    G.ch = warp % C; G.j = (warp / C) * 32 + lane;
    uint8_t *base = reinterpret_cast<uint8_t *>(smem) + table_bytes + TMA_BAR_BYTES + (size_t)gid * tma_group_bytes<C>(k);
    G.pix[0] = base; G.pix[1] = base + S::PIX_BYTES;
    G.RSQ = tile_run_stride(S::TB * (63 - k)); G.RSP = tile_run_stride(S::TB * (k + 1));
    G.s_pub = reinterpret_cast<uint32_t *>(base + 2 * S::PIX_BYTES);
    G.s_priv = G.s_pub + C * G.RSQ;
    G.bar[0] = smem_u32(reinterpret_cast<uint8_t *>(smem) + table_bytes + 16 * gid);
    G.bar[1] = G.bar[0] + 8;
    return G;
}

// ------------------------------------------------------------------------------------------------------------ fragment: steps 1-4
// One tile, from the pixel tile in shared memory (already waited for) to the stage: DCT, zigzag split, AES. Ends with the
// barrier after which the elected thread may issue the bulk stores. `pre_stage` runs between the arithmetic and the first write
// to the stage (the caller waits there until the previous tile's stores have read the stage).
template <int C, int V, bool SMALL = false, typename Tab, typename PreStage>
__device__ __forceinline__ void tma_fragment_tile(const DctParams &p, const Tab &sT, const TmaGroup<C> &G, const TmaTile &T, const uint8_t *s_pix,
                                                  PreStage &&pre_stage) {
    constexpr ZigzagTable ZZ = make_zigzag();
    constexpr int THREADS = TmaShape<C>::THREADS;
    const int P = p.k + 1, Q = 63 - p.k;
    const bool act = G.j < T.nb;
    float v[64];
    if (act) tma_block_dct<C>(s_pix, T, G.j, G.ch, v);
    pre_stage();
    if (act) {
        uint32_t *my_pub = G.s_pub + G.ch * G.RSQ + G.j * Q - P;   // indexed by z
        uint32_t *my_priv = G.s_priv + G.ch * G.RSP + G.j * P;
#pragma unroll
        for (int g = 0; g < 64; g += V) {
            uint32_t x[V];
#pragma unroll
            for (int q = 0; q < V; ++q) x[q] = __float_as_uint(v[ZZ.pos[g + q]]);
            vec_store<V>(g < P ? my_priv + g : my_pub + g, x);
        }
        if (V == 4) tma_aes_ctr_own<SMALL>(p, sT, T.n, ((unsigned long long)G.ch * p.nbr * p.nbc + T.B0 + G.j) * P, P, my_priv);
    }
    if (V != 4) {
        group_sync(G.gid, THREADS);
        tma_aes_ctr_runs<C, SMALL>(p, sT, T, G.s_priv, G.RSP, P, G.tid);
    }
    fence_proxy_async();
    group_sync(G.gid, THREADS);
}

template <int C, int V>
__global__ void __launch_bounds__(TmaShape<C>::CTA, 1) fragment_dct_tma_kernel(const __grid_constant__ DctParams p) {
    using S = TmaShape<C>;
    extern __shared__ __align__(128) uint32_t smem[];
    const int gid = threadIdx.x / S::THREADS, tid = threadIdx.x % S::THREADS;
    const TmaGroup<C> G = tma_group_setup<C>(smem, p.k, gid, tid);
    if (tid == 0) { mbar_init(G.bar[0], 1); mbar_init(G.bar[1], 1); mbar_init_fence(); }
    load_t0_replicated(smem);   // ends with __syncthreads
    T0Lane sT;
    sT.tab = reinterpret_cast<const char *>(smem);
    sT.lane4 = 4u * (threadIdx.x & 31);
    const unsigned tiles_per_plane = ((unsigned)p.nbr * p.nbc + S::TB - 1) / S::TB;
    const unsigned total = (unsigned)p.n_images * tiles_per_plane, step = gridDim.x * S::GROUPS;
    unsigned t = blockIdx.x * S::GROUPS + gid;
    if (t < total && tid == S::LOADER) tma_move_pixels<C, false>(p, tma_decode_tile<C>(p, t, tiles_per_plane), smem_u32(G.pix[0]), G.bar[0]);
#pragma unroll 1
    for (unsigned it = 0; t < total; t += step, ++it) {
        const int s = it & 1;
        const TmaTile T = tma_decode_tile<C>(p, t, tiles_per_plane);
        // the other pixel tile was last read one iteration ago, before that iteration's barriers: refill it now
        if (tid == S::LOADER && t + step < total) tma_move_pixels<C, false>(p, tma_decode_tile<C>(p, t + step, tiles_per_plane), smem_u32(G.pix[s ^ 1]), G.bar[s ^ 1]);
        mbar_wait(G.bar[s], (it >> 1) & 1);
        tma_fragment_tile<C, V>(p, sT, G, T, G.pix[s], [&]() {
            if (tid == 0) bulk_wait_read0();   // the previous tile's stores have read the stage
            group_sync(gid, S::THREADS);
        });
        if (tid == 0) tma_move_runs<C, true>(p, T, smem_u32(G.s_pub), G.RSQ, G.RSP, 0u);
    }
    if (tid == 0) bulk_wait0();
}

// ------------------------------------------------------------------------------------------------------------ defragment: steps 6-8
// stage (already waited for) -> decrypt, merge, IDCT -> packed rows of this thread's block in registers (2 words per row)
template <int C, int V, bool SMALL = false, typename Tab>
__device__ __forceinline__ void tma_defragment_block(const DctParams &p, const Tab &sT, const TmaGroup<C> &G, const TmaTile &T, uint32_t (&rows)[16]) {
    constexpr ZigzagTable ZZ = make_zigzag();
    const int P = p.k + 1, Q = 63 - p.k;
    uint32_t *my_pub = G.s_pub + G.ch * G.RSQ + G.j * Q - P;   // indexed by z
    uint32_t *my_priv = G.s_priv + G.ch * G.RSP + G.j * P;
    if (V == 4) tma_aes_ctr_own<SMALL>(p, sT, T.n, ((unsigned long long)G.ch * p.nbr * p.nbc + T.B0 + G.j) * P, P, my_priv);
    float v[64];
#pragma unroll
    for (int g = 0; g < 64; g += V) {
        uint32_t x[V];
        vec_load<V>(g < P ? my_priv + g : my_pub + g, x);
#pragma unroll
        for (int q = 0; q < V; ++q) v[ZZ.pos[g + q]] = __uint_as_float(x[q]);
    }
    idct8x8(v);
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        rows[2 * r] = pack4_u8(v[8 * r], v[8 * r + 1], v[8 * r + 2], v[8 * r + 3]);
        rows[2 * r + 1] = pack4_u8(v[8 * r + 4], v[8 * r + 5], v[8 * r + 6], v[8 * r + 7]);
    }
}
// planar rows [ch][r][TB x 8 bytes] -> pixel-interleaved out tile (segment layout of tma_pixel_slot), by the whole group
template <int C>
__device__ __forceinline__ void tma_interleave(const TmaTile &T, const uint8_t *planar, uint8_t *out, int tid) {
    constexpr int THREADS = TmaShape<C>::THREADS, TB = TmaShape<C>::TB;
    constexpr int PLANE = 8 * TB * 8;
#pragma unroll 1
    for (int q = tid; q < 8 * TB; q += THREADS) {
        const int r = q / TB, j = q % TB;
        if (j >= T.nb) continue;
        uint32_t off, pitch;
        tma_pixel_slot<C>(T, j, off, pitch);
        uint8_t *row = out + off + r * pitch;
        const uint8_t *src = planar + r * (TB * 8) + j * 8;
        const uint2 R = *reinterpret_cast<const uint2 *>(src), Gc = *reinterpret_cast<const uint2 *>(src + PLANE), B = *reinterpret_cast<const uint2 *>(src + 2 * PLANE);
        if (C == 3) {
            const uint32_t rg0 = __byte_perm(R.x, Gc.x, 0x5140), rg1 = __byte_perm(R.x, Gc.x, 0x7362);   // R0 G0 R1 G1 | R2 G2 R3 G3
            const uint32_t rg2 = __byte_perm(R.y, Gc.y, 0x5140), rg3 = __byte_perm(R.y, Gc.y, 0x7362);
            uint2 *o = reinterpret_cast<uint2 *>(row);
            o[0] = make_uint2(__byte_perm(rg0, B.x, 0x2410), __byte_perm(__byte_perm(rg0, B.x, 0x0053), rg1, 0x5410));   // R0 G0 B0 R1 | G1 B1 R2 G2
            o[1] = make_uint2(__byte_perm(rg1, B.x, 0x7326), __byte_perm(rg2, B.y, 0x2410));                             // B2 R3 G3 B3 | ...
            o[2] = make_uint2(__byte_perm(__byte_perm(rg2, B.y, 0x0053), rg3, 0x5410), __byte_perm(rg3, B.y, 0x7326));
        } else {
            const uint2 Al = *reinterpret_cast<const uint2 *>(src + 3 * PLANE);
            const uint32_t rg0 = __byte_perm(R.x, Gc.x, 0x5140), rg1 = __byte_perm(R.x, Gc.x, 0x7362);
            const uint32_t ba0 = __byte_perm(B.x, Al.x, 0x5140), ba1 = __byte_perm(B.x, Al.x, 0x7362);
            const uint32_t rg2 = __byte_perm(R.y, Gc.y, 0x5140), rg3 = __byte_perm(R.y, Gc.y, 0x7362);
            const uint32_t ba2 = __byte_perm(B.y, Al.y, 0x5140), ba3 = __byte_perm(B.y, Al.y, 0x7362);
            uint4 *o = reinterpret_cast<uint4 *>(row);
            o[0] = make_uint4(__byte_perm(rg0, ba0, 0x5410), __byte_perm(rg0, ba0, 0x7632), __byte_perm(rg1, ba1, 0x5410), __byte_perm(rg1, ba1, 0x7632));
            o[1] = make_uint4(__byte_perm(rg2, ba2, 0x5410), __byte_perm(rg2, ba2, 0x7632), __byte_perm(rg3, ba3, 0x5410), __byte_perm(rg3, ba3, 0x7632));
        }
    }
}
// One tile from the stage (already waited for) to the out tile in shared memory, ending with the barrier after which the elected
// thread may issue the pixel stores. `stage_read` runs right after the barrier that follows the last read of the stage (the caller
// refills the stage there); before that barrier the elected thread has waited for the previous out tile to be read.
template <int C, int V, bool SMALL = false, typename Tab, typename StageRead>
__device__ __forceinline__ void tma_defragment_tile(const DctParams &p, const Tab &sT, const TmaGroup<C> &G, const TmaTile &T, StageRead &&stage_read) {
    constexpr int THREADS = TmaShape<C>::THREADS, TB = TmaShape<C>::TB;
    const bool act = G.j < T.nb;
    if (V != 4) {
        tma_aes_ctr_runs<C, SMALL>(p, sT, T, G.s_priv, G.RSP, p.k + 1, G.tid);
        group_sync(G.gid, THREADS);
    }
    uint32_t rows[16];
    if (act) tma_defragment_block<C, V, SMALL>(p, sT, G, T, rows);
    if (G.tid == 0) bulk_wait_read0();   // the previous tile's pixel stores have read the out tile
    group_sync(G.gid, THREADS);
    stage_read();
    if constexpr (C == 1) {
        if (act) {
            uint32_t off, pitch;
            tma_pixel_slot<C>(T, G.j, off, pitch);
#pragma unroll
            for (int r = 0; r < 8; ++r) *reinterpret_cast<uint2 *>(G.pix[1] + off + r * pitch) = make_uint2(rows[2 * r], rows[2 * r + 1]);
        }
    } else {
        if (act) {
#pragma unroll
            for (int r = 0; r < 8; ++r) *reinterpret_cast<uint2 *>(G.pix[0] + (G.ch * 8 + r) * (TB * 8) + G.j * 8) = make_uint2(rows[2 * r], rows[2 * r + 1]);
        }
        group_sync(G.gid, THREADS);
        tma_interleave<C>(T, G.pix[0], G.pix[1], G.tid);
    }
    fence_proxy_async();
    group_sync(G.gid, THREADS);
}

template <int C, int V>
__global__ void __launch_bounds__(TmaShape<C>::CTA, 1) defragment_dct_tma_kernel(const __grid_constant__ DctParams p) {
    using S = TmaShape<C>;
    extern __shared__ __align__(128) uint32_t smem[];
    const int gid = threadIdx.x / S::THREADS, tid = threadIdx.x % S::THREADS;
    const TmaGroup<C> G = tma_group_setup<C>(smem, p.k, gid, tid);
    if (tid == 0) { mbar_init(G.bar[0], 1); mbar_init(G.bar[1], 1); mbar_init_fence(); }
    load_t0_replicated(smem);
    T0Lane sT;
    sT.tab = reinterpret_cast<const char *>(smem);
    sT.lane4 = 4u * (threadIdx.x & 31);
    const unsigned tiles_per_plane = ((unsigned)p.nbr * p.nbc + S::TB - 1) / S::TB;
    const unsigned total = (unsigned)p.n_images * tiles_per_plane, step = gridDim.x * S::GROUPS;
    unsigned t = blockIdx.x * S::GROUPS + gid;
    if (t < total && tid == S::LOADER) tma_move_runs<C, false>(p, tma_decode_tile<C>(p, t, tiles_per_plane), smem_u32(G.s_pub), G.RSQ, G.RSP, G.bar[0]);
#pragma unroll 1
    for (unsigned it = 0; t < total; t += step, ++it) {
        const TmaTile T = tma_decode_tile<C>(p, t, tiles_per_plane);
        mbar_wait(G.bar[0], it & 1);
        tma_defragment_tile<C, V>(p, sT, G, T, [&]() {
            if (tid == S::LOADER && t + step < total) tma_move_runs<C, false>(p, tma_decode_tile<C>(p, t + step, tiles_per_plane), smem_u32(G.s_pub), G.RSQ, G.RSP, G.bar[0]);
        });
        if (tid == 0) tma_move_pixels<C, true>(p, T, smem_u32(G.pix[1]), 0u);
    }
    if (tid == 0) bulk_wait0();
}

}  // namespace feds
