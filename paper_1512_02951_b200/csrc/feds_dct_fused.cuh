// feds_dct_fused.cuh — the DCT path WITH digests as one warp-specialised persistent kernel per direction (SURVEY.md 8(a) steps
// 1-5 and 6-8 with verification), sm_100a.
//
// The digest path is bound by the integer (ALU) pipe: one SHA-256 compression per 64 stored bytes is ~1040 shift / logic /
// byte-permute operations that only that pipe executes, against 5 bytes of HBM traffic per pixel, while the
// transform side (DCT, select, AES, data movement) is bound by instruction issue and memory latency and barely touches that pipe.
// Run one after the other the two cost their sum; in ONE kernel, on the same SMs, the transform hides in the hash's shadow:
//
//   * TILE warps (two warpgroups): the bulk-copy tile groups of feds_dct_tma.cuh, unchanged -- pixel rows and fragment runs move
//     as cp.async.bulk between HBM and shared memory, the arithmetic runs on 64 registers per 8x8 block.
//   * HASH warps (the other warpgroups, 72 registers): lane l owns one Merkle leaf (8 consecutive blocks of one channel,
//     DESIGN.md 2.1) and streams its bytes, 64 at a time, straight from the fragment buffers into the message registers -- the
//     registers-only loop of dct_leaves_hash_kernel. A hash item = the 32 leaves of one channel inside a UNIT of 256 consecutive
//     blocks of a plane; the warps take the CTA's items round-robin.
//
// Fragmenting, a unit is hashed once all of its tiles have been stored: every tile group publishes, in shared memory, how far
// along its tile sequence all bulk stores have completed (cp.async.bulk.wait_group, then a release fence), and a hash warp
// acquires that before its first load. Tile groups never wait for hash warps. Defragmenting, both kinds of warps only read the
// fragments, so they share nothing but the SM.
//
// Requirements (the host routes everything else to tile kernel + leaf-hash kernel): the bulk-copy tile kernels' (w % 32 == 0,
// at least one tile per block row) and (w / 8) % 8 == 0, so that leaves are 8 consecutive blocks in linear block order.
#pragma once
#include "feds_dct_tma.cuh"

namespace feds {

constexpr int FU_UNIT_BLOCKS = 32 * G_BLOCKS;   // 32 leaves of 8 blocks: one hash item per channel
constexpr int FU_TILE_WARPS = 8;                // two warpgroups (setmaxnreg acts on aligned groups of 4 warps)
constexpr int FU_HASH_REGS = 72;
constexpr int FU_CTL_OFFSET = 128;              // progress words sit behind the groups' mbarriers inside TMA_BAR_BYTES
// AES tables of the tile role: the four-table layout (feds_aes_rep.cuh), 128 KB: one ALU-pipe instruction per lookup instead of
// three -- in this kernel the ALU pipe is the contended resource, and the tile role's AES was 40 % of its ALU-pipe work
constexpr size_t FU_TABLE_BYTES = (size_t)REP4_TABLE_WORDS * 4;

template <int C, int HW> struct FuShape {
    static constexpr int THREADS = (HW + FU_TILE_WARPS) * 32;
    static constexpr int NP = FU_TILE_WARPS / TmaShape<C>::WARPS;            // tile groups: 4 / 2 / 2
    static constexpr int TPU = FU_UNIT_BLOCKS / TmaShape<C>::TB;             // tiles per unit: 4 / 8 / 8
    // registers: HW * 72 + 8 * TILE_REGS <= (HW + 8) * (registers per thread at launch)
    static constexpr int TILE_REGS = (HW >= 16) ? 96 : 128;
};
template <int C> __host__ __device__ inline size_t fu_smem_bytes(int k, int np) { return tma_smem_bytes<C>(k, np, FU_TABLE_BYTES); }
template <int C> __host__ __device__ inline bool fu_shape_ok(int w) { return tma_shape_ok<C>(w) && ((w / 8) % G_BLOCKS) == 0; }

__device__ __forceinline__ int fu_ld_volatile(const int *p) {
    int v;
    asm volatile("ld.volatile.shared.s32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void fu_st_volatile(int *p, int v) { asm volatile("st.volatile.shared.s32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory"); }
__device__ __forceinline__ void fu_fence() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }

// the CTA's units: U = blockIdx.x + i * gridDim.x, i = 0 .. n_units - 1; tile sequence number s = TPU * i + t
struct FuWork {
    unsigned units_per_plane, tiles_per_plane, n_units;
};
template <int C>
__device__ __forceinline__ FuWork fu_work(const DctParams &p) {
    FuWork W;
    const unsigned plane = (unsigned)p.nbr * p.nbc;
    W.units_per_plane = (plane + FU_UNIT_BLOCKS - 1) / FU_UNIT_BLOCKS;
    W.tiles_per_plane = (plane + TmaShape<C>::TB - 1) / TmaShape<C>::TB;
    const unsigned total = (unsigned)p.n_images * W.units_per_plane;
    W.n_units = blockIdx.x < total ? (total - blockIdx.x + gridDim.x - 1) / gridDim.x : 0u;
    return W;
}
// tile with sequence number s of this CTA; false when the unit has no such tile (the last unit of a plane may be short)
template <int C, int TPU>
__device__ __forceinline__ bool fu_tile(const DctParams &p, const FuWork &W, unsigned s, TmaTile &T) {
    const unsigned i = s / TPU, t = s % TPU;
    const unsigned U = blockIdx.x + i * gridDim.x;
    const unsigned n = U / W.units_per_plane, up = U % W.units_per_plane;
    const unsigned tile = up * TPU + t;
    if (tile >= W.tiles_per_plane) return false;
    T = tma_decode_tile<C>(p, n * W.tiles_per_plane + tile, W.tiles_per_plane);
    return true;
}

// ------------------------------------------------------------------------------------------------------------ HASH role
// SHA-256 of `nwords` 32-bit words at src (16-byte aligned; every byte is read once: no use for L1)
__device__ __forceinline__ void fu_hash_words(const uint32_t *src, unsigned nwords, const uint32_t one, uint32_t (&H)[8]) {
    uint32_t w[16];
    uint4 nx[4];
    sha256_init(H);
    const unsigned full = nwords >> 4, tail = nwords & 15u;
    const unsigned nblocks = full + (tail > 13u ? 2u : 1u);   // + the 0x80 marker and the bit length (FIPS 180-4 5.1.1)
    auto fetch = [&](unsigned blk) {
        const uint4 *q = reinterpret_cast<const uint4 *>(src + 16 * (size_t)blk);
#pragma unroll
        for (int i = 0; i < 4; ++i) nx[i] = __ldcg(q + i);
    };
    if (full > 0) fetch(0);
    // ONE compression site for data and padding blocks: the loop body is all the code a hash warp runs in steady state
#pragma unroll 1
    for (unsigned i = 0; i < nblocks; ++i) {
        if (i < full) {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                w[4 * q] = bswap32(nx[q].x); w[4 * q + 1] = bswap32(nx[q].y); w[4 * q + 2] = bswap32(nx[q].z); w[4 * q + 3] = bswap32(nx[q].w);
            }
            if (i + 1 < full) fetch(i + 1);
        } else {
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const unsigned idx = 16u * i + j;   // word index in the message
                uint32_t x = 0u;
                if (idx < nwords) x = bswap32(__ldcg(src + idx));
                else if (idx == nwords) x = 0x80000000u;
                w[j] = x;
            }
            if (i == nblocks - 1) w[15] = nwords * 32u;   // message bits (< 2^32: a leaf is at most 2 KB)
        }
        sha256_compress_rolled_fma(H, w, one);
    }
}

// hash warp hw of HW: items q = hw, hw + HW, ...; item q = (unit q / C of this CTA, channel q % C)
template <int C, int HW, int NP, int TPU, bool WAIT>
__device__ __forceinline__ void fu_hash_role(const DctParams &p, const FuWork &W, const int *progress, int hw, int lane) {
    const int P = p.k + 1, Q = 63 - p.k;
    const unsigned plane = (unsigned)p.nbr * p.nbc;
#pragma unroll 1
    for (unsigned q = (unsigned)hw;; q += HW) {
        const unsigned i = q / C, ch = q % C;
        if (i >= W.n_units) break;
        if (WAIT) {   // every tile of the unit has been stored (and of all earlier units)
            const int need = (int)(TPU * (i + 1));
#pragma unroll 1
            for (int g = 0; g < NP; ++g)
                while (fu_ld_volatile(progress + g) < need) __nanosleep(256);
            fu_fence();
        }
        const unsigned U = blockIdx.x + i * gridDim.x;
        const unsigned n = U / W.units_per_plane, up = U % W.units_per_plane;
        const unsigned B = up * FU_UNIT_BLOCKS + G_BLOCKS * lane;   // first block of this lane's leaf
        if (B >= plane) continue;                                   // a short last unit: no leaf for this lane
        const size_t b0 = (size_t)ch * plane + B;
        const size_t li = b0 / G_BLOCKS;                            // leaf index in fragment order
#pragma unroll 1
        for (int f = 0; f < 2; ++f) {   // 0: public, 1: private (ciphertext)
            const int Wd = f ? P : Q;
            if (Wd == 0) continue;      // k = 63: the public fragment is empty, its root is written elsewhere
            const uint32_t *src = reinterpret_cast<const uint32_t *>(f ? p.priv + (size_t)n * p.priv_stride : p.pub + (size_t)n * p.pub_stride) + b0 * Wd;
            uint32_t H[8];
            fu_hash_words(src, (unsigned)(G_BLOCKS * Wd), p.one, H);
            store_digest(p.leaves + (((size_t)n * 2 + (f ? 0 : 1)) * p.leaves_per_image + li) * 32, H);
        }
    }
}

// ------------------------------------------------------------------------------------------------------------ TILE roles
template <int C, int V, int NP, int TPU>
__device__ __forceinline__ void fu_fragment_tiles(const DctParams &p, const FuWork &W, const RepAes &sT, const TmaGroup<C> &G, int *progress) {
    using S = TmaShape<C>;
    const unsigned s_end = TPU * W.n_units;
    const int gid = G.gid, tid = G.tid;
    TmaTile T, Tn;
    unsigned s = (unsigned)gid;
    while (s < s_end && !fu_tile<C, TPU>(p, W, s, T)) s += NP;
    if (s < s_end && tid == TmaShape<C>::LOADER) tma_move_pixels<C, false>(p, T, smem_u32(G.pix[0]), G.bar[0]);
#pragma unroll 1
    for (unsigned it = 0; s < s_end; ++it) {
        const int st = it & 1;
        unsigned sn = s + NP;
        while (sn < s_end && !fu_tile<C, TPU>(p, W, sn, Tn)) sn += NP;
        if (tid == TmaShape<C>::LOADER && sn < s_end) tma_move_pixels<C, false>(p, Tn, smem_u32(G.pix[st ^ 1]), G.bar[st ^ 1]);
        mbar_wait(G.bar[st], (it >> 1) & 1);
        tma_fragment_tile<C, V, true>(p, sT, G, T, G.pix[st], [&]() {
            if (tid == 0) {
                bulk_wait0();    // the previous tile's stores are complete: its stage is free, and everything before s is in memory
                fu_fence();
                fu_st_volatile(progress + gid, (int)s);
            }
            group_sync(gid, S::THREADS);
        });
        if (tid == 0) tma_move_runs<C, true>(p, T, smem_u32(G.s_pub), G.RSQ, G.RSP, 0u);
        s = sn;
        T = Tn;
    }
    if (tid == 0) {
        bulk_wait0();
        fu_fence();
        fu_st_volatile(progress + gid, 0x7fffffff);
    }
}
template <int C, int V, int NP, int TPU>
__device__ __forceinline__ void fu_defragment_tiles(const DctParams &p, const FuWork &W, const RepAes &sT, const TmaGroup<C> &G) {
    const unsigned s_end = TPU * W.n_units;
    const int gid = G.gid, tid = G.tid;
    TmaTile T, Tn;
    unsigned s = (unsigned)gid;
    while (s < s_end && !fu_tile<C, TPU>(p, W, s, T)) s += NP;
    if (s < s_end && tid == TmaShape<C>::LOADER) tma_move_runs<C, false>(p, T, smem_u32(G.s_pub), G.RSQ, G.RSP, G.bar[0]);
#pragma unroll 1
    for (unsigned it = 0; s < s_end; ++it) {
        unsigned sn = s + NP;
        while (sn < s_end && !fu_tile<C, TPU>(p, W, sn, Tn)) sn += NP;
        mbar_wait(G.bar[0], it & 1);
        tma_defragment_tile<C, V, true>(p, sT, G, T, [&]() {
            if (tid == TmaShape<C>::LOADER && sn < s_end) tma_move_runs<C, false>(p, Tn, smem_u32(G.s_pub), G.RSQ, G.RSP, G.bar[0]);
        });
        if (tid == 0) tma_move_pixels<C, true>(p, T, smem_u32(G.pix[1]), 0u);
        s = sn;
        T = Tn;
    }
    if (tid == 0) bulk_wait0();
}

// ------------------------------------------------------------------------------------------------------------ kernel
template <int C, int V, int HW, bool FRAGMENT>
__global__ void __launch_bounds__(FuShape<C, HW>::THREADS, 1) dct_fused_kernel(const __grid_constant__ DctParams p) {
    using F = FuShape<C, HW>;
    using S = TmaShape<C>;
    extern __shared__ __align__(128) uint32_t smem[];
    int *progress = reinterpret_cast<int *>(reinterpret_cast<uint8_t *>(smem) + FU_TABLE_BYTES + FU_CTL_OFFSET);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // the tile warps come FIRST: the issue arbiter favours the CTA's oldest warps, and the tile warps, which are latency-bound and
    // ask for few issue slots, must never queue behind the always-ready hash warps (measured: placed last they were starved
    // to an eighth of their rate and the two roles ran one after the other)
    const bool tile_wg = warp < FU_TILE_WARPS;
    const int gid = tile_wg ? warp / S::WARPS : 0, tid = tile_wg ? (warp % S::WARPS) * 32 + lane : 0;
    const bool tile_warp = tile_wg && gid < F::NP;             // (C = 3: two warps of the tile warpgroups have no group)
    if (tile_warp && tid == 0) {
        const uint32_t bar = smem_u32(reinterpret_cast<uint8_t *>(smem) + FU_TABLE_BYTES + 16 * gid);
        mbar_init(bar, 1); mbar_init(bar + 8, 1); mbar_init_fence();
    }
    if (threadIdx.x < F::NP) progress[threadIdx.x] = 0;
    {   // T0..T3, every entry replicated 32 times (lane l reads copy l in bank l)
        const uint32_t *src = &g_aes.T[0][0];
        for (int i = threadIdx.x; i < REP4_TABLE_WORDS; i += blockDim.x) smem[i] = src[i >> 5];
        __syncthreads();
    }
    const FuWork W = fu_work<C>(p);
    if (!tile_wg) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(FU_HASH_REGS));
        fu_hash_role<C, HW, F::NP, F::TPU, FRAGMENT>(p, W, progress, warp - FU_TILE_WARPS, lane);
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(F::TILE_REGS));
        if (tile_warp) {
            const TmaGroup<C> G = tma_group_setup<C>(smem, p.k, gid, tid, FU_TABLE_BYTES);
            RepAes sT;
            sT.base = smem_u32(smem) + 4u * lane;
            sT.c128 = p.c128;
            if (FRAGMENT) fu_fragment_tiles<C, V, F::NP, F::TPU>(p, W, sT, G, progress);
            else fu_defragment_tiles<C, V, F::NP, F::TPU>(p, W, sT, G);
        }
    }
}

}  // namespace feds
