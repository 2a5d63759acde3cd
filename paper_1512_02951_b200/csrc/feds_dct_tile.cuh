// feds_dct_tile.cuh — the digest-free DCT path (FEDS_FLAG_NO_DIGEST; defragment without expected digests): steps 1-4
// and 6-8 of SURVEY.md 8(a) with no SHA-256, i.e. the report's own selective encryption (DCT + select + AES, P:488-494,
// P:607), which is bound by HBM and not by the integer pipe. Shaped for bandwidth instead of for a serial hash:
//
//   A CTA owns a tile of TB consecutive 8x8 blocks of one block row, all C channels; thread (j, ch) transforms one block
//   in 64 registers. The fragments of the tile are staged in shared memory in exactly their global byte order (the public
//   runs of consecutive blocks of one channel are contiguous), so the traffic with HBM is a flat,
//   fully coalesced 128-bit copy in both directions; AES-128-CTR is applied to the private words on their way through.
//   One persistent CTA per SM holds GROUPS independent thread groups (3-4 warps each, synchronised with their own named
//   barrier), each working on its own tile with its own stage, so one tile's loads overlap another's arithmetic and
//   stores. The groups share one AES table: T0 only, each entry replicated 32 times so that lane l reads copy l, which
//   lies in bank l -- every lookup is conflict-free (random lookups in a plain 4 KB table set collide ~3.4-fold and
//   were measured to cost a third of the kernel's time); T1..T3 are byte rotations of T0.
#pragma once
#include "feds_dct.cuh"
#include "feds_sha_coop.cuh"

namespace feds {

template <int C> struct TileShape {
    static constexpr int THREADS = (C == 3) ? 96 : 128;   // per group
    static constexpr int TB = THREADS / C;                // blocks per tile and channel
    static constexpr int GROUPS = (C == 3) ? 6 : 4;
    static constexpr int CTA = THREADS * GROUPS;
};
constexpr int T0_REPL = 32, T0_WORDS = 256 * T0_REPL;
// Words between the staged runs of two channels: the smallest count >= words that is 20 mod 32, so that the C lanes of one
// block column (adjacent lanes) and their neighbours land in different banks when they write their runs with 128-bit stores.
__host__ __device__ inline int tile_run_stride(int words) { return ((words + 11) / 32) * 32 + 20; }
// words of one group's shared memory: the two staged fragments
template <int C> __host__ __device__ inline int tile_group_words(int k) {
    return C * (tile_run_stride(TileShape<C>::TB * (63 - k)) + tile_run_stride(TileShape<C>::TB * (k + 1)));
}
template <int C> __host__ __device__ inline size_t tile_smem_bytes(int k) {
    return (size_t)(T0_WORDS + TileShape<C>::GROUPS * tile_group_words<C>(k)) * 4;
}

// AES-128 rounds on the lane's own copies of T0 (copy l of entry x at byte x * 128 + l * 4; lane4 = 4 * lane): every lookup
// is shift, mask-and-or-in-the-lane, LDS, and for T1..T3 one byte rotation of the T0 word. Same arithmetic as aes128_encrypt.
struct T0Lane {
    const char *tab;
    uint32_t lane4;
};
template <int BYTE, int TABLE>
__device__ __forceinline__ uint32_t t0_lookup(const T0Lane &T, uint32_t word) {
    uint32_t o;
    if (BYTE == 0) o = ((word << 7) & 0x7f80u) | T.lane4;
    else if (BYTE == 1) o = ((word >> 1) & 0x7f80u) | T.lane4;
    else if (BYTE == 2) o = ((word >> 9) & 0x7f80u) | T.lane4;
    else o = ((word >> 17) & 0x7f80u) | T.lane4;
    const uint32_t v = *reinterpret_cast<const uint32_t *>(T.tab + o);
    return TABLE == 0 ? v : __funnelshift_l(v, v, 8 * TABLE);
}
// ROLLED: the nine middle rounds as a loop (round keys indexed at run time): a tenth of the code, for kernels whose hot code
// must share the SM's 32 KB instruction cache with a SHA-256 loop (feds_dct_fused.cuh).
template <bool ROLLED = false, typename RkPtr>
__device__ __forceinline__ void aes128_encrypt(const T0Lane &T, const RkPtr rk, uint32_t (&s)[4]) {
    uint32_t s0 = s[0] ^ rk[0], s1 = s[1] ^ rk[1], s2 = s[2] ^ rk[2], s3 = s[3] ^ rk[3];
#define FEDS_ROUND(r)                                                                                                                       \
    {                                                                                                                                       \
        const uint32_t t0 = t0_lookup<0, 0>(T, s0) ^ t0_lookup<1, 1>(T, s1) ^ t0_lookup<2, 2>(T, s2) ^ t0_lookup<3, 3>(T, s3) ^ rk[4 * (r) + 0]; \
        const uint32_t t1 = t0_lookup<0, 0>(T, s1) ^ t0_lookup<1, 1>(T, s2) ^ t0_lookup<2, 2>(T, s3) ^ t0_lookup<3, 3>(T, s0) ^ rk[4 * (r) + 1]; \
        const uint32_t t2 = t0_lookup<0, 0>(T, s2) ^ t0_lookup<1, 1>(T, s3) ^ t0_lookup<2, 2>(T, s0) ^ t0_lookup<3, 3>(T, s1) ^ rk[4 * (r) + 2]; \
        const uint32_t t3 = t0_lookup<0, 0>(T, s3) ^ t0_lookup<1, 1>(T, s0) ^ t0_lookup<2, 2>(T, s1) ^ t0_lookup<3, 3>(T, s2) ^ rk[4 * (r) + 3]; \
        s0 = t0; s1 = t1; s2 = t2; s3 = t3;                                                                                                 \
    }
    if (ROLLED) {
#pragma unroll 1
        for (int r = 1; r < 10; ++r) FEDS_ROUND(r)
    } else {
#pragma unroll
        for (int r = 1; r < 10; ++r) FEDS_ROUND(r)
    }
#undef FEDS_ROUND
    // final round: SubBytes + ShiftRows; T0 = (2S, S, S, 3S): S is byte 1 (and 2) of every T0 word
#define FEDS_LAST(a, b, c, d)                                                                                          \
    __byte_perm(__byte_perm(t0_lookup<0, 0>(T, a), t0_lookup<1, 0>(T, b), 0x3251), __byte_perm(t0_lookup<2, 0>(T, c), t0_lookup<3, 0>(T, d), 0x5210), 0x7610)
    const uint32_t u0 = FEDS_LAST(s0, s1, s2, s3), u1 = FEDS_LAST(s1, s2, s3, s0), u2 = FEDS_LAST(s2, s3, s0, s1), u3 = FEDS_LAST(s3, s0, s1, s2);
#undef FEDS_LAST
    s[0] = u0 ^ rk[40]; s[1] = u1 ^ rk[41]; s[2] = u2 ^ rk[42]; s[3] = u3 ^ rk[43];
}
__device__ __forceinline__ void load_t0_replicated(uint32_t *sTab) {
    const uint32_t *src = &g_aes.T[0][0];
    for (int i = threadIdx.x; i < T0_WORDS; i += blockDim.x) sTab[i] = src[i / T0_REPL];
    __syncthreads();
}
__device__ __forceinline__ void group_sync(int gid, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(gid + 1), "r"(nthreads) : "memory"); }

struct TileCoord {
    int n, br, bc0, nb;  // image, block row, first block column, blocks in the tile
};
template <int C>
__device__ __forceinline__ TileCoord decode_tile(const DctParams &p, unsigned t, int tiles_per_row) {
    TileCoord T;
    const unsigned per_image = (unsigned)p.nbr * tiles_per_row;
    T.n = (int)(t / per_image);
    const unsigned r = t % per_image;
    T.br = (int)(r / tiles_per_row);
    T.bc0 = (int)(r % tiles_per_row) * TileShape<C>::TB;
    T.nb = min(TileShape<C>::TB, p.nbc - T.bc0);
    return T;
}

// flat copy of `words` 32-bit words between shared and global memory by the whole CTA; 128-bit when both ends allow.
// Global -> shared goes through cp.async (LDGSTS): no register staging, every thread keeps all of its 16-byte pieces in
// flight at once; the caller waits with tile_copy_wait() before the barrier.
template <bool TO_GLOBAL, int THREADS>
__device__ __forceinline__ void tile_copy(uint32_t *g, uint32_t *s, int words, int tid) {
    if (((reinterpret_cast<uintptr_t>(g) & 15u) == 0) && ((words & 3) == 0)) {
        uint4 *g4 = reinterpret_cast<uint4 *>(g);
        uint4 *s4 = reinterpret_cast<uint4 *>(s);
        if (TO_GLOBAL) {
            for (int i = tid; i < (words >> 2); i += THREADS) g4[i] = s4[i];
        } else {
            const uint32_t sa = (uint32_t)__cvta_generic_to_shared(s4);
            for (int i = tid; i < (words >> 2); i += THREADS)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa + 16u * i), "l"(g4 + i) : "memory");
        }
    } else {
        for (int i = tid; i < words; i += THREADS) {
            if (TO_GLOBAL) g[i] = s[i]; else s[i] = __ldg(g + i);
        }
    }
}
__device__ __forceinline__ void tile_copy_wait() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// AES-128-CTR over the staged private runs of a tile, by the whole group: every 16-byte counter block that overlaps a run
// is computed once, by one thread, whatever k is (a thread that followed its own block's words would compute 2-3 AES
// blocks per 8x8 block whenever 4 does not divide k + 1). Run c holds words [W0_c, W0_c + nw) of the image's private stream.
template <int C, int THREADS>
__device__ __forceinline__ void tile_aes_ctr(const DctParams &p, const T0Lane &sT, const TileCoord &T, uint32_t *s_priv, int RSP, int P, int tid) {
    uint32_t nonce[4];
    load_nonce(p, T.n, nonce);
    const int nw = T.nb * P;
    const int per = (TileShape<C>::TB * P + 3) / 4 + 1;   // >= counter blocks overlapping one run
    for (int idx = tid; idx < C * per; idx += THREADS) {
        const int c = idx / per, i = idx % per;
        const unsigned long long W0 = ((unsigned long long)(c * p.nbr + T.br) * p.nbc + T.bc0) * P;
        const unsigned long long blk = (W0 >> 2) + i;
        const long long first = (long long)(blk << 2) - (long long)W0;   // run-relative index of the block's first word
        if (first >= nw) continue;
        uint32_t ks[4];
        ctr_block(nonce, blk, ks);
        aes128_encrypt(sT, p.rk, ks);
        uint32_t *run = s_priv + c * RSP;
        if (first >= 0 && first + 4 <= nw) {
            uint4 *q = reinterpret_cast<uint4 *>(run + first);   // first is a multiple of 4 here iff W0 is: else fall through
            if ((first & 3) == 0) {
                uint4 x = *q;
                x.x ^= ks[0]; x.y ^= ks[1]; x.z ^= ks[2]; x.w ^= ks[3];
                *q = x;
                continue;
            }
        }
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const long long r = first + w;
            if (r >= 0 && r < nw) run[r] ^= ks[w];
        }
    }
}

// Stage layout (words): [AES tables 1024][public: C runs of TB*Q, tile_run_stride apart][private: C runs of TB*P likewise];
// every run starts 16-byte aligned.
template <int C, int V>
__global__ void __launch_bounds__(TileShape<C>::CTA, 1) fragment_dct_tile_kernel(const __grid_constant__ DctParams p) {
    constexpr int THREADS = TileShape<C>::THREADS, TB = TileShape<C>::TB, GROUPS = TileShape<C>::GROUPS;
    extern __shared__ __align__(16) uint32_t smem[];
    load_t0_replicated(smem);
    T0Lane sT;
    sT.tab = reinterpret_cast<const char *>(smem);
    sT.lane4 = 4u * (threadIdx.x & 31);
    constexpr ZigzagTable ZZ = make_zigzag();
    const int k = p.k, P = k + 1, Q = 63 - k;
    const int RSQ = tile_run_stride(TB * Q), RSP = tile_run_stride(TB * P);
    const int gid = threadIdx.x / THREADS, tid = threadIdx.x % THREADS;
    uint32_t *s_pub = smem + T0_WORDS + gid * tile_group_words<C>(k), *s_priv = s_pub + C * RSQ;
    const int j = tid / C, ch = tid % C;
    const int tiles_per_row = (p.nbc + TB - 1) / TB;
    const unsigned total = (unsigned)p.n_images * p.nbr * tiles_per_row;
#pragma unroll 1
    for (unsigned t = blockIdx.x * GROUPS + gid; t < total; t += gridDim.x * GROUPS) {
        const TileCoord T = decode_tile<C>(p, t, tiles_per_row);
        const bool act = j < T.nb;
        uint32_t *my_pub = s_pub + ch * RSQ + j * Q - P;  // indexed by z
        uint32_t *my_priv = s_priv + ch * RSP + j * P;
        if (act) {
            float v[64];
            load_block<C>(p.images + (size_t)T.n * p.image_stride, p.w, 8 * T.br, 8 * (T.bc0 + j), ch, v);
            dct8x8(v);
#pragma unroll
            for (int g = 0; g < 64; g += V) {
                uint32_t x[V];
#pragma unroll
                for (int q = 0; q < V; ++q) x[q] = __float_as_uint(v[ZZ.pos[g + q]]);
                vec_store<V>(g < P ? my_priv + g : my_pub + g, x);
            }
            if (V == 4) {   // 4 | k + 1: the block's private words are whole counter blocks of their own -- encrypt them here
                uint32_t nonce[4];
                load_nonce(p, T.n, nonce);
                const unsigned long long w0 = ((unsigned long long)(ch * p.nbr + T.br) * p.nbc + T.bc0 + j) * P;
#pragma unroll 1
                for (int g = 0; g < P; g += 4) {
                    uint32_t ks[4];
                    ctr_block(nonce, (w0 + g) >> 2, ks);
                    aes128_encrypt(sT, p.rk, ks);
                    uint4 x = *reinterpret_cast<uint4 *>(my_priv + g);
                    x.x ^= ks[0]; x.y ^= ks[1]; x.z ^= ks[2]; x.w ^= ks[3];
                    *reinterpret_cast<uint4 *>(my_priv + g) = x;
                }
            }
        }
        group_sync(gid, THREADS);
#pragma unroll
        for (int c = 0; c < C; ++c) {   // the public runs leave first; their stores drain while the private runs are encrypted
            const size_t b0 = (size_t)(c * p.nbr + T.br) * p.nbc + T.bc0;
            tile_copy<true, THREADS>(reinterpret_cast<uint32_t *>(p.pub + (size_t)T.n * p.pub_stride) + b0 * Q, s_pub + c * RSQ, T.nb * Q, tid);
        }
        if (V != 4) {
            tile_aes_ctr<C, THREADS>(p, sT, T, s_priv, RSP, P, tid);
            group_sync(gid, THREADS);
        }
#pragma unroll
        for (int c = 0; c < C; ++c) {
            const size_t b0 = (size_t)(c * p.nbr + T.br) * p.nbc + T.bc0;
            tile_copy<true, THREADS>(reinterpret_cast<uint32_t *>(p.priv + (size_t)T.n * p.priv_stride) + b0 * P, s_priv + c * RSP, T.nb * P, tid);
        }
        group_sync(gid, THREADS);
    }
}

template <int C, int V>
__global__ void __launch_bounds__(TileShape<C>::CTA, 1) defragment_dct_tile_kernel(const __grid_constant__ DctParams p) {
    constexpr int THREADS = TileShape<C>::THREADS, TB = TileShape<C>::TB, GROUPS = TileShape<C>::GROUPS;
    extern __shared__ __align__(16) uint32_t smem[];
    load_t0_replicated(smem);
    T0Lane sT;
    sT.tab = reinterpret_cast<const char *>(smem);
    sT.lane4 = 4u * (threadIdx.x & 31);
    constexpr ZigzagTable ZZ = make_zigzag();
    const int k = p.k, P = k + 1, Q = 63 - k;
    const int RSQ = tile_run_stride(TB * Q), RSP = tile_run_stride(TB * P);
    const int gid = threadIdx.x / THREADS, tid = threadIdx.x % THREADS;
    uint32_t *s_pub = smem + T0_WORDS + gid * tile_group_words<C>(k), *s_priv = s_pub + C * RSQ;
    const int j = tid / C, ch = tid % C;
    const int tiles_per_row = (p.nbc + TB - 1) / TB;
    const unsigned total = (unsigned)p.n_images * p.nbr * tiles_per_row;
#pragma unroll 1
    for (unsigned t = blockIdx.x * GROUPS + gid; t < total; t += gridDim.x * GROUPS) {
        const TileCoord T = decode_tile<C>(p, t, tiles_per_row);
        const bool act = j < T.nb;
#pragma unroll
        for (int c = 0; c < C; ++c) {
            const size_t b0 = (size_t)(c * p.nbr + T.br) * p.nbc + T.bc0;
            tile_copy<false, THREADS>(reinterpret_cast<uint32_t *>(p.pub + (size_t)T.n * p.pub_stride) + b0 * Q, s_pub + c * RSQ, T.nb * Q, tid);
            tile_copy<false, THREADS>(reinterpret_cast<uint32_t *>(p.priv + (size_t)T.n * p.priv_stride) + b0 * P, s_priv + c * RSP, T.nb * P, tid);
        }
        tile_copy_wait();
        group_sync(gid, THREADS);
        if (V != 4) {
            tile_aes_ctr<C, THREADS>(p, sT, T, s_priv, RSP, P, tid);
            group_sync(gid, THREADS);
        }
        float v[64];
        if (act) {
            uint32_t *my_pub = s_pub + ch * RSQ + j * Q - P;  // indexed by z
            uint32_t *my_priv = s_priv + ch * RSP + j * P;
            if (V == 4) {   // decrypt this block's own counter blocks in place
                uint32_t nonce[4];
                load_nonce(p, T.n, nonce);
                const unsigned long long w0 = ((unsigned long long)(ch * p.nbr + T.br) * p.nbc + T.bc0 + j) * P;
#pragma unroll 1
                for (int g = 0; g < P; g += 4) {
                    uint32_t ks[4];
                    ctr_block(nonce, (w0 + g) >> 2, ks);
                    aes128_encrypt(sT, p.rk, ks);
                    uint4 x = *reinterpret_cast<uint4 *>(my_priv + g);
                    x.x ^= ks[0]; x.y ^= ks[1]; x.z ^= ks[2]; x.w ^= ks[3];
                    *reinterpret_cast<uint4 *>(my_priv + g) = x;
                }
            }
#pragma unroll
            for (int g = 0; g < 64; g += V) {
                uint32_t x[V];
                vec_load<V>(g < P ? my_priv + g : my_pub + g, x);
#pragma unroll
                for (int q = 0; q < V; ++q) v[ZZ.pos[g + q]] = __uint_as_float(x[q]);
            }
            idct8x8(v);
        }
        store_block<C>(p.images_out + (size_t)T.n * p.image_stride, p.w, 8 * T.br, 8 * (T.bc0 + j), ch, act, v);
        group_sync(gid, THREADS);
    }
}

// ------------------------------------------------------------------------------------------------------------
// Leaf digests of DCT fragments as they lie in memory, nothing else (the verification half of steps 6-8, and
// all of feds_verify_dct): one thread per (fragment, leaf), registers only, 28 warps per SM. A leaf's bytes are contiguous in its fragment (G consecutive blocks of one block row), so this is SHA-256
// of a word-aligned byte range; needs no key. Threads [0, total_leaves) take the public leaves (31 compressions at k = 3),
// the rest the private ones (3 compressions), so that the lanes of a warp walk chains of equal length.
// ------------------------------------------------------------------------------------------------------------
constexpr int LEAFHASH_THREADS = 128;
template <int C>
__global__ void __launch_bounds__(LEAFHASH_THREADS) dct_leaves_hash_kernel(const __grid_constant__ DctParams p) {
    const unsigned long long gid = (unsigned long long)blockIdx.x * LEAFHASH_THREADS + threadIdx.x;
    if (gid >= 2 * p.total_leaves) return;
    const bool priv = gid >= p.total_leaves;
    const LeafCoord L = decode_leaf<C>(p, priv ? gid - p.total_leaves : gid);
    const int W = priv ? p.priv_words : p.pub_words;   // words per block in this fragment
    if (W == 0) return;                           // k = 63 at the first level: the public fragment is empty, its root is written elsewhere
    const uint32_t *src = reinterpret_cast<const uint32_t *>(priv ? p.priv + (size_t)L.n * p.priv_stride : p.pub + (size_t)L.n * p.pub_stride) +
                          (size_t)L.b0 * W;
    const unsigned nwords = (unsigned)(L.nblk * W);
    const bool al16 = (reinterpret_cast<uintptr_t>(src) & 15u) == 0;
    uint32_t H[8], w[16], nx[16];
    sha256_init(H);
    const unsigned full = nwords >> 4, tail = nwords & 15u;
    auto fetch = [&](unsigned blk) {
        const uint32_t *q = src + 16 * (size_t)blk;
        if (al16) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const uint4 v = __ldg(reinterpret_cast<const uint4 *>(q) + i);
                nx[4 * i] = v.x; nx[4 * i + 1] = v.y; nx[4 * i + 2] = v.z; nx[4 * i + 3] = v.w;
            }
        } else {
#pragma unroll
            for (int i = 0; i < 16; ++i) nx[i] = __ldg(q + i);
        }
    };
    if (full > 0) fetch(0);
#pragma unroll 1
    for (unsigned i = 0; i < full; ++i) {
#pragma unroll
        for (int j = 0; j < 16; ++j) w[j] = bswap32(nx[j]);
        if (i + 1 < full) fetch(i + 1);
        sha256_compress_rolled_fma(H, w, p.one);
    }
    // tail words, the 0x80 marker and the bit length (FIPS 180-4 5.1.1); one more block when fewer than 3 words are free
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        uint32_t x = 0u;
        if ((unsigned)j < tail) x = bswap32(__ldg(src + 16 * (size_t)full + j));
        else if ((unsigned)j == tail) x = 0x80000000u;
        w[j] = x;
    }
    const unsigned long long bits = (unsigned long long)nwords * 32ull;
    if (tail > 13u) {
        sha256_compress_rolled_fma(H, w, p.one);
#pragma unroll
        for (int j = 0; j < 16; ++j) w[j] = 0u;
    }
    w[14] = (uint32_t)(bits >> 32); w[15] = (uint32_t)bits;
    sha256_compress_rolled_fma(H, w, p.one);
    store_digest(p.leaves + (((size_t)L.n * 2 + (priv ? 0 : 1)) * p.leaves_per_image + L.li) * 32, H);
}

// The same digests for SMALL inputs, where what counts is the latency of one leaf's chain of compressions and not throughput:
// one WARP per public leaf (sha256_warp_coop, feds_sha_coop.cuh: ~23 us for 31 compressions instead of ~60), the short private
// leaves one per thread behind them. The host takes this kernel while there are at most COOP_MAX_LEAVES public leaves: one
// cooperating warp per warp scheduler of the chip (more would share the ALU pipes: measured slower from two per scheduler on).
constexpr int COOP_WARPS = 4, COOP_STRIDE = 32;
constexpr unsigned COOP_MAX_LEAVES = 592;
constexpr size_t COOP_SMEM_BYTES = (size_t)COOP_WARPS * coop_ws_words<COOP_STRIDE>() * 4;
template <int C>
__global__ void __launch_bounds__(COOP_WARPS * 32) dct_leaves_hash_coop_kernel(const __grid_constant__ DctParams p) {
    extern __shared__ __align__(16) uint32_t coop_smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned long long wid = (unsigned long long)blockIdx.x * COOP_WARPS + warp;
    const int P = p.priv_words, Q = p.pub_words;
    if (wid < p.total_leaves) {   // a public leaf, by the whole warp
        if (Q == 0) return;
        const LeafCoord L = decode_leaf<C>(p, wid);
        const uint8_t *src = p.pub + (size_t)L.n * p.pub_stride + (size_t)L.b0 * Q * 4;
        uint32_t H[8];
        sha256_warp_coop<COOP_STRIDE>(src, (unsigned)(L.nblk * Q) * 4u, coop_smem + warp * coop_ws_words<COOP_STRIDE>(), lane, p.one, H);
        if (lane == 0) store_digest(p.leaves + (((size_t)L.n * 2 + 1) * p.leaves_per_image + L.li) * 32, H);
        return;
    }
    // 32 private leaves, one per lane
    const unsigned long long gid = (wid - p.total_leaves) * 32 + lane;
    if (gid >= p.total_leaves || P == 0) return;
    const LeafCoord L = decode_leaf<C>(p, gid);
    const uint32_t *src = reinterpret_cast<const uint32_t *>(p.priv + (size_t)L.n * p.priv_stride) + (size_t)L.b0 * P;
    const unsigned nwords = (unsigned)(L.nblk * P), nblocks = (nwords * 4u + 9u + 63u) / 64u;
    uint32_t H[8], w[16];
    sha256_init(H);
#pragma unroll 1
    for (unsigned i = 0; i < nblocks; ++i) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const unsigned idx = 16u * i + j;
            w[j] = idx < nwords ? bswap32(__ldg(src + idx)) : (idx == nwords ? 0x80000000u : 0u);
        }
        if (i == nblocks - 1) w[15] = nwords * 32u;
        sha256_compress_rolled_fma(H, w, p.one);
    }
    store_digest(p.leaves + (((size_t)L.n * 2 + 0) * p.leaves_per_image + L.li) * 32, H);
}

}  // namespace feds
