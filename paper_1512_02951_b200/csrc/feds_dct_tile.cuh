// feds_dct_tile.cuh — the digest-free DCT path (FEDS_FLAG_NO_DIGEST; defragment without expected digests): steps 1-4
// and 6-8 of SURVEY.md 8(a) with no SHA-256, i.e. the report's own selective encryption (DCT + select + AES, P:488-494,
// P:607), which is bound by HBM and not by the integer pipe. Shaped for bandwidth instead of for a serial hash:
//
//   A CTA owns a tile of TB consecutive 8x8 blocks of one block row, all C channels; thread (j, ch) transforms one block
//   in 64 registers. The fragments of the tile are staged in shared memory in exactly their global byte order (the public
//   runs of consecutive blocks of one channel are contiguous), so the traffic with HBM is a flat,
//   fully coalesced 128-bit copy in both directions; AES-128-CTR is applied to the private words on their way through.
//   CTAs are persistent (the AES tables are filled once) and several share an SM, which overlaps one tile's loads with
//   another's arithmetic and stores.
#pragma once
#include "feds_dct.cuh"

namespace feds {

template <int C> struct TileShape { static constexpr int THREADS = (C == 3) ? 96 : 128, TB = THREADS / C; };
// Words between the staged runs of two channels: the smallest count >= words that is 20 mod 32, so that the C lanes of one
// block column (adjacent lanes) and their neighbours land in different banks when they write their runs with 128-bit stores.
__host__ __device__ inline int tile_run_stride(int words) { return ((words + 11) / 32) * 32 + 20; }
template <int C> __host__ __device__ inline size_t tile_smem_bytes(int k) {
    return (size_t)(AES_TABLE_WORDS + C * (tile_run_stride(TileShape<C>::TB * (63 - k)) + tile_run_stride(TileShape<C>::TB * (k + 1)))) * 4;
}

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
__device__ __forceinline__ void tile_copy(uint32_t *g, uint32_t *s, int words) {
    if (((reinterpret_cast<uintptr_t>(g) & 15u) == 0) && ((words & 3) == 0)) {
        uint4 *g4 = reinterpret_cast<uint4 *>(g);
        uint4 *s4 = reinterpret_cast<uint4 *>(s);
        if (TO_GLOBAL) {
            for (int i = threadIdx.x; i < (words >> 2); i += THREADS) g4[i] = s4[i];
        } else {
            const uint32_t sa = (uint32_t)__cvta_generic_to_shared(s4);
            for (int i = threadIdx.x; i < (words >> 2); i += THREADS)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa + 16u * i), "l"(g4 + i) : "memory");
        }
    } else {
        for (int i = threadIdx.x; i < words; i += THREADS) {
            if (TO_GLOBAL) g[i] = s[i]; else s[i] = __ldg(g + i);
        }
    }
}
__device__ __forceinline__ void tile_copy_wait() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Stage layout (words): [AES tables 1024][public: C runs of TB*Q, tile_run_stride apart][private: C runs of TB*P likewise];
// every run starts 16-byte aligned.
template <int C, int V>
__global__ void __launch_bounds__(TileShape<C>::THREADS) fragment_dct_tile_kernel(const __grid_constant__ DctParams p) {
    constexpr int THREADS = TileShape<C>::THREADS, TB = TileShape<C>::TB;
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *sT = smem;
    load_aes_tables(sT);
    constexpr ZigzagTable ZZ = make_zigzag();
    const int k = p.k, P = k + 1, Q = 63 - k;
    const int RSQ = tile_run_stride(TB * Q), RSP = tile_run_stride(TB * P);
    uint32_t *s_pub = smem + AES_TABLE_WORDS, *s_priv = s_pub + C * RSQ;
    const int j = threadIdx.x / C, ch = threadIdx.x % C;
    const int tiles_per_row = (p.nbc + TB - 1) / TB;
    const unsigned total = (unsigned)p.n_images * p.nbr * tiles_per_row;
#pragma unroll 1
    for (unsigned t = blockIdx.x; t < total; t += gridDim.x) {
        const TileCoord T = decode_tile<C>(p, t, tiles_per_row);
        const bool act = j < T.nb;
        uint32_t *my_pub = s_pub + ch * RSQ + j * Q - P;  // indexed by z
        uint32_t *my_priv = s_priv + ch * RSP + j * P;
        if (act) {
            float v[64];
            load_block<C>(p.images + (size_t)T.n * p.image_stride, p.w, 8 * T.br, 8 * (T.bc0 + j), ch, v);
            dct8x8(v);
            uint32_t nonce[4];
            load_nonce(p, T.n, nonce);
            Keystream K;
            K.blk = ~0ull;
            const unsigned long long w0 = ((unsigned long long)(ch * p.nbr + T.br) * p.nbc + T.bc0 + j) * P;
#pragma unroll
            for (int g = 0; g < 64; g += V) {
                uint32_t x[V];
#pragma unroll
                for (int q = 0; q < V; ++q) x[q] = __float_as_uint(v[ZZ.pos[g + q]]);
                vec_store<V>(g < P ? my_priv + g : my_pub + g, x);
            }
#pragma unroll 1
            for (int g = 0; g < P; g += V) {   // AES-128-CTR on the private words, in place in the stage
                uint32_t ks[V], x[V];
                keystream_words<V>(K, sT, p.rk, nonce, w0 + g, ks);
                vec_load<V>(my_priv + g, x);
#pragma unroll
                for (int q = 0; q < V; ++q) x[q] ^= ks[q];
                vec_store<V>(my_priv + g, x);
            }
        }
        __syncthreads();
#pragma unroll
        for (int c = 0; c < C; ++c) {
            const size_t b0 = (size_t)(c * p.nbr + T.br) * p.nbc + T.bc0;
            tile_copy<true, THREADS>(reinterpret_cast<uint32_t *>(p.pub + (size_t)T.n * p.pub_stride) + b0 * Q, s_pub + c * RSQ, T.nb * Q);
            tile_copy<true, THREADS>(reinterpret_cast<uint32_t *>(p.priv + (size_t)T.n * p.priv_stride) + b0 * P, s_priv + c * RSP, T.nb * P);
        }
        __syncthreads();
    }
}

template <int C, int V>
__global__ void __launch_bounds__(TileShape<C>::THREADS) defragment_dct_tile_kernel(const __grid_constant__ DctParams p) {
    constexpr int THREADS = TileShape<C>::THREADS, TB = TileShape<C>::TB;
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *sT = smem;
    load_aes_tables(sT);
    constexpr ZigzagTable ZZ = make_zigzag();
    const int k = p.k, P = k + 1, Q = 63 - k;
    const int RSQ = tile_run_stride(TB * Q), RSP = tile_run_stride(TB * P);
    uint32_t *s_pub = smem + AES_TABLE_WORDS, *s_priv = s_pub + C * RSQ;
    const int j = threadIdx.x / C, ch = threadIdx.x % C;
    const int tiles_per_row = (p.nbc + TB - 1) / TB;
    const unsigned total = (unsigned)p.n_images * p.nbr * tiles_per_row;
#pragma unroll 1
    for (unsigned t = blockIdx.x; t < total; t += gridDim.x) {
        const TileCoord T = decode_tile<C>(p, t, tiles_per_row);
        const bool act = j < T.nb;
#pragma unroll
        for (int c = 0; c < C; ++c) {
            const size_t b0 = (size_t)(c * p.nbr + T.br) * p.nbc + T.bc0;
            tile_copy<false, THREADS>(reinterpret_cast<uint32_t *>(p.pub + (size_t)T.n * p.pub_stride) + b0 * Q, s_pub + c * RSQ, T.nb * Q);
            tile_copy<false, THREADS>(reinterpret_cast<uint32_t *>(p.priv + (size_t)T.n * p.priv_stride) + b0 * P, s_priv + c * RSP, T.nb * P);
        }
        tile_copy_wait();
        __syncthreads();
        float v[64];
        if (act) {
            uint32_t *my_pub = s_pub + ch * RSQ + j * Q - P;  // indexed by z
            uint32_t *my_priv = s_priv + ch * RSP + j * P;
            uint32_t nonce[4];
            load_nonce(p, T.n, nonce);
            Keystream K;
            K.blk = ~0ull;
            const unsigned long long w0 = ((unsigned long long)(ch * p.nbr + T.br) * p.nbc + T.bc0 + j) * P;
#pragma unroll 1
            for (int g = 0; g < P; g += V) {   // decrypt in place in the stage
                uint32_t ks[V], x[V];
                keystream_words<V>(K, sT, p.rk, nonce, w0 + g, ks);
                vec_load<V>(my_priv + g, x);
#pragma unroll
                for (int q = 0; q < V; ++q) x[q] ^= ks[q];
                vec_store<V>(my_priv + g, x);
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
        __syncthreads();
    }
}

}  // namespace feds
