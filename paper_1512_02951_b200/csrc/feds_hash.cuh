// feds_hash.cuh — stream-level kernels shared by both transform paths: SHA-256 over fixed-size leaves of a byte
// stream (DWT path), the upper Merkle levels (2.1), AES-128-CTR over a byte stream, digest compare.
#pragma once
#include "feds_device.cuh"
#include "feds_dct.cuh"  // g_aes, load_aes_tables, store_digest
#include "feds_sha_coop.cuh"
#include "feds_aes_rep.cuh"

namespace feds {

constexpr int HASH_THREADS = 128;

// ------------------------------------------------------------------------------------------------------------
// Upper Merkle levels: node j of tree t = SHA-256(children [j*F, min((j+1)*F, n_in)) concatenated), 32 B each.
// Trees are (image, fragment) pairs laid out [tree][n][32]; the last level writes straight into the digest buffer.
// ------------------------------------------------------------------------------------------------------------
struct MerkleLevelParams {
    const uint8_t *in;
    uint8_t *out;
    unsigned n_in, n_out;       // per tree
    unsigned n_trees;
    size_t in_tree_stride, out_tree_stride;  // bytes
    int odd_trees_only_if_nonempty;  // 1: skip odd trees (public fragments) because they are empty (k = 63)
    uint32_t one;                    // = 1, opaque to the compiler (sha256_compress_rolled_fma)
    // merkle_tail_kernel only: an optional second family of n_trees2 trees of another shape, reduced by CTAs n_trees ..
    // n_trees + n_trees2 - 1 (DWT: the private and the public trees finish in one launch)
    const uint8_t *in2;
    uint8_t *out2;
    unsigned n_in2, n_trees2;
    size_t in2_tree_stride, out2_tree_stride;
    // merkle_top_kernel only: global scratch for the two levels under the root of each family ([tree][node][32] per level, the
    // level of <= 256 nodes first) and TOP_CTRL_WORDS zeroed arrival counters per tree (trees of family 2 after those of family 1)
    uint8_t *scratch, *scratch2;
    unsigned *ctrl;
};

// SHA-256 of `cnt` (1..16) concatenated 32-byte child digests at src (global memory via the read-only path, or shared).
template <bool GLOBAL, bool LATENCY = false>
__device__ __forceinline__ void hash_children(const uint4 *src, unsigned cnt, uint32_t (&H)[8], const uint32_t one) {
    sha256_init(H);
    const unsigned pairs = cnt >> 1;
    uint32_t w[16];
#pragma unroll 1
    for (unsigned i = 0; i <= pairs; ++i) {
        // block i holds children 2i, 2i+1; the last iteration holds the odd child (if any) and the padding
        if (i < pairs) {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const uint4 v = GLOBAL ? __ldg(src + 4 * i + q) : src[4 * i + q];
                w[4 * q] = bswap32(v.x); w[4 * q + 1] = bswap32(v.y); w[4 * q + 2] = bswap32(v.z); w[4 * q + 3] = bswap32(v.w);
            }
        } else {
#pragma unroll
            for (int q = 0; q < 16; ++q) w[q] = 0u;
            if (cnt & 1u) {
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    const uint4 v = GLOBAL ? __ldg(src + 4 * i + q) : src[4 * i + q];
                    w[4 * q] = bswap32(v.x); w[4 * q + 1] = bswap32(v.y); w[4 * q + 2] = bswap32(v.z); w[4 * q + 3] = bswap32(v.w);
                }
                w[8] = 0x80000000u;
            } else {
                w[0] = 0x80000000u;
            }
            w[15] = cnt * 256u;  // message bits = cnt * 32 bytes * 8
        }
        // LATENCY: a lone warp walks the chain, so the shortest dependency path wins (3-input adds, full unroll);
        // otherwise throughput wins (rolled loop, additions on the FMA pipe).
        if (LATENCY) sha256_compress(H, w); else sha256_compress_rolled_fma(H, w, one);
    }
}

__device__ __forceinline__ void digest_to_words(const uint32_t (&H)[8], uint4 &a, uint4 &b) {
    a = make_uint4(bswap32(H[0]), bswap32(H[1]), bswap32(H[2]), bswap32(H[3]));
    b = make_uint4(bswap32(H[4]), bswap32(H[5]), bswap32(H[6]), bswap32(H[7]));
}

__global__ void __launch_bounds__(HASH_THREADS) merkle_level_kernel(const __grid_constant__ MerkleLevelParams p) {
    const unsigned long long gid = (unsigned long long)blockIdx.x * HASH_THREADS + threadIdx.x;
    if (gid >= (unsigned long long)p.n_trees * p.n_out) return;
    const unsigned t = (unsigned)(gid / p.n_out), j = (unsigned)(gid % p.n_out);
    if (p.odd_trees_only_if_nonempty && (t & 1u)) return;
    const unsigned lo = j * FANOUT, hi = min(lo + FANOUT, p.n_in), cnt = hi - lo;
    const uint4 *src = reinterpret_cast<const uint4 *>(p.in + (size_t)t * p.in_tree_stride + (size_t)lo * 32);
    uint32_t H[8];
    hash_children<true>(src, cnt, H, p.one);
    store_digest(p.out + (size_t)t * p.out_tree_stride + (size_t)j * 32, H);
}

// The top of a tree in one launch: one CTA per tree reduces n_in <= 4096 digests to the root (up to three levels of
// fan-out 16: <= 256 nodes, <= 16 nodes, 1), intermediate levels in shared memory. The levels run one after the other on a
// nearly empty SM, so what counts is the length of the dependent chain: a level with more than TAIL_WARPS nodes is hashed one
// node per thread (nine dependent compressions, ~18 us), a level with at most TAIL_WARPS nodes one node per WARP, each warp on
// its own scheduler (sha256_warp_coop: the nine message schedules side by side, then 9 x 64 short rounds, ~6 us). More
// cooperating warps than schedulers would share the ALU pipes and lose again (measured: 32 warps, 47 us).
constexpr int TAIL_THREADS = 256, TAIL_WARPS = 4, TAIL_STRIDE = 16;   // TAIL_WARPS: one cooperating warp per warp scheduler; a node is at most 9 blocks
constexpr unsigned TAIL_MAX_IN = 256 * FANOUT;
constexpr size_t TAIL_SMEM_BYTES = (size_t)(256 * 2 + FANOUT * 2) * 16 + (size_t)TAIL_WARPS * coop_ws_words<TAIL_STRIDE>() * 4;
__global__ void __launch_bounds__(TAIL_THREADS) merkle_tail_kernel(const __grid_constant__ MerkleLevelParams p) {
    extern __shared__ __align__(16) uint4 tail_smem[];
    uint4 *sA = tail_smem, *sB = tail_smem + 256 * 2;
    uint32_t *ws = reinterpret_cast<uint32_t *>(sB + FANOUT * 2) + (threadIdx.x >> 5) * coop_ws_words<TAIL_STRIDE>();
    const unsigned t = blockIdx.x, tid = threadIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool extra = t >= p.n_trees;
    if (!extra && p.odd_trees_only_if_nonempty && (t & 1u)) return;
    const unsigned t2 = extra ? t - p.n_trees : 0u;
    uint4 *root = reinterpret_cast<uint4 *>(extra ? p.out2 + (size_t)t2 * p.out2_tree_stride : p.out + (size_t)t * p.out_tree_stride);
    // Level sources and sinks are generic pointers (global input, then the two shared buffers).
    const uint4 *src = reinterpret_cast<const uint4 *>(extra ? p.in2 + (size_t)t2 * p.in2_tree_stride : p.in + (size_t)t * p.in_tree_stride);
    unsigned n = extra ? p.n_in2 : p.n_in;
    uint4 *dst = sA;
#pragma unroll 1
    for (int level = 0; level < 3; ++level) {
        const unsigned m = (n + FANOUT - 1) / FANOUT;
        uint32_t H[8];
        bool mine = false;
        unsigned node = 0;
        if (m > (unsigned)TAIL_WARPS) {
            if (tid < m) {
                const unsigned lo = tid * FANOUT, cnt = min(lo + FANOUT, n) - lo;
                hash_children<false>(src + 2 * (size_t)lo, cnt, H, p.one);
                mine = true; node = tid;
            }
        } else if (warp < m) {
            const unsigned lo = warp * FANOUT, cnt = min(lo + FANOUT, n) - lo;
            sha256_warp_coop<TAIL_STRIDE>(reinterpret_cast<const uint8_t *>(src + 2 * (size_t)lo), cnt * 32u, ws, (int)lane, p.one, H);
            mine = lane == 0; node = warp;
        }
        if (mine) {
            uint4 a, b;
            digest_to_words(H, a, b);
            if (m == 1) { root[0] = a; root[1] = b; }
            else { dst[2 * node] = a; dst[2 * node + 1] = b; }
        }
        if (m == 1) return;
        __syncthreads();
        src = dst; dst = (dst == sA) ? sB : sA; n = m;
    }
}

// The same top of a tree spread over the chip, for calls with only a few trees (a single image): merkle_tail_kernel walks three
// levels on ONE SM -- 18 + 18 + 13 us of dependent compressions for the 4096 -> 256 -> 16 -> 1 top of a 134 MB stream. Here every
// node of every level is hashed by a cooperating warp (sha256_warp_coop, ~13 us for the nine blocks of a 16-child node: a lone
// warp sustains one round per ~45 cycles) and a CTA holds only four of them, one per warp scheduler: CTA c of a tree hashes nodes
// 4c .. 4c+3 of the first level into global scratch; the LAST of the (up to four) CTAs under one second-level node to finish -- an
// arrival counter per node, the threadfence + atomic ticket pattern -- hashes that node with its warp 0, and the last of those
// hashes the root. Three levels in 3 x 13 us (measured 44 us against 56), no grid-wide barrier, counters zeroed by a memset node in
// front of the launch.
constexpr int TOP_WARPS = 4, TOP_THREADS = TOP_WARPS * 32, TOP_CTRL_WORDS = 32, TOP_MAX_TREES = 8;   // TOP_CTRL_BYTES (feds_host.h) covers two trees
constexpr unsigned TOP_CTAS_PER_TREE = 256 / TOP_WARPS;
__global__ void __launch_bounds__(TOP_THREADS) merkle_top_kernel(const __grid_constant__ MerkleLevelParams p) {
    __shared__ __align__(16) uint32_t s_ws[TOP_WARPS * coop_ws_words<TAIL_STRIDE>()];
    __shared__ __align__(16) uint4 s_kids[2 * FANOUT];
    __shared__ unsigned s_ticket;
    const unsigned t = blockIdx.y, c = blockIdx.x, tid = threadIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool extra = t >= p.n_trees;
    if (!extra && p.odd_trees_only_if_nonempty && (t & 1u)) return;
    const unsigned t2 = extra ? t - p.n_trees : t;
    const unsigned n = extra ? p.n_in2 : p.n_in, m1 = (n + FANOUT - 1) / FANOUT, m2 = (m1 + FANOUT - 1) / FANOUT;
    if (c * TOP_WARPS >= m1) return;
    const unsigned trees = extra ? p.n_trees2 : p.n_trees;
    const uint8_t *src = extra ? p.in2 + (size_t)t2 * p.in2_tree_stride : p.in + (size_t)t2 * p.in_tree_stride;
    uint8_t *root = extra ? p.out2 + (size_t)t2 * p.out2_tree_stride : p.out + (size_t)t2 * p.out_tree_stride;
    uint8_t *sc = extra ? p.scratch2 : p.scratch;
    uint8_t *lvA = sc + (size_t)t2 * m1 * 32, *lvB = sc + (size_t)trees * m1 * 32 + (size_t)t2 * m2 * 32;
    unsigned *ctrl = p.ctrl + (size_t)t * TOP_CTRL_WORDS;
    uint32_t *ws = s_ws + warp * coop_ws_words<TAIL_STRIDE>();
    uint32_t H[8];
    const unsigned a = c * TOP_WARPS + warp;
    if (a < m1) {
        const unsigned lo = a * FANOUT, cnt = min(lo + FANOUT, n) - lo;
        sha256_warp_coop<TAIL_STRIDE>(src + (size_t)lo * 32, cnt * 32u, ws, (int)lane, p.one, H);
        if (lane == 0) { store_digest(m1 == 1 ? root : lvA + (size_t)a * 32, H); __threadfence(); }
    }
    if (m1 == 1) return;
    const unsigned b = c * TOP_WARPS / FANOUT;   // second-level node over this CTA's four nodes
    const unsigned kids = min(b * FANOUT + FANOUT, m1) - b * FANOUT;
    __syncthreads();
    if (tid == 0) { __threadfence(); s_ticket = atomicAdd(&ctrl[b], 1u); }
    __syncthreads();
    if (s_ticket != (kids + TOP_WARPS - 1) / TOP_WARPS - 1 || warp != 0) return;
    __threadfence();
    if (lane < 2 * kids) s_kids[lane] = __ldcg(reinterpret_cast<const uint4 *>(lvA + (size_t)b * FANOUT * 32) + lane);
    __syncwarp();
    sha256_warp_coop<TAIL_STRIDE>(reinterpret_cast<const uint8_t *>(s_kids), kids * 32u, ws, (int)lane, p.one, H);
    unsigned ticket = 0;
    if (lane == 0) {
        store_digest(m2 == 1 ? root : lvB + (size_t)b * 32, H);
        if (m2 > 1) { __threadfence(); ticket = atomicAdd(&ctrl[FANOUT], 1u); }
    }
    if (m2 == 1) return;
    ticket = __shfl_sync(0xffffffffu, ticket, 0);
    if (ticket != m2 - 1) return;
    __threadfence();
    __syncwarp();
    if (lane < 2 * m2) s_kids[lane] = __ldcg(reinterpret_cast<const uint4 *>(lvB) + lane);
    __syncwarp();
    sha256_warp_coop<TAIL_STRIDE>(reinterpret_cast<const uint8_t *>(s_kids), m2 * 32u, ws, (int)lane, p.one, H);
    if (lane == 0) store_digest(root, H);
}

// ------------------------------------------------------------------------------------------------------------
// Leaves of a byte stream: leaf j of stream t = SHA-256(bytes [j*LEAF, min((j+1)*LEAF, n))). One thread per leaf.
// Stream length is a multiple of 4 bytes here (int16 pairs are guaranteed by even subband widths: every band
// row has w>>l >= 1 elements but the whole fragment length is a multiple of 4 unless a band is 1 element wide;
// the generic byte tail below handles any length).
// ------------------------------------------------------------------------------------------------------------
struct StreamLeavesParams {
    const uint8_t *data[2];        // the two fragment streams (private, public) of image 0; hashed in one launch
    unsigned long long n_bytes[2]; // per image
    unsigned n_leaves[2];          // per image
    uint8_t *out[2];               // leaf digests [image][leaf][32] per stream
    size_t data_stride[2];         // bytes between consecutive images' streams
    unsigned n_images;
    uint32_t one;                  // = 1, opaque to the compiler (sha256_compress_rolled_fma)
};

// 64-thread CTAs: a fragment of tens of MB has only tens of thousands of leaves (well under one full wave of the chip), so
// small CTAs are what spreads them evenly over the SMs.
constexpr int LEAF_THREADS = 64;
__global__ void __launch_bounds__(LEAF_THREADS) stream_leaves_kernel(const __grid_constant__ StreamLeavesParams p) {
    const unsigned long long gid0 = (unsigned long long)blockIdx.x * LEAF_THREADS + threadIdx.x;
    const unsigned per_image = p.n_leaves[0] + p.n_leaves[1];
    if (gid0 >= (unsigned long long)per_image * p.n_images) return;
    const unsigned img = (unsigned)(gid0 / per_image), gid = (unsigned)(gid0 % per_image);
    const int f = gid >= p.n_leaves[0] ? 1 : 0;
    const unsigned j = f ? gid - p.n_leaves[0] : gid;
    const unsigned long long lo = (unsigned long long)j * DWT_LEAF_BYTES;
    const unsigned len = (unsigned)min((unsigned long long)DWT_LEAF_BYTES, p.n_bytes[f] - lo);
    const uint8_t *src = p.data[f] + (size_t)img * p.data_stride[f] + lo;
    uint32_t H[8];
    sha256_init(H);
    const unsigned full = len >> 6, tail = len & 63u;
    const unsigned nblocks = full + ((tail + 9 <= 64) ? 1u : 2u);
    uint32_t w[16];
    uint4 nx[4];  // the next 64-byte block is in flight while the current one is compressed
    if (full > 0) {
#pragma unroll
        for (int q = 0; q < 4; ++q) nx[q] = __ldg(reinterpret_cast<const uint4 *>(src) + q);
    }
#pragma unroll 1
    for (unsigned i = 0; i < nblocks; ++i) {
        if (i < full) {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                w[4 * q] = bswap32(nx[q].x); w[4 * q + 1] = bswap32(nx[q].y); w[4 * q + 2] = bswap32(nx[q].z); w[4 * q + 3] = bswap32(nx[q].w);
            }
            if (i + 1 < full) {
                const uint4 *s4 = reinterpret_cast<const uint4 *>(src + 64 * (size_t)(i + 1));
#pragma unroll
                for (int q = 0; q < 4; ++q) nx[q] = __ldg(s4 + q);
            }
        } else {
            // tail + padding, byte by byte (only the last leaf of a stream ever has a tail)
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                uint32_t word = 0;
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const unsigned pos = 64u * i + 4u * q + b;  // byte position within the leaf
                    uint32_t byte = 0;
                    if (pos < len) byte = src[pos];
                    else if (pos == len) byte = 0x80u;
                    word = (word << 8) | byte;
                }
                w[q] = word;
            }
            if (i == nblocks - 1) { w[14] = 0u; w[15] = len * 8u; }
        }
        sha256_compress_rolled_fma(H, w, p.one);
    }
    store_digest(p.out[f] + ((size_t)img * p.n_leaves[f] + j) * 32, H);
}

// The same leaves for SHORT streams (at most STREAM_COOP_MAX leaves in the launch): one warp per leaf, sha256_warp_coop.
constexpr int STREAM_COOP_WARPS = 4, STREAM_COOP_STRIDE = 32;
constexpr unsigned STREAM_COOP_MAX = 592;   // one warp per warp scheduler of the chip: more would share the ALU pipes and lose
constexpr size_t STREAM_COOP_SMEM_BYTES = (size_t)STREAM_COOP_WARPS * coop_ws_words<STREAM_COOP_STRIDE>() * 4;
__global__ void __launch_bounds__(STREAM_COOP_WARPS * 32) stream_leaves_coop_kernel(const __grid_constant__ StreamLeavesParams p) {
    extern __shared__ __align__(16) uint32_t coop_smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned long long gid0 = (unsigned long long)blockIdx.x * STREAM_COOP_WARPS + warp;
    const unsigned per_image = p.n_leaves[0] + p.n_leaves[1];
    if (gid0 >= (unsigned long long)per_image * p.n_images) return;
    const unsigned img = (unsigned)(gid0 / per_image), gid = (unsigned)(gid0 % per_image);
    const int f = gid >= p.n_leaves[0] ? 1 : 0;
    const unsigned j = f ? gid - p.n_leaves[0] : gid;
    const unsigned long long lo = (unsigned long long)j * DWT_LEAF_BYTES;
    const unsigned len = (unsigned)min((unsigned long long)DWT_LEAF_BYTES, p.n_bytes[f] - lo);
    uint32_t H[8];
    sha256_warp_coop<STREAM_COOP_STRIDE>(p.data[f] + (size_t)img * p.data_stride[f] + lo, len, coop_smem + warp * coop_ws_words<STREAM_COOP_STRIDE>(), lane,
                                         p.one, H);
    if (lane == 0) store_digest(p.out[f] + ((size_t)img * p.n_leaves[f] + j) * 32, H);
}

// ------------------------------------------------------------------------------------------------------------
// AES-128-CTR over a byte stream (A6): out = in XOR keystream, in place when out == in. Persistent CTAs,
// threads stride over the 16-byte blocks with 128-bit accesses. REPL = copies of each round-table entry in shared
// memory: 1 (4 KB; random lookups collide in the 32 banks, ~3.4 wavefronts each) for short streams, 32 (128 KB; lane l
// reads copy l, which lies in bank l: every lookup is one wavefront) for long ones, where the table fill is amortised.
// ------------------------------------------------------------------------------------------------------------
struct CtrParams {
    const uint8_t *in;
    uint8_t *out;
    unsigned long long n_bytes;       // per message
    size_t in_stride, out_stride;     // bytes between consecutive messages (batch); each message has its own counter from 0
    unsigned n_msgs;
    const uint8_t *d_nonces;          // device uint8[n_msgs][16], or nullptr: nonce_be for the single message
    uint32_t nonce_be[4];
    uint32_t rk[44];
    uint32_t c128;                    // = 128, opaque to the compiler (rep_lookup)
};
__device__ __forceinline__ void ctr_load_nonce(const CtrParams &p, unsigned m, uint32_t (&nonce)[4]) {
    if (p.d_nonces) {
        const uint4 q = __ldg(reinterpret_cast<const uint4 *>(p.d_nonces) + m);
        nonce[0] = bswap32(q.x); nonce[1] = bswap32(q.y); nonce[2] = bswap32(q.z); nonce[3] = bswap32(q.w);
    } else {
        nonce[0] = p.nonce_be[0]; nonce[1] = p.nonce_be[1]; nonce[2] = p.nonce_be[2]; nonce[3] = p.nonce_be[3];
    }
}
constexpr int AES_THREADS = 512;

template <int REPL>
struct ReplTable {
    const uint32_t *b;
    __device__ __forceinline__ uint32_t operator[](unsigned i) const { return b[i * REPL]; }
};

template <int REPL>
__global__ void __launch_bounds__(AES_THREADS) aes_ctr_stream_kernel(const __grid_constant__ CtrParams p) {
    extern __shared__ __align__(16) uint32_t sTab[];
    {
        const uint32_t *src = &g_aes.T[0][0];
        for (int i = threadIdx.x; i < AES_TABLE_WORDS * REPL; i += AES_THREADS) sTab[i] = src[i / REPL];
        __syncthreads();
    }
    ReplTable<REPL> T;
    T.b = sTab + (REPL > 1 ? (threadIdx.x & (REPL - 1)) : 0);
    RepAes A;
    A.base = (uint32_t)__cvta_generic_to_shared(sTab) + 4u * (threadIdx.x & 31);
    A.c128 = p.c128;
    const unsigned long long nfull = p.n_bytes >> 4;
    const unsigned long long stride = (unsigned long long)gridDim.x * AES_THREADS;
    const unsigned long long total = nfull * p.n_msgs;
    unsigned cur = 0xffffffffu;
    uint32_t nonce[4] = {0u, 0u, 0u, 0u};
    for (unsigned long long i = (unsigned long long)blockIdx.x * AES_THREADS + threadIdx.x; i < total; i += stride) {
        const unsigned m = p.n_msgs > 1 ? (unsigned)(i / nfull) : 0u;
        const unsigned long long blk = p.n_msgs > 1 ? i - (unsigned long long)m * nfull : i;
        if (m != cur) { ctr_load_nonce(p, m, nonce); cur = m; }
        uint4 v = __ldg(reinterpret_cast<const uint4 *>(p.in + (size_t)m * p.in_stride) + blk);
        uint32_t ks[4];
        ctr_block(nonce, blk, ks);
        if (REPL == 32) aes128_encrypt_rep32(A, p.rk, ks); else aes128_encrypt(T, p.rk, ks);
        v.x ^= ks[0]; v.y ^= ks[1]; v.z ^= ks[2]; v.w ^= ks[3];
        reinterpret_cast<uint4 *>(p.out + (size_t)m * p.out_stride)[blk] = v;
    }
    const unsigned rem = (unsigned)(p.n_bytes & 15u);
    if (rem && blockIdx.x == 0) {  // keystream of the partial last block of each message is truncated
        for (unsigned m = threadIdx.x; m < p.n_msgs; m += AES_THREADS) {
            uint32_t ks[4];
            ctr_load_nonce(p, m, nonce);
            ctr_block(nonce, nfull, ks);
            aes128_encrypt(T, p.rk, ks);
            const uint8_t *src = p.in + (size_t)m * p.in_stride + 16 * nfull;
            uint8_t *dst = p.out + (size_t)m * p.out_stride + 16 * nfull;
            for (unsigned b = 0; b < rem; ++b) dst[b] = src[b] ^ (uint8_t)(ks[b >> 2] >> (8 * (b & 3)));
        }
    }
}

// verify: flags[n] = bit0 (private root mismatch) | bit1 (public root mismatch); one thread per image
__global__ void compare_digests_kernel(const uint8_t *computed, const uint8_t *expected, uint32_t *flags, int n_images) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_images) return;
    const uint32_t *a = reinterpret_cast<const uint32_t *>(computed) + 16 * n;
    const uint32_t *b = reinterpret_cast<const uint32_t *>(expected) + 16 * n;
    uint32_t d0 = 0, d1 = 0;
    for (int i = 0; i < 8; ++i) { d0 |= a[i] ^ b[i]; d1 |= a[8 + i] ^ b[8 + i]; }
    flags[n] = (d0 ? 1u : 0u) | (d1 ? 2u : 0u);
}

// root of an empty fragment = SHA-256(""), written to digests[64 n + 32 .. 64 n + 63]
__global__ void write_empty_public_root_kernel(uint8_t *digests, int n_images) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_images) return;
    uint32_t H[8], w[16];
    sha256_init(H);
#pragma unroll
    for (int i = 0; i < 16; ++i) w[i] = 0u;
    w[0] = 0x80000000u;
    sha256_compress(H, w);
    store_digest(digests + 64 * (size_t)n + 32, H);
}

// SHA-256("") as the root of an empty stream
__global__ void write_empty_root_kernel(uint8_t *root) {
    if (threadIdx.x != 0) return;
    uint32_t H[8], w[16];
    sha256_init(H);
#pragma unroll
    for (int i = 0; i < 16; ++i) w[i] = 0u;
    w[0] = 0x80000000u;
    sha256_compress(H, w);
    store_digest(root, H);
}

}  // namespace feds
