// feds_api.cu — the C ABI of libfeds (include/feds.h): argument checks, workspace carving, key expansion, launches.
// Nothing here allocates, synchronises or keeps state across calls (one thread-local last-error slot aside).
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "../../include/feds.h"
#include "feds_dct.cuh"
#include "feds_dct_tile.cuh"
#include "feds_device.cuh"
#include "feds_dwt.cuh"
#include "feds_dwt_fast.cuh"
#include "feds_hash.cuh"

using namespace feds;

namespace {

thread_local int t_last_cuda_error = 0;
thread_local cudaEvent_t t_prof_start = nullptr, t_prof_stop = nullptr;
constexpr AesTables h_aes = make_aes_tables();
constexpr ZigzagTable h_zigzag = make_zigzag();

inline size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline bool misaligned(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

feds_status cuda_fail(cudaError_t e) {
    t_last_cuda_error = (int)e;
    return FEDS_ERR_CUDA;
}
#define FEDS_CUDA(call)                                   \
    do {                                                  \
        cudaError_t e__ = (call);                         \
        if (e__ != cudaSuccess) return cuda_fail(e__);    \
    } while (0)
#define FEDS_LAUNCH_CHECK() FEDS_CUDA(cudaGetLastError())

// SMs of the current device (the persistent DCT kernels launch one CTA per SM); asked per call, nothing is cached
int sm_count() {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) n = 148;
    return n;
}

bool dct_dims_ok(int w, int h) { return w > 0 && h > 0 && (w % 8) == 0 && (h % 8) == 0; }
bool chan_ok(int c) { return c == 1 || c == 3 || c == 4; }
bool dwt_dims_ok(int w, int h, int L) { return w > 0 && h > 0 && L >= 1 && L <= 6 && (w % (1 << L)) == 0 && (h % (1 << L)) == 0; }

// Merkle level sizes: n[0] = leaves, n[i+1] = ceil(n[i] / F) ... 1. Returns the number of levels (>= 1).
int tree_levels(unsigned leaves, unsigned n[40]) {
    int L = 0;
    n[L++] = leaves;
    while (n[L - 1] > 1) { n[L] = (n[L - 1] + FANOUT - 1) / FANOUT; ++L; }
    return L;
}
// bytes of digest storage for one tree, all levels with more than one node (the single-node level is the root)
size_t tree_bytes(unsigned leaves) {
    unsigned n[40];
    const int L = tree_levels(leaves, n);
    size_t b = 0;
    for (int i = 0; i < L; ++i) if (n[i] > 1) b += (size_t)n[i] * 32;
    return b;
}

unsigned dct_leaves(int w, int h, int c) { return (unsigned)c * (unsigned)(h / 8) * (unsigned)((w / 8 + G_BLOCKS - 1) / G_BLOCKS); }

void nonce_to_be(const uint8_t nonce[16], uint32_t out[4]) {
    for (int i = 0; i < 4; ++i)
        out[i] = ((uint32_t)nonce[4 * i] << 24) | ((uint32_t)nonce[4 * i + 1] << 16) | ((uint32_t)nonce[4 * i + 2] << 8) | nonce[4 * i + 3];
}

// Reduce level-0 digests [tree][n0][32] (tree stride = n0*32) to roots written at roots + tree*root_stride.
// `scratch` holds the intermediate levels. n_trees trees of identical shape.
// wide levels of n_trees equal trees: one thread per node until at most TAIL_MAX_IN digests per tree remain
feds_status reduce_wide(const uint8_t *&in, unsigned &n, unsigned n_trees, uint8_t *&sc, int skip_odd, cudaStream_t stream) {
    MerkleLevelParams mp{};
    mp.n_trees = n_trees;
    mp.odd_trees_only_if_nonempty = skip_odd;
    mp.one = 1u;
    while (n > TAIL_MAX_IN) {
        const unsigned m = (n + FANOUT - 1) / FANOUT;
        mp.in = in; mp.n_in = n; mp.n_out = m; mp.in_tree_stride = (size_t)n * 32;
        mp.out = sc; mp.out_tree_stride = (size_t)m * 32;
        const unsigned long long threads = (unsigned long long)n_trees * m;
        merkle_level_kernel<<<(unsigned)((threads + HASH_THREADS - 1) / HASH_THREADS), HASH_THREADS, 0, stream>>>(mp);
        FEDS_LAUNCH_CHECK();
        in = sc;
        sc += (size_t)n_trees * m * 32;
        n = m;
    }
    return FEDS_OK;
}

feds_status run_tree(const uint8_t *level0, unsigned n0, unsigned n_trees, uint8_t *scratch, uint8_t *roots, size_t root_stride,
                     int skip_odd, cudaStream_t stream) {
    const uint8_t *in = level0;
    uint8_t *sc = scratch;
    unsigned n = n0;
    feds_status st = reduce_wide(in, n, n_trees, sc, skip_odd, stream);
    if (st != FEDS_OK) return st;
    if (n > 1) {  // the top (<= 4096 digests per tree): one CTA per tree, up to three levels in one launch
        MerkleLevelParams mp{};
        mp.n_trees = n_trees; mp.odd_trees_only_if_nonempty = skip_odd; mp.one = 1u;
        mp.in = in; mp.n_in = n; mp.n_out = 1; mp.in_tree_stride = (size_t)n * 32;
        mp.out = roots; mp.out_tree_stride = root_stride;
        merkle_tail_kernel<<<n_trees, TAIL_THREADS, 0, stream>>>(mp);
        FEDS_LAUNCH_CHECK();
    }
    return FEDS_OK;
}

// two single trees of different shapes (DWT private / public): wide levels separately, both tops in one launch
feds_status run_two_trees(const uint8_t *l0a, unsigned na, uint8_t *sca, uint8_t *roota, const uint8_t *l0b, unsigned nb, uint8_t *scb,
                          uint8_t *rootb, cudaStream_t stream) {
    const uint8_t *ina = l0a, *inb = l0b;
    feds_status st = reduce_wide(ina, na, 1, sca, 0, stream);
    if (st != FEDS_OK) return st;
    st = reduce_wide(inb, nb, 1, scb, 0, stream);
    if (st != FEDS_OK) return st;
    if (na <= 1 && nb <= 1) return FEDS_OK;  // one-leaf trees: the leaf kernel already wrote the roots
    MerkleLevelParams mp{};
    mp.one = 1u; mp.n_out = 1;
    unsigned ctas = 0;
    if (na > 1) { mp.n_trees = 1; mp.in = ina; mp.n_in = na; mp.in_tree_stride = 0; mp.out = roota; mp.out_tree_stride = 0; ctas = 1; }
    if (nb > 1) {
        if (ctas == 0) { mp.n_trees = 1; mp.in = inb; mp.n_in = nb; mp.out = rootb; ctas = 1; }
        else { mp.in2 = inb; mp.n_in2 = nb; mp.out2 = rootb; ctas = 2; }
    }
    merkle_tail_kernel<<<ctas, TAIL_THREADS, 0, stream>>>(mp);
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

template <typename K>
feds_status set_smem(K kernel, size_t bytes) {
    FEDS_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return FEDS_OK;
}

struct DctPlan {
    unsigned nl;          // leaves per fragment per image
    size_t level0_bytes;  // per image: 2 * nl * 32 (0 when nl == 1: leaves are the roots)
    size_t upper_bytes;   // per image: intermediate levels, both fragments
    size_t per_image;     // workspace per image incl. 64 B for recomputed roots
};
DctPlan dct_plan(int w, int h, int c) {
    DctPlan pl;
    pl.nl = dct_leaves(w, h, c);
    pl.level0_bytes = pl.nl > 1 ? (size_t)2 * pl.nl * 32 : 0;
    pl.upper_bytes = pl.nl > 1 ? 2 * (tree_bytes(pl.nl) - (size_t)pl.nl * 32) : 0;
    pl.per_image = round_up(pl.level0_bytes + pl.upper_bytes + 64, 256);
    return pl;
}

feds_status check_dct_args(int n_images, int w, int h, int c, int k) {
    if (!dct_dims_ok(w, h)) return FEDS_ERR_BAD_DIMS;
    if (!chan_ok(c) || k < 0 || k > 63 || n_images < 1) return FEDS_ERR_BAD_PARAM;
    return FEDS_OK;
}

void fill_dct_params(DctParams &p, int n_images, int w, int h, int c, int k, const uint8_t key[16], const uint8_t *d_nonces,
                     const uint8_t *nonce_host, bool digest) {
    memset(&p, 0, sizeof p);
    p.n_images = n_images; p.w = w; p.h = h; p.k = k;
    p.nbr = h / 8; p.nbc = w / 8; p.nlr = (p.nbc + G_BLOCKS - 1) / G_BLOCKS;
    p.leaves_per_image = (unsigned)c * p.nbr * p.nlr;
    p.total_leaves = (unsigned long long)p.leaves_per_image * n_images;
    p.slot_stride = dct_slot_words(k);
    p.one = 1u;
    p.n_groups = (unsigned)((p.total_leaves + 31) / 32);
    (void)digest;
    p.d_nonces = d_nonces;
    if (nonce_host) nonce_to_be(nonce_host, p.nonce_be);
    aes128_expand_key_host(key, p.rk, h_aes);
}

template <template <int, int> class Launcher>
feds_status dispatch_cv(const DctParams &p, int c, cudaStream_t stream) {
    const int V = dct_vec_width(p.k);
#define FEDS_V(CC)                                                                  \
    (V == 4 ? Launcher<CC, 4>::go(p, stream) : V == 2 ? Launcher<CC, 2>::go(p, stream) : Launcher<CC, 1>::go(p, stream))
    return c == 1 ? FEDS_V(1) : c == 3 ? FEDS_V(3) : FEDS_V(4);
#undef FEDS_V
}

template <typename Kernel>
feds_status launch_dct(Kernel kernel, const DctParams &p, cudaStream_t stream, int max_threads = DCT_THREADS) {
    // persistent: one CTA per SM, its warps stride over the leaf groups. 16 warps unless their slots exceed the SM's
    // shared memory (k >= 32: the padding slack grows), then 8.
    int threads = max_threads;
    size_t smem = (size_t)(AES_TABLE_WORDS + threads * p.slot_stride) * 4;
    if (smem > DCT_SMEM_MAX) { threads = 256; smem = (size_t)(AES_TABLE_WORDS + threads * p.slot_stride) * 4; }
    const unsigned grid = std::min<unsigned>(p.n_groups, (unsigned)sm_count());
    feds_status s = set_smem(kernel, smem);
    if (s != FEDS_OK) return s;
    if (t_prof_start) FEDS_CUDA(cudaEventRecord(t_prof_start, stream));
    kernel<<<grid, threads, smem, stream>>>(p);
    if (t_prof_stop) FEDS_CUDA(cudaEventRecord(t_prof_stop, stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

// digest-free path: one persistent CTA per SM, GROUPS tile groups inside it (feds_dct_tile.cuh)
template <int C, typename Kernel>
feds_status launch_dct_tile(Kernel kernel, const DctParams &p, cudaStream_t stream, bool record_start = true) {
    constexpr int TB = TileShape<C>::TB, GROUPS = TileShape<C>::GROUPS;
    const size_t smem = tile_smem_bytes<C>(p.k);
    feds_status s = set_smem(kernel, smem);
    if (s != FEDS_OK) return s;
    const unsigned long long tiles = (unsigned long long)p.n_images * p.nbr * ((p.nbc + TB - 1) / TB);
    const unsigned grid = (unsigned)std::min<unsigned long long>((tiles + GROUPS - 1) / GROUPS, (unsigned long long)sm_count());
    if (t_prof_start && record_start) FEDS_CUDA(cudaEventRecord(t_prof_start, stream));
    kernel<<<grid, TileShape<C>::CTA, smem, stream>>>(p);
    if (t_prof_stop) FEDS_CUDA(cudaEventRecord(t_prof_stop, stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

// leaf digests of fragments as they lie in memory (feds_dct_tile.cuh): the verification half of a verified defragment
feds_status launch_leaves_hash(const DctParams &p, int c, cudaStream_t stream) {
    const unsigned long long threads = 2 * p.total_leaves;
    const unsigned grid = (unsigned)((threads + LEAFHASH_THREADS - 1) / LEAFHASH_THREADS);
    if (c == 1) dct_leaves_hash_kernel<1><<<grid, LEAFHASH_THREADS, 0, stream>>>(p);
    else if (c == 3) dct_leaves_hash_kernel<3><<<grid, LEAFHASH_THREADS, 0, stream>>>(p);
    else dct_leaves_hash_kernel<4><<<grid, LEAFHASH_THREADS, 0, stream>>>(p);
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

template <int C, int V> struct FragDigest { static feds_status go(const DctParams &p, cudaStream_t s) { return launch_dct(fragment_dct_kernel<C, V>, p, s); } };
template <int C, int V> struct FragPlain { static feds_status go(const DctParams &p, cudaStream_t s) { return launch_dct_tile<C>(fragment_dct_tile_kernel<C, V>, p, s); } };
template <int C, int V> struct DefragPlain { static feds_status go(const DctParams &p, cudaStream_t s) { return launch_dct_tile<C>(defragment_dct_tile_kernel<C, V>, p, s); } };
template <int C, int V> struct DefragAfterHash { static feds_status go(const DctParams &p, cudaStream_t s) { return launch_dct_tile<C>(defragment_dct_tile_kernel<C, V>, p, s, false); } };

feds_status launch_fragment_tile(const DctParams &p, int c, cudaStream_t stream) { return dispatch_cv<FragPlain>(p, c, stream); }
// the fused kernel exists for V = 4 and V = 2 only
feds_status launch_fragment_fused(const DctParams &p, int c, cudaStream_t stream) {
    const int V = dct_vec_width(p.k);
#define FEDS_V(CC) (V == 4 ? FragDigest<CC, 4>::go(p, stream) : FragDigest<CC, 2>::go(p, stream))
    return c == 1 ? FEDS_V(1) : c == 3 ? FEDS_V(3) : FEDS_V(4);
#undef FEDS_V
}
// Steps 1-5 in one fused kernel pay when its persistent grid is full (16 warps per SM for at least two rounds) and the runs
// are 8- or 16-byte multiples; otherwise the digest-free tile kernel followed by the leaf-hash kernel of what it wrote is
// faster (measured: 11 % at 512^2, 3 % at one 4096^2 image, 2-4 % for odd k + 1 at any size; 3 % slower at cfg3).
bool fragment_fused_pays(const DctParams &p) {
    if (dct_vec_width(p.k) == 1) return false;
    if (const char *force = getenv("FEDS_FRAGMENT_PATH")) {   // test hook: "fused" | "split"
        if (force[0] == 'f') return true;
        if (force[0] == 's') return false;
    }
    return p.n_groups >= 2u * (DCT_THREADS / 32) * (unsigned)sm_count();
}
feds_status launch_defragment(const DctParams &p, int c, cudaStream_t stream, bool after_hash = false) {
    return after_hash ? dispatch_cv<DefragAfterHash>(p, c, stream) : dispatch_cv<DefragPlain>(p, c, stream);
}

feds_status fragment_dct_impl(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c, int k,
                              const uint8_t key[16], const uint8_t *d_nonces, const uint8_t *nonce_host, uint8_t *d_private,
                              size_t private_stride, uint8_t *d_public, size_t public_stride, uint8_t *d_digests,
                              void *d_workspace, size_t workspace_bytes, unsigned flags, cudaStream_t stream) {
    feds_status st = check_dct_args(n_images, w, h, c, k);
    if (st != FEDS_OK) return st;
    if (flags & ~FEDS_FLAG_NO_DIGEST) return FEDS_ERR_BAD_PARAM;
    const bool digest = !(flags & FEDS_FLAG_NO_DIGEST);
    const size_t priv_b = feds_dct_private_bytes(w, h, c, k), pub_b = feds_dct_public_bytes(w, h, c, k);
    if (!d_images || !key || !d_private || (!d_public && pub_b) || (digest && (!d_digests || !d_workspace)) || (!d_nonces && !nonce_host))
        return FEDS_ERR_NULL_POINTER;
    if (image_stride < (size_t)w * h * c || private_stride < priv_b || public_stride < pub_b) return FEDS_ERR_BAD_PARAM;
    if (misaligned(d_images) || misaligned(d_private) || misaligned(d_public) || misaligned(d_digests) || misaligned(d_workspace) ||
        misaligned(d_nonces) || (n_images > 1 && ((image_stride | private_stride | public_stride) & 15u)))
        return FEDS_ERR_MISALIGNED;
    const DctPlan pl = dct_plan(w, h, c);
    if (digest && workspace_bytes < pl.per_image * (size_t)n_images) return FEDS_ERR_WORKSPACE_TOO_SMALL;

    DctParams p;
    fill_dct_params(p, n_images, w, h, c, k, key, d_nonces, nonce_host, digest);
    p.images = d_images; p.image_stride = image_stride;
    p.priv = d_private; p.priv_stride = private_stride;
    p.pub = d_public; p.pub_stride = public_stride;
    uint8_t *ws = static_cast<uint8_t *>(d_workspace);
    p.leaves = (pl.nl > 1) ? ws : d_digests;  // a one-leaf fragment's root is its leaf digest
    if (digest) {
        if (fragment_fused_pays(p)) {
            st = launch_fragment_fused(p, c, stream);
        } else {
            st = launch_fragment_tile(p, c, stream);   // records the profiling start; the stop follows the leaf hash
            if (st != FEDS_OK) return st;
            st = launch_leaves_hash(p, c, stream);
            if (t_prof_stop) FEDS_CUDA(cudaEventRecord(t_prof_stop, stream));
        }
        if (st != FEDS_OK) return st;
        if (pl.nl > 1) {
            st = run_tree(ws, pl.nl, 2u * n_images, ws + pl.level0_bytes * n_images, d_digests, 32, k == 63 ? 1 : 0, stream);
            if (st != FEDS_OK) return st;
        }
        if (k == 63) {
            write_empty_public_root_kernel<<<(n_images + 127) / 128, 128, 0, stream>>>(d_digests, n_images);
            FEDS_LAUNCH_CHECK();
        }
    } else {
        st = launch_fragment_tile(p, c, stream);
        if (st != FEDS_OK) return st;
    }
    return FEDS_OK;
}

// Verification workspace: [leaf digests][upper levels][n][64] recomputed roots (one-leaf fragments: the leaves ARE the roots)
uint8_t *verification_roots(const DctPlan &pl, int n_images, uint8_t *ws) { return ws + (pl.level0_bytes + pl.upper_bytes) * n_images; }
uint8_t *verification_leaves(const DctPlan &pl, int n_images, uint8_t *ws) { return (pl.nl > 1) ? ws : verification_roots(pl, n_images, ws); }
// leaf digests (already enqueued) -> roots -> flags[n] = bit0 private mismatch | bit1 public mismatch
feds_status finish_verification(const DctParams &p, const DctPlan &pl, int n_images, int k, uint8_t *ws, const uint8_t *d_expected,
                                uint32_t *d_flags, cudaStream_t stream) {
    (void)p;
    uint8_t *roots = verification_roots(pl, n_images, ws);
    if (pl.nl > 1) {
        const feds_status st = run_tree(ws, pl.nl, 2u * n_images, ws + pl.level0_bytes * n_images, roots, 32, k == 63 ? 1 : 0, stream);
        if (st != FEDS_OK) return st;
    }
    if (k == 63) {
        write_empty_public_root_kernel<<<(n_images + 127) / 128, 128, 0, stream>>>(roots, n_images);
        FEDS_LAUNCH_CHECK();
    }
    compare_digests_kernel<<<(n_images + 127) / 128, 128, 0, stream>>>(roots, d_expected, d_flags, n_images);
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

feds_status defragment_dct_impl(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                int n_images, int w, int h, int c, int k, const uint8_t key[16], const uint8_t *d_nonces,
                                const uint8_t *nonce_host, const uint8_t *d_expected, uint8_t *d_images_out, size_t image_stride,
                                uint32_t *d_flags, void *d_workspace, size_t workspace_bytes, unsigned flags, cudaStream_t stream) {
    feds_status st = check_dct_args(n_images, w, h, c, k);
    if (st != FEDS_OK) return st;
    if (flags & ~FEDS_FLAG_NO_DIGEST) return FEDS_ERR_BAD_PARAM;
    const bool verify = d_expected != nullptr && !(flags & FEDS_FLAG_NO_DIGEST);
    const size_t priv_b = feds_dct_private_bytes(w, h, c, k), pub_b = feds_dct_public_bytes(w, h, c, k);
    if (!d_private || (!d_public && pub_b) || !key || !d_images_out || (!d_nonces && !nonce_host) || (verify && (!d_flags || !d_workspace)))
        return FEDS_ERR_NULL_POINTER;
    if (image_stride < (size_t)w * h * c || private_stride < priv_b || public_stride < pub_b) return FEDS_ERR_BAD_PARAM;
    if (misaligned(d_images_out) || misaligned(d_private) || misaligned(d_public) || misaligned(d_expected) || misaligned(d_workspace) ||
        misaligned(d_nonces) || (n_images > 1 && ((image_stride | private_stride | public_stride) & 15u)))
        return FEDS_ERR_MISALIGNED;
    const DctPlan pl = dct_plan(w, h, c);
    if (verify && workspace_bytes < pl.per_image * (size_t)n_images) return FEDS_ERR_WORKSPACE_TOO_SMALL;

    DctParams p;
    fill_dct_params(p, n_images, w, h, c, k, key, d_nonces, nonce_host, verify);
    p.images_out = d_images_out; p.image_stride = image_stride;
    p.priv = const_cast<uint8_t *>(d_private); p.priv_stride = private_stride;
    p.pub = const_cast<uint8_t *>(d_public); p.pub_stride = public_stride;
    if (verify) {
        p.leaves = verification_leaves(pl, n_images, static_cast<uint8_t *>(d_workspace));
        // Verification and reconstruction are independent readers of the fragments: the leaf digests come from a
        // registers-only hash kernel (28 warps per SM, 0.89 of the ALU roofline), the pixels from the digest-free tile kernel.
        // Measured against one fused kernel doing both per leaf (round 1: 9.68 ms at cfg3): 9.21 ms, and 5-13 % faster for
        // every k whose runs are not 16-byte multiples.
        if (t_prof_start) FEDS_CUDA(cudaEventRecord(t_prof_start, stream));
        st = launch_leaves_hash(p, c, stream);
        if (st != FEDS_OK) return st;
        st = launch_defragment(p, c, stream, true);
        if (st != FEDS_OK) return st;
        return finish_verification(p, pl, n_images, k, static_cast<uint8_t *>(d_workspace), d_expected, d_flags, stream);
    }
    return launch_defragment(p, c, stream);
}

// verification alone: what a holder of the fragments can do without the key (A8)
feds_status verify_dct_impl(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride, int n_images,
                            int w, int h, int c, int k, const uint8_t *d_expected, uint32_t *d_flags, void *d_workspace,
                            size_t workspace_bytes, cudaStream_t stream) {
    feds_status st = check_dct_args(n_images, w, h, c, k);
    if (st != FEDS_OK) return st;
    const size_t priv_b = feds_dct_private_bytes(w, h, c, k), pub_b = feds_dct_public_bytes(w, h, c, k);
    if (!d_private || (!d_public && pub_b) || !d_expected || !d_flags || !d_workspace) return FEDS_ERR_NULL_POINTER;
    if (private_stride < priv_b || public_stride < pub_b) return FEDS_ERR_BAD_PARAM;
    if (misaligned(d_private) || misaligned(d_public) || misaligned(d_expected) || misaligned(d_workspace) ||
        (n_images > 1 && ((private_stride | public_stride) & 15u)))
        return FEDS_ERR_MISALIGNED;
    const DctPlan pl = dct_plan(w, h, c);
    if (workspace_bytes < pl.per_image * (size_t)n_images) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    DctParams p;
    static const uint8_t no_key[16] = {0};
    fill_dct_params(p, n_images, w, h, c, k, no_key, nullptr, no_key, true);
    p.priv = const_cast<uint8_t *>(d_private); p.priv_stride = private_stride;
    p.pub = const_cast<uint8_t *>(d_public); p.pub_stride = public_stride;
    p.leaves = verification_leaves(pl, n_images, static_cast<uint8_t *>(d_workspace));
    if (t_prof_start) FEDS_CUDA(cudaEventRecord(t_prof_start, stream));
    st = launch_leaves_hash(p, c, stream);
    if (t_prof_stop) FEDS_CUDA(cudaEventRecord(t_prof_stop, stream));
    if (st != FEDS_OK) return st;
    return finish_verification(p, pl, n_images, k, static_cast<uint8_t *>(d_workspace), d_expected, d_flags, stream);
}

// ---------------------------------------------------------------------------------------------- DWT plan
struct DwtPlan {
    size_t priv_b, pub_b;
    unsigned priv_nl, pub_nl;
    size_t planes_bytes;       // LL_1 .. LL_L planes (forward uses 1..L-1; inverse uses L (decrypted copy) .. 1)
    size_t plane_off[8];       // byte offset of the LL_l planes block, l = 1..L
    size_t priv_tree, pub_tree;  // bytes: all levels with > 1 node
    size_t per_image;
};
DwtPlan dwt_plan(int w, int h, int c, int L) {
    DwtPlan pl{};
    pl.priv_b = feds_dwt_private_bytes(w, h, c, L);
    pl.pub_b = feds_dwt_public_bytes(w, h, c, L);
    pl.priv_nl = (unsigned)((pl.priv_b + DWT_LEAF_BYTES - 1) / DWT_LEAF_BYTES);
    pl.pub_nl = (unsigned)((pl.pub_b + DWT_LEAF_BYTES - 1) / DWT_LEAF_BYTES);
    size_t off = 0;
    for (int l = 1; l <= L; ++l) {
        pl.plane_off[l] = off;
        off += round_up((size_t)c * (w >> l) * (h >> l) * 2, 256);
    }
    pl.planes_bytes = off;
    pl.priv_tree = tree_bytes(pl.priv_nl);
    pl.pub_tree = tree_bytes(pl.pub_nl);
    pl.per_image = round_up(pl.planes_bytes + round_up(pl.priv_tree, 256) + round_up(pl.pub_tree, 256) + 64, 256);
    return pl;
}

size_t dwt_level_off_elems(int w, int h, int L, int l) {  // elements before level l's bands inside one channel's public run
    size_t off = 0;
    for (int m = L; m > l; --m) off += (size_t)3 * (w >> m) * (h >> m);
    return off;
}

// Which level kernel: the register-streaming ones (feds_dwt_fast.cuh) need whole per-thread runs and aligned vector
// accesses; returns the pixels per thread (16: planar int16 or gray uint8; 8: interleaved RGB uint8) or 0 = tiled kernel.
int dwt_fast_px(const DwtLevelParams &p, bool u8, int c_img) {
    if (getenv("FEDS_DWT_TILED")) return 0;
    const int px = u8 ? (c_img == 1 ? 16 : c_img == 3 ? 8 : 0) : 16;
    if (px == 0 || p.cw % px != 0 || (p.ch & 1)) return 0;
    const size_t a = (size_t)px / 2;  // subband elements per thread and row: every offset must be a multiple of it
    if (p.level_off % a || (c_img > 1 && (p.pub_chan_stride % a || p.ll_band_chan_stride % a))) return 0;
    if ((reinterpret_cast<uintptr_t>(p.ll_band) | reinterpret_cast<uintptr_t>(p.pub)) & 15u) return 0;
    if (u8) { if (p.img_w % (c_img == 1 ? 16 : 8)) return 0; }
    return px;
}
// picks the rows per warp tile (p.rows) so that the launch has at least ~12 warps per SM, and returns the grid
dim3 dwt_fast_grid(DwtLevelParams &p, int px, int planes) {
    const int runs = p.cw / px, bh = p.ch >> 1;
    const unsigned strips = (unsigned)((runs + DWTF_LANES_OUT - 1) / DWTF_LANES_OUT);
    const unsigned long long want = 12ull * (unsigned)sm_count();
    int rows = DWTF_ROWS;
    while (rows > 4 && (unsigned long long)strips * planes * ((bh + rows - 1) / rows) < want) rows /= 2;
    p.rows = rows;
    return dim3(strips, (unsigned)((bh + DWTF_WARPS * rows - 1) / (DWTF_WARPS * rows)), planes);
}

// AES-128-CTR of a byte stream: the conflict-free 128 KB table layout pays once the stream is a few MB long
feds_status launch_aes_ctr(const uint8_t *d_in, uint8_t *d_out, size_t n_bytes, const uint8_t key[16], const uint8_t nonce[16],
                           cudaStream_t stream) {
    if (n_bytes == 0) return FEDS_OK;
    CtrParams cp{};
    cp.in = d_in; cp.out = d_out; cp.n_bytes = n_bytes;
    nonce_to_be(nonce, cp.nonce_be);
    aes128_expand_key_host(key, cp.rk, h_aes);
    const unsigned long long nblk = (n_bytes + 15) / 16;
    const unsigned sms = (unsigned)sm_count();
    if (n_bytes >= ((size_t)4 << 20)) {
        const size_t smem = (size_t)AES_TABLE_WORDS * 32 * 4;
        feds_status st = set_smem(aes_ctr_stream_kernel<32>, smem);
        if (st != FEDS_OK) return st;
        aes_ctr_stream_kernel<32><<<sms, AES_THREADS, smem, stream>>>(cp);
    } else {
        const unsigned want = (unsigned)((nblk + AES_THREADS - 1) / AES_THREADS);
        aes_ctr_stream_kernel<1><<<std::min(want, 2 * sms), AES_THREADS, (size_t)AES_TABLE_WORDS * 4, stream>>>(cp);
    }
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

feds_status dwt_digests(const uint8_t *d_private, const uint8_t *d_public, const DwtPlan &pl, uint8_t *tree_ws, uint8_t *roots,
                        cudaStream_t stream) {
    const unsigned nls[2] = {pl.priv_nl, pl.pub_nl};
    uint8_t *ws[2] = {tree_ws, tree_ws + round_up(pl.priv_tree, 256)};
    StreamLeavesParams sp;
    sp.data[0] = d_private; sp.data[1] = d_public;
    sp.n_bytes[0] = pl.priv_b; sp.n_bytes[1] = pl.pub_b;
    sp.one = 1u;
    for (int f = 0; f < 2; ++f) {
        sp.n_leaves[f] = nls[f];
        sp.out[f] = nls[f] > 1 ? ws[f] : roots + 32 * f;  // a one-leaf fragment's root is its leaf digest
    }
    const unsigned total = nls[0] + nls[1];
    if (t_prof_start) FEDS_CUDA(cudaEventRecord(t_prof_start, stream));
    stream_leaves_kernel<<<(total + LEAF_THREADS - 1) / LEAF_THREADS, LEAF_THREADS, 0, stream>>>(sp);
    if (t_prof_stop) FEDS_CUDA(cudaEventRecord(t_prof_stop, stream));
    FEDS_LAUNCH_CHECK();
    return run_two_trees(ws[0], nls[0], ws[0] + (size_t)nls[0] * 32, roots, ws[1], nls[1], ws[1] + (size_t)nls[1] * 32, roots + 32, stream);
}

}  // namespace

// =================================================================================================== C ABI
extern "C" {

const char *feds_status_string(feds_status s) {
    switch (s) {
        case FEDS_OK: return "ok";
        case FEDS_ERR_NULL_POINTER: return "null pointer";
        case FEDS_ERR_BAD_DIMS: return "bad dimensions";
        case FEDS_ERR_BAD_PARAM: return "bad parameter";
        case FEDS_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
        case FEDS_ERR_CUDA: return "CUDA error";
        case FEDS_ERR_MISALIGNED: return "pointer or stride not 16-byte aligned";
    }
    return "unknown status";
}
int feds_last_cuda_error(void) { return t_last_cuda_error; }

void feds_merkle_params(int *g_blocks, int *fanout, int *dwt_leaf_bytes) {
    if (g_blocks) *g_blocks = G_BLOCKS;
    if (fanout) *fanout = FANOUT;
    if (dwt_leaf_bytes) *dwt_leaf_bytes = DWT_LEAF_BYTES;
}

size_t feds_dct_private_bytes(int w, int h, int c, int k) {
    if (!dct_dims_ok(w, h) || !chan_ok(c) || k < 0 || k > 63) return 0;
    return (size_t)(w / 8) * (h / 8) * c * (k + 1) * 4;
}
size_t feds_dct_public_bytes(int w, int h, int c, int k) {
    if (!dct_dims_ok(w, h) || !chan_ok(c) || k < 0 || k > 63) return 0;
    return (size_t)(w / 8) * (h / 8) * c * (63 - k) * 4;
}
size_t feds_dwt_private_bytes(int w, int h, int c, int L) {
    if (!dwt_dims_ok(w, h, L) || !chan_ok(c)) return 0;
    return (size_t)(w >> L) * (h >> L) * c * 2;
}
size_t feds_dwt_public_bytes(int w, int h, int c, int L) {
    if (!dwt_dims_ok(w, h, L) || !chan_ok(c)) return 0;
    return ((size_t)w * h - (size_t)(w >> L) * (h >> L)) * c * 2;
}
size_t feds_workspace_bytes(int w, int h, int c, int k_or_levels, int is_dwt) {
    if (is_dwt) {
        if (!dwt_dims_ok(w, h, k_or_levels) || !chan_ok(c)) return 0;
        return dwt_plan(w, h, c, k_or_levels).per_image;
    }
    if (!dct_dims_ok(w, h) || !chan_ok(c) || k_or_levels < 0 || k_or_levels > 63) return 0;
    return dct_plan(w, h, c).per_image;
}

feds_status feds_fragment_dct(const uint8_t *d_image, int w, int h, int c, int k, const uint8_t key[16], const uint8_t nonce[16],
                              uint8_t *d_private, uint8_t *d_public, uint8_t *d_digests, void *d_workspace, size_t workspace_bytes,
                              feds_stream_t stream) {
    if (!nonce) return FEDS_ERR_NULL_POINTER;
    return fragment_dct_impl(d_image, 1, (size_t)(w > 0 ? w : 0) * (h > 0 ? h : 0) * (c > 0 ? c : 0), w, h, c, k, key, nullptr, nonce,
                             d_private, feds_dct_private_bytes(w, h, c, k), d_public, feds_dct_public_bytes(w, h, c, k), d_digests,
                             d_workspace, workspace_bytes, FEDS_FLAG_NONE, stream);
}

feds_status feds_fragment_dct_batch(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c, int k,
                                    const uint8_t key[16], const uint8_t *d_nonces, uint8_t *d_private, size_t private_stride,
                                    uint8_t *d_public, size_t public_stride, uint8_t *d_digests, void *d_workspace,
                                    size_t workspace_bytes, unsigned flags, feds_stream_t stream) {
    if (!d_nonces) return FEDS_ERR_NULL_POINTER;
    return fragment_dct_impl(d_images, n_images, image_stride, w, h, c, k, key, d_nonces, nullptr, d_private, private_stride, d_public,
                             public_stride, d_digests, d_workspace, workspace_bytes, flags, stream);
}

feds_status feds_defragment_dct(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int k, const uint8_t key[16],
                                const uint8_t nonce[16], const uint8_t *d_expected_digests, uint8_t *d_image_out,
                                uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes, feds_stream_t stream) {
    if (!nonce) return FEDS_ERR_NULL_POINTER;
    return defragment_dct_impl(d_private, feds_dct_private_bytes(w, h, c, k), d_public, feds_dct_public_bytes(w, h, c, k), 1, w, h, c, k,
                               key, nullptr, nonce, d_expected_digests, d_image_out,
                               (size_t)(w > 0 ? w : 0) * (h > 0 ? h : 0) * (c > 0 ? c : 0), d_verify_flags, d_workspace, workspace_bytes,
                               FEDS_FLAG_NONE, stream);
}

feds_status feds_defragment_dct_batch(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                      int n_images, int w, int h, int c, int k, const uint8_t key[16], const uint8_t *d_nonces,
                                      const uint8_t *d_expected_digests, uint8_t *d_images_out, size_t image_stride,
                                      uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes, unsigned flags,
                                      feds_stream_t stream) {
    if (!d_nonces) return FEDS_ERR_NULL_POINTER;
    return defragment_dct_impl(d_private, private_stride, d_public, public_stride, n_images, w, h, c, k, key, d_nonces, nullptr,
                               d_expected_digests, d_images_out, image_stride, d_verify_flags, d_workspace, workspace_bytes, flags,
                               stream);
}

feds_status feds_verify_dct(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int k,
                            const uint8_t *d_expected_digests, uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes,
                            feds_stream_t stream) {
    return verify_dct_impl(d_private, feds_dct_private_bytes(w, h, c, k), d_public, feds_dct_public_bytes(w, h, c, k), 1, w, h, c, k,
                           d_expected_digests, d_verify_flags, d_workspace, workspace_bytes, stream);
}

feds_status feds_verify_dct_batch(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                  int n_images, int w, int h, int c, int k, const uint8_t *d_expected_digests,
                                  uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes, feds_stream_t stream) {
    return verify_dct_impl(d_private, private_stride, d_public, public_stride, n_images, w, h, c, k, d_expected_digests, d_verify_flags,
                           d_workspace, workspace_bytes, stream);
}

// ------------------------------------------------------------------------------------------------ DWT
feds_status feds_fragment_dwt(const uint8_t *d_image, int w, int h, int c, int levels, const uint8_t key[16], const uint8_t nonce[16],
                              uint8_t *d_private, uint8_t *d_public, uint8_t *d_digests, void *d_workspace, size_t workspace_bytes,
                              feds_stream_t stream) {
    if (w <= 0 || h <= 0) return FEDS_ERR_BAD_DIMS;
    if (!chan_ok(c) || levels < 1 || levels > 6) return FEDS_ERR_BAD_PARAM;
    if (!dwt_dims_ok(w, h, levels)) return FEDS_ERR_BAD_DIMS;
    if (!d_image || !key || !nonce || !d_private || !d_public || !d_digests || !d_workspace) return FEDS_ERR_NULL_POINTER;
    if (misaligned(d_image) || misaligned(d_private) || misaligned(d_public) || misaligned(d_digests) || misaligned(d_workspace))
        return FEDS_ERR_MISALIGNED;
    const DwtPlan pl = dwt_plan(w, h, c, levels);
    if (workspace_bytes < pl.per_image) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    uint8_t *ws = static_cast<uint8_t *>(d_workspace);
    const int L = levels;

    for (int l = 1; l <= L; ++l) {
        DwtLevelParams p{};
        p.C = c; p.img_w = w; p.image_stride = (size_t)w * h * c;
        p.cw = w >> (l - 1); p.ch = h >> (l - 1);
        const int bw = w >> l, bh = h >> l;
        p.img_in = d_image;
        if (l > 1) { p.ll_in = reinterpret_cast<const int16_t *>(ws + pl.plane_off[l - 1]); p.ll_in_plane_stride = (size_t)p.cw * p.ch; }
        if (l < L) {
            p.ll_band = reinterpret_cast<int16_t *>(ws + pl.plane_off[l]);
            p.ll_band_image_stride = (size_t)c * bw * bh; p.ll_band_chan_stride = (size_t)bw * bh;
        } else {
            p.ll_band = reinterpret_cast<int16_t *>(d_private);
            p.ll_band_image_stride = pl.priv_b / 2; p.ll_band_chan_stride = (size_t)bw * bh;
        }
        p.pub = reinterpret_cast<int16_t *>(d_public);
        p.pub_image_stride = pl.pub_b / 2;
        p.pub_chan_stride = pl.pub_b / 2 / c;
        p.level_off = dwt_level_off_elems(w, h, L, l);
        const int px = dwt_fast_px(p, l == 1, c);
        const dim3 fgrid = px ? dwt_fast_grid(p, px, l == 1 ? 1 : c) : dim3();   // also sets p.rows
        if (px && l == 1 && c == 1) dwt_fwd_fast_kernel<1, 16, true><<<fgrid, DWTF_WARPS * 32, 0, stream>>>(p);
        else if (px && l == 1) dwt_fwd_fast_kernel<3, 8, true><<<fgrid, DWTF_WARPS * 32, 0, stream>>>(p);
        else if (px) dwt_fwd_fast_kernel<1, 16, false><<<fgrid, DWTF_WARPS * 32, 0, stream>>>(p);
        else {
            const dim3 grid((bw + DWT_TW - 1) / DWT_TW, (bh + DWT_TH - 1) / DWT_TH, c);
            if (l == 1) dwt_fwd_level_kernel<true><<<grid, DWT_THREADS, 0, stream>>>(p);
            else dwt_fwd_level_kernel<false><<<grid, DWT_THREADS, 0, stream>>>(p);
        }
        FEDS_LAUNCH_CHECK();
    }
    const feds_status st = launch_aes_ctr(d_private, d_private, pl.priv_b, key, nonce, stream);
    if (st != FEDS_OK) return st;
    return dwt_digests(d_private, d_public, pl, ws + pl.planes_bytes, d_digests, stream);
}

feds_status feds_defragment_dwt(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int levels,
                                const uint8_t key[16], const uint8_t nonce[16], const uint8_t *d_expected_digests,
                                uint8_t *d_image_out, uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes,
                                feds_stream_t stream) {
    if (w <= 0 || h <= 0) return FEDS_ERR_BAD_DIMS;
    if (!chan_ok(c) || levels < 1 || levels > 6) return FEDS_ERR_BAD_PARAM;
    if (!dwt_dims_ok(w, h, levels)) return FEDS_ERR_BAD_DIMS;
    if (!d_private || !d_public || !key || !nonce || !d_image_out || !d_workspace || (d_expected_digests && !d_verify_flags))
        return FEDS_ERR_NULL_POINTER;
    if (misaligned(d_image_out) || misaligned(d_private) || misaligned(d_public) || misaligned(d_expected_digests) || misaligned(d_workspace))
        return FEDS_ERR_MISALIGNED;
    const DwtPlan pl = dwt_plan(w, h, c, levels);
    if (workspace_bytes < pl.per_image) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    uint8_t *ws = static_cast<uint8_t *>(d_workspace);
    const int L = levels;

    if (d_expected_digests) {
        uint8_t *roots = ws + pl.per_image - 64;
        feds_status st = dwt_digests(d_private, d_public, pl, ws + pl.planes_bytes, roots, stream);
        if (st != FEDS_OK) return st;
        compare_digests_kernel<<<1, 32, 0, stream>>>(roots, d_expected_digests, d_verify_flags, 1);
        FEDS_LAUNCH_CHECK();
    }
    // decrypt LL_L into the level-L plane block (the received fragment stays untouched)
    uint8_t *lldec = ws + pl.plane_off[L];
    {
        const feds_status st = launch_aes_ctr(d_private, lldec, pl.priv_b, key, nonce, stream);
        if (st != FEDS_OK) return st;
    }

    for (int l = L; l >= 1; --l) {
        DwtLevelParams p{};
        p.C = c; p.img_w = w; p.image_stride = (size_t)w * h * c;
        p.cw = w >> (l - 1); p.ch = h >> (l - 1);
        const int bw = w >> l, bh = h >> l;
        p.ll_band = reinterpret_cast<int16_t *>(ws + pl.plane_off[l]);
        p.ll_band_image_stride = (size_t)c * bw * bh; p.ll_band_chan_stride = (size_t)bw * bh;
        p.pub = reinterpret_cast<int16_t *>(const_cast<uint8_t *>(d_public));
        p.pub_image_stride = pl.pub_b / 2;
        p.pub_chan_stride = pl.pub_b / 2 / c;
        p.level_off = dwt_level_off_elems(w, h, L, l);
        p.img_out = d_image_out;
        if (l > 1) { p.ll_out_plane = reinterpret_cast<int16_t *>(ws + pl.plane_off[l - 1]); p.ll_out_plane_stride = (size_t)p.cw * p.ch; }
        const int px = dwt_fast_px(p, l == 1, c);
        const dim3 fgrid = px ? dwt_fast_grid(p, px, l == 1 ? 1 : c) : dim3();   // also sets p.rows
        if (px && l == 1 && c == 1) dwt_inv_fast_kernel<1, 16, true><<<fgrid, DWTF_WARPS * 32, 0, stream>>>(p);
        else if (px && l == 1) dwt_inv_fast_kernel<3, 8, true><<<fgrid, DWTF_WARPS * 32, 0, stream>>>(p);
        else if (px) dwt_inv_fast_kernel<1, 16, false><<<fgrid, DWTF_WARPS * 32, 0, stream>>>(p);
        else {
            const dim3 grid((bw + DWT_TW - 1) / DWT_TW, (bh + DWT_TH - 1) / DWT_TH, c);
            if (l == 1) dwt_inv_level_kernel<true><<<grid, DWT_THREADS, 0, stream>>>(p);
            else dwt_inv_level_kernel<false><<<grid, DWT_THREADS, 0, stream>>>(p);
        }
        FEDS_LAUNCH_CHECK();
    }
    return FEDS_OK;
}

feds_status feds_verify_dwt(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int levels,
                            const uint8_t *d_expected_digests, uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes,
                            feds_stream_t stream) {
    if (w <= 0 || h <= 0) return FEDS_ERR_BAD_DIMS;
    if (!chan_ok(c) || levels < 1 || levels > 6) return FEDS_ERR_BAD_PARAM;
    if (!dwt_dims_ok(w, h, levels)) return FEDS_ERR_BAD_DIMS;
    if (!d_private || !d_public || !d_expected_digests || !d_verify_flags || !d_workspace) return FEDS_ERR_NULL_POINTER;
    if (misaligned(d_private) || misaligned(d_public) || misaligned(d_expected_digests) || misaligned(d_workspace)) return FEDS_ERR_MISALIGNED;
    const DwtPlan pl = dwt_plan(w, h, c, levels);
    if (workspace_bytes < pl.per_image) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    uint8_t *ws = static_cast<uint8_t *>(d_workspace);
    uint8_t *roots = ws + pl.per_image - 64;
    const feds_status st = dwt_digests(d_private, d_public, pl, ws + pl.planes_bytes, roots, stream);
    if (st != FEDS_OK) return st;
    compare_digests_kernel<<<1, 32, 0, stream>>>(roots, d_expected_digests, d_verify_flags, 1);
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

// ------------------------------------------------------------------------------------------------ stream primitives
feds_status feds_aes128_ctr(const uint8_t *d_in, uint8_t *d_out, size_t n_bytes, const uint8_t key[16], const uint8_t nonce[16],
                            feds_stream_t stream) {
    if (!key || !nonce || (n_bytes && (!d_in || !d_out))) return FEDS_ERR_NULL_POINTER;
    if (misaligned(d_in) || misaligned(d_out)) return FEDS_ERR_MISALIGNED;
    return launch_aes_ctr(d_in, d_out, n_bytes, key, nonce, stream);
}

size_t feds_sha256_merkle_workspace_bytes(size_t n_bytes) {
    const size_t nl = (n_bytes + DWT_LEAF_BYTES - 1) / DWT_LEAF_BYTES;
    if (nl > 0xffffffffull) return 0;
    return round_up(tree_bytes((unsigned)nl) + 32, 256);
}

feds_status feds_sha256_merkle(const uint8_t *d_data, size_t n_bytes, uint8_t *d_root, void *d_workspace, size_t workspace_bytes,
                               feds_stream_t stream) {
    if (!d_root || (n_bytes && !d_data)) return FEDS_ERR_NULL_POINTER;
    if (misaligned(d_data) || misaligned(d_root) || misaligned(d_workspace)) return FEDS_ERR_MISALIGNED;
    const size_t nl64 = (n_bytes + DWT_LEAF_BYTES - 1) / DWT_LEAF_BYTES;
    if (nl64 > 0xffffffffull) return FEDS_ERR_BAD_PARAM;
    const unsigned nl = (unsigned)nl64;
    if (nl > 1 && (!d_workspace || workspace_bytes < feds_sha256_merkle_workspace_bytes(n_bytes))) return d_workspace ? FEDS_ERR_WORKSPACE_TOO_SMALL : FEDS_ERR_NULL_POINTER;
    if (nl == 0) {  // SHA-256(""): the kernel writes it at digests + 32
        uint8_t *ws = static_cast<uint8_t *>(d_workspace);
        (void)ws;
        write_empty_root_kernel<<<1, 32, 0, stream>>>(d_root);
        FEDS_LAUNCH_CHECK();
        return FEDS_OK;
    }
    uint8_t *ws = static_cast<uint8_t *>(d_workspace);
    StreamLeavesParams sp{};
    sp.data[0] = d_data; sp.n_bytes[0] = n_bytes; sp.n_leaves[0] = nl;
    sp.out[0] = nl > 1 ? ws : d_root;
    sp.one = 1u;
    stream_leaves_kernel<<<(nl + LEAF_THREADS - 1) / LEAF_THREADS, LEAF_THREADS, 0, stream>>>(sp);
    FEDS_LAUNCH_CHECK();
    if (nl > 1) return run_tree(ws, nl, 1, ws + (size_t)nl * 32, d_root, 32, 0, stream);
    return FEDS_OK;
}

// ------------------------------------------------------------------------------------------------ host-staged batch
static size_t host_slot_bytes(int ipc, int w, int h, int c, int k) {
    const size_t img = round_up((size_t)ipc * w * h * c, 256), non = round_up((size_t)ipc * 16, 256);
    const size_t pv = round_up((size_t)ipc * feds_dct_private_bytes(w, h, c, k), 256);
    const size_t pb = round_up((size_t)ipc * feds_dct_public_bytes(w, h, c, k), 256);
    const size_t dg = round_up((size_t)ipc * 64, 256), wsb = round_up((size_t)ipc * feds_workspace_bytes(w, h, c, k, 0), 256);
    // + the verify flags of the defragment call: ONE slot size for both directions, so that stream j owns the same scratch
    // bytes in either call and the two may be interleaved on the same streams without synchronisation
    return img + non + pv + pb + dg + wsb + round_up((size_t)ipc * 4, 256);
}

size_t feds_fragment_dct_host_scratch_bytes(int images_per_chunk, int n_streams, int w, int h, int c, int k) {
    if (images_per_chunk < 1 || n_streams < 1 || check_dct_args(1, w, h, c, k) != FEDS_OK) return 0;
    return host_slot_bytes(images_per_chunk, w, h, c, k) * (size_t)n_streams;
}

feds_status feds_fragment_dct_host(const uint8_t *h_images, int n_images, int w, int h, int c, int k, const uint8_t key[16],
                                   const uint8_t *h_nonces, uint8_t *h_private, uint8_t *h_public, uint8_t *h_digests,
                                   int images_per_chunk, void *d_scratch, size_t scratch_bytes, feds_stream_t *streams, int n_streams,
                                   unsigned flags) {
    feds_status st = check_dct_args(n_images, w, h, c, k);
    if (st != FEDS_OK) return st;
    if (images_per_chunk < 1 || n_streams < 1 || (flags & ~FEDS_FLAG_NO_DIGEST)) return FEDS_ERR_BAD_PARAM;
    const bool digest = !(flags & FEDS_FLAG_NO_DIGEST);
    const size_t img_b = (size_t)w * h * c, priv_b = feds_dct_private_bytes(w, h, c, k), pub_b = feds_dct_public_bytes(w, h, c, k);
    if (!h_images || !key || !h_nonces || !h_private || (!h_public && pub_b) || (digest && !h_digests) || !d_scratch || !streams)
        return FEDS_ERR_NULL_POINTER;
    if (misaligned(d_scratch)) return FEDS_ERR_MISALIGNED;
    const int ipc = images_per_chunk;
    const size_t slot = host_slot_bytes(ipc, w, h, c, k);
    if (scratch_bytes < slot * (size_t)n_streams) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    const size_t ws_b = feds_workspace_bytes(w, h, c, k, 0);
    int chunk = 0;
    for (int i0 = 0; i0 < n_images; i0 += ipc, ++chunk) {
        const int m = (n_images - i0 < ipc) ? n_images - i0 : ipc;
        cudaStream_t s = streams[chunk % n_streams];
        uint8_t *base = static_cast<uint8_t *>(d_scratch) + slot * (size_t)(chunk % n_streams);
        uint8_t *d_img = base;
        uint8_t *d_non = d_img + round_up((size_t)ipc * img_b, 256);
        uint8_t *d_pv = d_non + round_up((size_t)ipc * 16, 256);
        uint8_t *d_pb = d_pv + round_up((size_t)ipc * priv_b, 256);
        uint8_t *d_dg = d_pb + round_up((size_t)ipc * pub_b, 256);
        uint8_t *d_ws = d_dg + round_up((size_t)ipc * 64, 256);
        FEDS_CUDA(cudaMemcpyAsync(d_img, h_images + (size_t)i0 * img_b, (size_t)m * img_b, cudaMemcpyHostToDevice, s));
        FEDS_CUDA(cudaMemcpyAsync(d_non, h_nonces + (size_t)i0 * 16, (size_t)m * 16, cudaMemcpyHostToDevice, s));
        st = fragment_dct_impl(d_img, m, img_b, w, h, c, k, key, d_non, nullptr, d_pv, priv_b, d_pb, pub_b, d_dg, d_ws, (size_t)ipc * ws_b,
                               flags, s);
        if (st != FEDS_OK) return st;
        FEDS_CUDA(cudaMemcpyAsync(h_private + (size_t)i0 * priv_b, d_pv, (size_t)m * priv_b, cudaMemcpyDeviceToHost, s));
        if (pub_b) FEDS_CUDA(cudaMemcpyAsync(h_public + (size_t)i0 * pub_b, d_pb, (size_t)m * pub_b, cudaMemcpyDeviceToHost, s));
        if (digest) FEDS_CUDA(cudaMemcpyAsync(h_digests + (size_t)i0 * 64, d_dg, (size_t)m * 64, cudaMemcpyDeviceToHost, s));
    }
    return FEDS_OK;
}

size_t feds_defragment_dct_host_scratch_bytes(int images_per_chunk, int n_streams, int w, int h, int c, int k) {
    if (images_per_chunk < 1 || n_streams < 1 || check_dct_args(1, w, h, c, k) != FEDS_OK) return 0;
    return host_slot_bytes(images_per_chunk, w, h, c, k) * (size_t)n_streams;
}

feds_status feds_defragment_dct_host(const uint8_t *h_private, const uint8_t *h_public, int n_images, int w, int h, int c, int k,
                                     const uint8_t key[16], const uint8_t *h_nonces, const uint8_t *h_expected_digests,
                                     uint8_t *h_images_out, uint32_t *h_verify_flags, int images_per_chunk, void *d_scratch,
                                     size_t scratch_bytes, feds_stream_t *streams, int n_streams, unsigned flags) {
    feds_status st = check_dct_args(n_images, w, h, c, k);
    if (st != FEDS_OK) return st;
    if (images_per_chunk < 1 || n_streams < 1 || (flags & ~FEDS_FLAG_NO_DIGEST)) return FEDS_ERR_BAD_PARAM;
    const bool verify = h_expected_digests != nullptr && !(flags & FEDS_FLAG_NO_DIGEST);
    const size_t img_b = (size_t)w * h * c, priv_b = feds_dct_private_bytes(w, h, c, k), pub_b = feds_dct_public_bytes(w, h, c, k);
    if (!h_private || (!h_public && pub_b) || !key || !h_nonces || !h_images_out || (verify && !h_verify_flags) || !d_scratch || !streams)
        return FEDS_ERR_NULL_POINTER;
    if (misaligned(d_scratch)) return FEDS_ERR_MISALIGNED;
    const int ipc = images_per_chunk;
    const size_t slot = host_slot_bytes(ipc, w, h, c, k);
    if (scratch_bytes < slot * (size_t)n_streams) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    const size_t ws_b = feds_workspace_bytes(w, h, c, k, 0);
    int chunk = 0;
    for (int i0 = 0; i0 < n_images; i0 += ipc, ++chunk) {
        const int m = (n_images - i0 < ipc) ? n_images - i0 : ipc;
        cudaStream_t s = streams[chunk % n_streams];
        uint8_t *base = static_cast<uint8_t *>(d_scratch) + slot * (size_t)(chunk % n_streams);
        uint8_t *d_img = base;
        uint8_t *d_non = d_img + round_up((size_t)ipc * img_b, 256);
        uint8_t *d_pv = d_non + round_up((size_t)ipc * 16, 256);
        uint8_t *d_pb = d_pv + round_up((size_t)ipc * priv_b, 256);
        uint8_t *d_dg = d_pb + round_up((size_t)ipc * pub_b, 256);
        uint8_t *d_ws = d_dg + round_up((size_t)ipc * 64, 256);
        uint32_t *d_fl = reinterpret_cast<uint32_t *>(d_ws + round_up((size_t)ipc * ws_b, 256));
        FEDS_CUDA(cudaMemcpyAsync(d_pv, h_private + (size_t)i0 * priv_b, (size_t)m * priv_b, cudaMemcpyHostToDevice, s));
        if (pub_b) FEDS_CUDA(cudaMemcpyAsync(d_pb, h_public + (size_t)i0 * pub_b, (size_t)m * pub_b, cudaMemcpyHostToDevice, s));
        FEDS_CUDA(cudaMemcpyAsync(d_non, h_nonces + (size_t)i0 * 16, (size_t)m * 16, cudaMemcpyHostToDevice, s));
        if (verify) FEDS_CUDA(cudaMemcpyAsync(d_dg, h_expected_digests + (size_t)i0 * 64, (size_t)m * 64, cudaMemcpyHostToDevice, s));
        st = defragment_dct_impl(d_pv, priv_b, d_pb, pub_b, m, w, h, c, k, key, d_non, nullptr, verify ? d_dg : nullptr, d_img, img_b, d_fl,
                                 d_ws, (size_t)ipc * ws_b, flags, s);
        if (st != FEDS_OK) return st;
        FEDS_CUDA(cudaMemcpyAsync(h_images_out + (size_t)i0 * img_b, d_img, (size_t)m * img_b, cudaMemcpyDeviceToHost, s));
        if (verify) FEDS_CUDA(cudaMemcpyAsync(h_verify_flags + i0, d_fl, (size_t)m * 4, cudaMemcpyDeviceToHost, s));
    }
    return FEDS_OK;
}

void feds_profile_events(void *ev_start, void *ev_stop) {
    t_prof_start = static_cast<cudaEvent_t>(ev_start);
    t_prof_stop = static_cast<cudaEvent_t>(ev_stop);
}

// ------------------------------------------------------------------------------------------------ host self-checks
void feds_debug_sha256_host(const uint8_t *msg, size_t n, uint8_t out[32]) {
    uint32_t H[8], w[16];
    sha256_init(H);
    const size_t full = n / 64, tail = n % 64;
    const size_t nblocks = full + ((tail + 9 <= 64) ? 1 : 2);
    for (size_t i = 0; i < nblocks; ++i) {
        uint8_t blk[64];
        for (int b = 0; b < 64; ++b) {
            const size_t pos = 64 * i + b;
            blk[b] = pos < n ? msg[pos] : (pos == n ? 0x80 : 0);
        }
        if (i == nblocks - 1) {
            const unsigned long long bits = (unsigned long long)n * 8;
            for (int b = 0; b < 8; ++b) blk[63 - b] = (uint8_t)(bits >> (8 * b));
        }
        for (int q = 0; q < 16; ++q) {
            uint32_t le;
            memcpy(&le, blk + 4 * q, 4);
            w[q] = bswap32(le);  // the kernels load little-endian words and byte-swap
        }
        sha256_compress(H, w);
    }
    for (int i = 0; i < 8; ++i) { const uint32_t v = bswap32(H[i]); memcpy(out + 4 * i, &v, 4); }
}

void feds_debug_aes128_host(const uint8_t key[16], const uint8_t in[16], uint8_t out[16]) {
    uint32_t rk[44], s[4];
    aes128_expand_key_host(key, rk, h_aes);
    memcpy(s, in, 16);
    aes128_encrypt(&h_aes.T[0][0], rk, s);
    memcpy(out, s, 16);
}

void feds_debug_dct8x8_host(const float in[64], float out[64], int inverse) {
    float v[64];
    memcpy(v, in, sizeof v);
    if (inverse) idct8x8(v); else dct8x8(v);
    memcpy(out, v, sizeof v);
}

void feds_debug_zigzag_host(int out[64]) {
    for (int z = 0; z < 64; ++z) out[z] = h_zigzag.pos[z];
}

}  // extern "C"
