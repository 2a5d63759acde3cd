// feds_api.cu — the C ABI of libfeds (include/feds.h): argument checks, workspace carving, key expansion, launches.
// Nothing here allocates, synchronises or keeps state across calls (one thread-local last-error slot aside).
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "../../include/feds.h"
#include "../../include/feds_debug.h"
#include "feds_dct.cuh"
#include "feds_device.cuh"
#include "feds_dwt.cuh"
#include "feds_host.h"

using namespace feds;

namespace {
thread_local int t_last_cuda_error = 0;
thread_local cudaEvent_t t_prof_start = nullptr, t_prof_stop = nullptr;
thread_local unsigned long long t_launches = 0;
}  // namespace

namespace feds {
feds_status cuda_fail(cudaError_t e) {
    t_last_cuda_error = (int)e;
    return FEDS_ERR_CUDA;
}
// SMs of the current device; asked per call, nothing is cached
int sm_count() {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) n = 148;
    return n;
}
cudaEvent_t prof_start_event() { return t_prof_start; }
cudaEvent_t prof_stop_event() { return t_prof_stop; }
void count_launch() { ++t_launches; }
}  // namespace feds

namespace {

constexpr AesTables h_aes = make_aes_tables();
constexpr ZigzagTable h_zigzag = make_zigzag();

inline size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline bool misaligned(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

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
// bytes of digest storage for one tree, all levels with more than one node (the single-node level is the root), and the
// arrival counters of the spread-out tree top
size_t tree_bytes(unsigned leaves) {
    unsigned n[40];
    const int L = tree_levels(leaves, n);
    size_t b = 0;
    for (int i = 0; i < L; ++i) if (n[i] > 1) b += (size_t)n[i] * 32;
    if (leaves > 1) b += TOP_CTRL_BYTES;   // arrival counters of merkle_top_kernel
    return b;
}

unsigned dct_leaves(int w, int h, int c) { return (unsigned)c * (unsigned)(h / 8) * (unsigned)((w / 8 + G_BLOCKS - 1) / G_BLOCKS); }

void nonce_to_be(const uint8_t nonce[16], uint32_t out[4]) {
    for (int i = 0; i < 4; ++i)
        out[i] = ((uint32_t)nonce[4 * i] << 24) | ((uint32_t)nonce[4 * i + 1] << 16) | ((uint32_t)nonce[4 * i + 2] << 8) | nonce[4 * i + 3];
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
                     const uint8_t *nonce_host, bool digest, bool strong = false) {
    memset(&p, 0, sizeof p);
    p.n_images = n_images; p.w = w; p.h = h; p.k = k;
    p.nbr = h / 8; p.nbc = w / 8; p.nlr = (p.nbc + G_BLOCKS - 1) / G_BLOCKS;
    p.leaves_per_image = (unsigned)c * p.nbr * p.nlr;
    p.total_leaves = (unsigned long long)p.leaves_per_image * n_images;
    p.one = 1u;
    p.c128 = 128u;
    p.pub_words = strong ? 16 : 63 - k;
    p.priv_words = k + 1;
    (void)digest;
    p.d_nonces = d_nonces;
    if (nonce_host) nonce_to_be(nonce_host, p.nonce_be);
    aes128_expand_key_host(key, p.rk, h_aes);
}

// Which route runs the path with digests: the warp-specialised fused kernels (feds_dct_fused.cuh: w % 32 == 0, whole 8-block
// leaves in linear block order) or the digest-free tile kernel and the leaf-hash kernel one after the other.
constexpr unsigned DCT_FLAGS = FEDS_FLAG_NO_DIGEST | FEDS_FLAG_FORCE_FUSED | FEDS_FLAG_FORCE_SPLIT | FEDS_FLAG_GENERIC_TILES;
enum class Route { Fused, Split, Unsupported };
Route pick_route(const DctParams &p, int c, unsigned flags) {
    const bool ws_ok = dct_fused_supported(p, c);
    if (flags & FEDS_FLAG_FORCE_FUSED) return ws_ok ? Route::Fused : Route::Unsupported;
    if (flags & FEDS_FLAG_FORCE_SPLIT) return Route::Split;
    return Route::Split;   // measured faster at every size since the tile kernels moved to bulk copies
}

feds_status fragment_dct_impl(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c, int k,
                              const uint8_t key[16], const uint8_t *d_nonces, const uint8_t *nonce_host, uint8_t *d_private,
                              size_t private_stride, uint8_t *d_public, size_t public_stride, uint8_t *d_digests,
                              void *d_workspace, size_t workspace_bytes, unsigned flags, cudaStream_t stream, bool strong = false) {
    feds_status st = check_dct_args(n_images, w, h, c, k);
    if (st != FEDS_OK) return st;
    if (flags & ~(strong ? FEDS_FLAG_NO_DIGEST : DCT_FLAGS)) return FEDS_ERR_BAD_PARAM;
    if ((flags & FEDS_FLAG_FORCE_FUSED) && (flags & FEDS_FLAG_FORCE_SPLIT)) return FEDS_ERR_BAD_PARAM;
    const bool digest = !(flags & FEDS_FLAG_NO_DIGEST);
    const size_t priv_b = feds_dct_private_bytes(w, h, c, k), pub_b = strong ? feds_dct_strong_public_bytes(w, h, c) : feds_dct_public_bytes(w, h, c, k);
    if (!d_images || !key || !d_private || (!d_public && pub_b) || (digest && (!d_digests || !d_workspace)) || (!d_nonces && !nonce_host))
        return FEDS_ERR_NULL_POINTER;
    if (image_stride < (size_t)w * h * c || private_stride < priv_b || public_stride < pub_b) return FEDS_ERR_BAD_PARAM;
    if (misaligned(d_images) || misaligned(d_private) || misaligned(d_public) || misaligned(d_digests) || misaligned(d_workspace) ||
        misaligned(d_nonces) || (n_images > 1 && ((image_stride | private_stride | public_stride) & 15u)))
        return FEDS_ERR_MISALIGNED;
    const DctPlan pl = dct_plan(w, h, c);
    if (digest && workspace_bytes < pl.per_image * (size_t)n_images) return FEDS_ERR_WORKSPACE_TOO_SMALL;

    DctParams p;
    fill_dct_params(p, n_images, w, h, c, k, key, d_nonces, nonce_host, digest, strong);
    p.generic_tiles = (flags & FEDS_FLAG_GENERIC_TILES) ? 1 : 0;
    p.images = d_images; p.image_stride = image_stride;
    p.priv = d_private; p.priv_stride = private_stride;
    p.pub = d_public; p.pub_stride = public_stride;
    uint8_t *ws = static_cast<uint8_t *>(d_workspace);
    p.leaves = (pl.nl > 1) ? ws : d_digests;  // a one-leaf fragment's root is its leaf digest
    const bool pub_empty = !strong && k == 63;
    if (strong) {   // PAPER.md 6.3.2: Part 1 under AES, the remainder pixels under a SHA-512 keystream; then the same Merkle digests
        st = launch_fragment_strong(p, c, stream, !digest);
        if (st != FEDS_OK) return st;
        if (!digest) return FEDS_OK;
        st = launch_leaves_hash(p, c, stream, true);
        if (st != FEDS_OK) return st;
        if (pl.nl > 1) return run_tree(ws, pl.nl, 2u * n_images, ws + pl.level0_bytes * n_images, d_digests, 32, 0, stream);
        return FEDS_OK;
    }
    if (digest) {
        const Route route = pick_route(p, c, flags);
        if (route == Route::Unsupported) return FEDS_ERR_BAD_PARAM;
        if (route == Route::Fused) {
            st = launch_fragment_fused(p, c, stream);
        } else {
            st = launch_fragment_tile(p, c, stream, false);
            if (st != FEDS_OK) return st;
            st = launch_leaves_hash(p, c, stream, true);   // the dominant kernel: the profiling events bracket it
        }
        if (st != FEDS_OK) return st;
        if (pl.nl > 1) {
            st = run_tree(ws, pl.nl, 2u * n_images, ws + pl.level0_bytes * n_images, d_digests, 32, pub_empty ? 1 : 0, stream);
            if (st != FEDS_OK) return st;
        }
        if (pub_empty) {
            st = launch_empty_public_roots(d_digests, n_images, stream);
            if (st != FEDS_OK) return st;
        }
    } else {
        st = launch_fragment_tile(p, c, stream, true);
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
    if (p.pub_words != 0) k = 0;   // only an EMPTY public fragment (first level, k = 63) takes the SHA-256("") root
    uint8_t *roots = verification_roots(pl, n_images, ws);
    if (pl.nl > 1) {
        const feds_status st = run_tree(ws, pl.nl, 2u * n_images, ws + pl.level0_bytes * n_images, roots, 32, k == 63 ? 1 : 0, stream);
        if (st != FEDS_OK) return st;
    }
    if (k == 63) {
        const feds_status st = launch_empty_public_roots(roots, n_images, stream);
        if (st != FEDS_OK) return st;
    }
    return launch_compare_digests(roots, d_expected, d_flags, n_images, stream);
}

feds_status defragment_dct_impl(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                int n_images, int w, int h, int c, int k, const uint8_t key[16], const uint8_t *d_nonces,
                                const uint8_t *nonce_host, const uint8_t *d_expected, uint8_t *d_images_out, size_t image_stride,
                                uint32_t *d_flags, void *d_workspace, size_t workspace_bytes, unsigned flags, cudaStream_t stream, bool strong = false) {
    feds_status st = check_dct_args(n_images, w, h, c, k);
    if (st != FEDS_OK) return st;
    if (flags & ~(strong ? FEDS_FLAG_NO_DIGEST : DCT_FLAGS)) return FEDS_ERR_BAD_PARAM;
    if ((flags & FEDS_FLAG_FORCE_FUSED) && (flags & FEDS_FLAG_FORCE_SPLIT)) return FEDS_ERR_BAD_PARAM;
    const bool verify = d_expected != nullptr && !(flags & FEDS_FLAG_NO_DIGEST);
    const size_t priv_b = feds_dct_private_bytes(w, h, c, k), pub_b = strong ? feds_dct_strong_public_bytes(w, h, c) : feds_dct_public_bytes(w, h, c, k);
    if (!d_private || (!d_public && pub_b) || !key || !d_images_out || (!d_nonces && !nonce_host) || (verify && (!d_flags || !d_workspace)))
        return FEDS_ERR_NULL_POINTER;
    if (image_stride < (size_t)w * h * c || private_stride < priv_b || public_stride < pub_b) return FEDS_ERR_BAD_PARAM;
    if (misaligned(d_images_out) || misaligned(d_private) || misaligned(d_public) || misaligned(d_expected) || misaligned(d_workspace) ||
        misaligned(d_nonces) || (n_images > 1 && ((image_stride | private_stride | public_stride) & 15u)))
        return FEDS_ERR_MISALIGNED;
    const DctPlan pl = dct_plan(w, h, c);
    if (verify && workspace_bytes < pl.per_image * (size_t)n_images) return FEDS_ERR_WORKSPACE_TOO_SMALL;

    DctParams p;
    fill_dct_params(p, n_images, w, h, c, k, key, d_nonces, nonce_host, verify, strong);
    p.generic_tiles = (flags & FEDS_FLAG_GENERIC_TILES) ? 1 : 0;
    p.images_out = d_images_out; p.image_stride = image_stride;
    p.priv = const_cast<uint8_t *>(d_private); p.priv_stride = private_stride;
    p.pub = const_cast<uint8_t *>(d_public); p.pub_stride = public_stride;
    if (strong) {
        if (verify) {
            p.leaves = verification_leaves(pl, n_images, static_cast<uint8_t *>(d_workspace));
            st = launch_leaves_hash(p, c, stream, true);
            if (st != FEDS_OK) return st;
        }
        st = launch_defragment_strong(p, c, stream, !verify);
        if (st != FEDS_OK) return st;
        return verify ? finish_verification(p, pl, n_images, k, static_cast<uint8_t *>(d_workspace), d_expected, d_flags, stream) : FEDS_OK;
    }
    if (verify) {
        p.leaves = verification_leaves(pl, n_images, static_cast<uint8_t *>(d_workspace));
        // Verification and reconstruction read the same fragments. Fused route: one warp-specialised kernel whose hash warps
        // and reconstruction warps walk the leaves together, so the fragments come from HBM once (feds_dct_fused.cuh; forced route only). Split
        // route: the registers-only leaf-hash kernel, then the digest-free tile kernel.
        const Route route = pick_route(p, c, flags);
        if (route == Route::Unsupported) return FEDS_ERR_BAD_PARAM;
        if (route == Route::Fused) {
            st = launch_defragment_fused(p, c, stream);
        } else {
            st = launch_leaves_hash(p, c, stream, true);
            if (st != FEDS_OK) return st;
            st = launch_defragment_tile(p, c, stream, false);
        }
        if (st != FEDS_OK) return st;
        return finish_verification(p, pl, n_images, k, static_cast<uint8_t *>(d_workspace), d_expected, d_flags, stream);
    }
    return launch_defragment_tile(p, c, stream, true);
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
    st = launch_leaves_hash(p, c, stream, true);
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
    pl.priv_tree = std::max<size_t>(tree_bytes(pl.priv_nl), 32);   // a one-leaf tree still parks its leaf digest here in a batch
    pl.pub_tree = std::max<size_t>(tree_bytes(pl.pub_nl), 32);
    pl.per_image = round_up(pl.planes_bytes + round_up(pl.priv_tree, 256) + round_up(pl.pub_tree, 256) + 64, 256);
    return pl;
}

size_t dwt_level_off_elems(int w, int h, int L, int l) {  // elements before level l's bands inside one channel's public run
    size_t off = 0;
    for (int m = L; m > l; --m) off += (size_t)3 * (w >> m) * (h >> m);
    return off;
}

// leaf digests + trees of the two fragments of n_images images -> roots[i][64] (private root || public root).
// tree_ws: [private leaves of all images][private upper levels][public leaves of all images][public upper levels]
feds_status dwt_digests(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride, int n_images,
                        const DwtPlan &pl, uint8_t *tree_ws, uint8_t *roots, cudaStream_t stream) {
    const unsigned nls[2] = {pl.priv_nl, pl.pub_nl};
    uint8_t *ws[2] = {tree_ws, tree_ws + round_up(pl.priv_tree, 256) * (size_t)n_images};
    const uint8_t *const data[2] = {d_private, d_public};
    const size_t strides[2] = {private_stride, public_stride};
    const unsigned long long nbytes[2] = {pl.priv_b, pl.pub_b};
    // a one-leaf fragment's root is its leaf digest: with one image it is written in place; a batch of one-leaf fragments
    // goes through the workspace and the tail kernel is skipped by copying (n0 == 1 trees need no reduction, see below)
    uint8_t *out[2];
    for (int f = 0; f < 2; ++f) out[f] = (nls[f] > 1 || n_images > 1) ? ws[f] : roots + 32 * f;
    feds_status st = launch_stream_leaves(data, strides, nbytes, nls, out, (unsigned)n_images, true, stream);
    if (st != FEDS_OK) return st;
    if (n_images > 1) {
        for (int f = 0; f < 2; ++f)
            if (nls[f] == 1) FEDS_CUDA(cudaMemcpy2DAsync(roots + 32 * f, 64, ws[f], 32, 32, (size_t)n_images, cudaMemcpyDeviceToDevice, stream));
    }
    return run_two_trees(ws[0], nls[0], ws[0] + (size_t)nls[0] * 32 * n_images, roots, ws[1], nls[1], ws[1] + (size_t)nls[1] * 32 * n_images,
                         roots + 32, (unsigned)n_images, 64, stream);
}

feds_status check_dwt_args(int n_images, int w, int h, int c, int levels) {
    if (w <= 0 || h <= 0) return FEDS_ERR_BAD_DIMS;
    if (!chan_ok(c) || levels < 1 || levels > 6 || n_images < 1) return FEDS_ERR_BAD_PARAM;
    if (!dwt_dims_ok(w, h, levels)) return FEDS_ERR_BAD_DIMS;
    return FEDS_OK;
}

// Workspace of a DWT batch, level-major so that the planes of one level are contiguous over the images (the level kernels
// index planes by n * C + c): [LL_1 planes of all images] ... [LL_L planes][trees][n x 64 B recomputed roots].
size_t dwt_plane_off(const DwtPlan &pl, int l, int n_images) { return pl.plane_off[l] * (size_t)n_images; }

feds_status fragment_dwt_impl(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c, int levels,
                              const uint8_t key[16], const uint8_t *nonce_host, const uint8_t *d_nonces, uint8_t *d_private,
                              size_t private_stride, uint8_t *d_public, size_t public_stride, uint8_t *d_digests, void *d_workspace,
                              size_t workspace_bytes, unsigned flags, cudaStream_t stream) {
    feds_status st = check_dwt_args(n_images, w, h, c, levels);
    if (st != FEDS_OK) return st;
    if (flags & ~FEDS_FLAG_DWT_TILED) return FEDS_ERR_BAD_PARAM;
    if (!d_images || !key || (!nonce_host && !d_nonces) || !d_private || !d_public || !d_digests || !d_workspace) return FEDS_ERR_NULL_POINTER;
    const DwtPlan pl = dwt_plan(w, h, c, levels);
    if (image_stride < (size_t)w * h * c || private_stride < pl.priv_b || public_stride < pl.pub_b) return FEDS_ERR_BAD_PARAM;
    if (misaligned(d_images) || misaligned(d_private) || misaligned(d_public) || misaligned(d_digests) || misaligned(d_workspace) ||
        misaligned(d_nonces) || (n_images > 1 && ((image_stride | private_stride | public_stride) & 15u)))
        return FEDS_ERR_MISALIGNED;
    if (workspace_bytes < pl.per_image * (size_t)n_images) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    uint8_t *ws = static_cast<uint8_t *>(d_workspace);
    const int L = levels;
    const bool tiled = (flags & FEDS_FLAG_DWT_TILED) != 0;

    for (int l = 1; l <= L; ++l) {
        DwtLevelParams p{};
        p.C = c; p.img_w = w; p.image_stride = image_stride;
        p.cw = w >> (l - 1); p.ch = h >> (l - 1);
        const int bw = w >> l, bh = h >> l;
        p.img_in = d_images;
        if (l > 1) { p.ll_in = reinterpret_cast<const int16_t *>(ws + dwt_plane_off(pl, l - 1, n_images)); p.ll_in_plane_stride = (size_t)p.cw * p.ch; }
        if (l < L) {
            p.ll_band = reinterpret_cast<int16_t *>(ws + dwt_plane_off(pl, l, n_images));
            p.ll_band_image_stride = (size_t)c * bw * bh; p.ll_band_chan_stride = (size_t)bw * bh;
        } else {
            p.ll_band = reinterpret_cast<int16_t *>(d_private);
            p.ll_band_image_stride = private_stride / 2; p.ll_band_chan_stride = (size_t)bw * bh;
        }
        p.pub = reinterpret_cast<int16_t *>(d_public);
        p.pub_image_stride = public_stride / 2;
        p.pub_chan_stride = pl.pub_b / 2 / c;
        p.level_off = dwt_level_off_elems(w, h, L, l);
        st = launch_dwt_fwd_level(p, l == 1, c, n_images, tiled, stream);
        if (st != FEDS_OK) return st;
    }
    st = launch_aes_ctr(d_private, private_stride, d_private, private_stride, pl.priv_b, (unsigned)n_images, key, nonce_host, d_nonces, stream);
    if (st != FEDS_OK) return st;
    return dwt_digests(d_private, private_stride, d_public, public_stride, n_images, pl, ws + pl.planes_bytes * (size_t)n_images, d_digests, stream);
}

feds_status defragment_dwt_impl(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                int n_images, int w, int h, int c, int levels, const uint8_t key[16], const uint8_t *nonce_host,
                                const uint8_t *d_nonces, const uint8_t *d_expected_digests, uint8_t *d_images_out, size_t image_stride,
                                uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes, unsigned flags, cudaStream_t stream,
                                cudaStream_t aux_stream = nullptr, cudaEvent_t fork_event = nullptr, cudaEvent_t join_event = nullptr) {
    feds_status st = check_dwt_args(n_images, w, h, c, levels);
    if (st != FEDS_OK) return st;
    if (flags & ~FEDS_FLAG_DWT_TILED) return FEDS_ERR_BAD_PARAM;
    if (!d_private || !d_public || !key || (!nonce_host && !d_nonces) || !d_images_out || !d_workspace || (d_expected_digests && !d_verify_flags))
        return FEDS_ERR_NULL_POINTER;
    const bool two_streams = fork_event != nullptr;   // verification on aux_stream (feds_defragment_dwt_batch_2s)
    const DwtPlan pl = dwt_plan(w, h, c, levels);
    if (image_stride < (size_t)w * h * c || private_stride < pl.priv_b || public_stride < pl.pub_b) return FEDS_ERR_BAD_PARAM;
    if (misaligned(d_images_out) || misaligned(d_private) || misaligned(d_public) || misaligned(d_expected_digests) || misaligned(d_workspace) ||
        misaligned(d_nonces) || (n_images > 1 && ((image_stride | private_stride | public_stride) & 15u)))
        return FEDS_ERR_MISALIGNED;
    if (workspace_bytes < pl.per_image * (size_t)n_images) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    uint8_t *ws = static_cast<uint8_t *>(d_workspace);
    const int L = levels;
    const bool tiled = (flags & FEDS_FLAG_DWT_TILED) != 0;

    if (d_expected_digests) {
        cudaStream_t vs = stream;
        if (two_streams) {
            FEDS_CUDA(cudaEventRecord(fork_event, stream));
            FEDS_CUDA(cudaStreamWaitEvent(aux_stream, fork_event, 0));
            vs = aux_stream;
        }
        uint8_t *roots = ws + pl.per_image * (size_t)n_images - 64 * (size_t)n_images;
        st = dwt_digests(d_private, private_stride, d_public, public_stride, n_images, pl, ws + pl.planes_bytes * (size_t)n_images, roots, vs);
        if (st == FEDS_OK) st = launch_compare_digests(roots, d_expected_digests, d_verify_flags, n_images, vs);
        if (two_streams) FEDS_CUDA(cudaEventRecord(join_event, aux_stream));
    }
    // the reconstruction runs on `stream` meanwhile; `stream` waits for the verification at the very end (also after a failed
    // launch: a capture must not be left forked)
    auto joined = [&](feds_status s) {
        if (two_streams && cudaStreamWaitEvent(stream, join_event, 0) != cudaSuccess && s == FEDS_OK) return FEDS_ERR_CUDA;
        return s;
    };
    if (st != FEDS_OK) return joined(st);
    // decrypt LL_L into the level-L plane block (the received fragment stays untouched)
    // (image stride rounded up to 16 bytes: the CTR kernel moves 128-bit words; the plane block has 256-byte slack per image)
    uint8_t *lldec = ws + dwt_plane_off(pl, L, n_images);
    const size_t lldec_stride = round_up(pl.priv_b, 16);
    st = launch_aes_ctr(d_private, private_stride, lldec, lldec_stride, pl.priv_b, (unsigned)n_images, key, nonce_host, d_nonces, stream);
    if (st != FEDS_OK) return joined(st);

    for (int l = L; l >= 1; --l) {
        DwtLevelParams p{};
        p.C = c; p.img_w = w; p.image_stride = image_stride;
        p.cw = w >> (l - 1); p.ch = h >> (l - 1);
        const int bw = w >> l, bh = h >> l;
        p.ll_band = reinterpret_cast<int16_t *>(ws + dwt_plane_off(pl, l, n_images));
        p.ll_band_image_stride = (l == L) ? lldec_stride / 2 : (size_t)c * bw * bh; p.ll_band_chan_stride = (size_t)bw * bh;
        p.pub = reinterpret_cast<int16_t *>(const_cast<uint8_t *>(d_public));
        p.pub_image_stride = public_stride / 2;
        p.pub_chan_stride = pl.pub_b / 2 / c;
        p.level_off = dwt_level_off_elems(w, h, L, l);
        p.img_out = d_images_out;
        if (l > 1) { p.ll_out_plane = reinterpret_cast<int16_t *>(ws + dwt_plane_off(pl, l - 1, n_images)); p.ll_out_plane_stride = (size_t)p.cw * p.ch; }
        st = launch_dwt_inv_level(p, l == 1, c, n_images, tiled, stream);
        if (st != FEDS_OK) return joined(st);
    }
    return joined(FEDS_OK);
}

// ---------------------------------------------------------------------------------------------- packed integer storage
bool packed_args_ok(int ac_bits) { return ac_bits == 11 || ac_bits == 8; }
unsigned packed_bits_per_block(int k, int ac_bits) { return 11u + (unsigned)k * (unsigned)ac_bits; }
size_t packed_row_bytes(int w, int k, int ac_bits) {
    const unsigned nbc = (unsigned)(w / 8), b = packed_bits_per_block(k, ac_bits);
    return (size_t)(nbc / G_BLOCKS) * b + ((nbc % G_BLOCKS) ? ((size_t)(nbc % G_BLOCKS) * b + 7) / 8 : 0);
}
void fill_packed_params(DctParams &p, int w, int k, int ac_bits) {
    p.pub_words = 16;
    p.priv_words = 0;   // the word-wise leaf-hash kernels skip the private fragment: packed_private_leaves_kernel hashes it
    p.ac_bits = ac_bits;
    p.packed_group_bytes = packed_bits_per_block(k, ac_bits);
    p.packed_row_bytes = packed_row_bytes(w, k, ac_bits);
}

feds_status fragment_packed_impl(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c, int k, int ac_bits,
                                 const uint8_t key[16], const uint8_t *nonce_host, const uint8_t *d_nonces, uint8_t *d_private,
                                 size_t private_stride, uint8_t *d_public, size_t public_stride, uint8_t *d_digests, void *d_workspace,
                                 size_t workspace_bytes, cudaStream_t stream) {
    feds_status st = check_dct_args(n_images, w, h, c, k);
    if (st != FEDS_OK) return st;
    if (!packed_args_ok(ac_bits)) return FEDS_ERR_BAD_PARAM;
    const size_t priv_b = feds_dct_packed_private_bytes(w, h, c, k, ac_bits), pub_b = (size_t)w * h * c;
    if (!d_images || !key || !d_private || !d_public || !d_digests || !d_workspace || (!d_nonces && !nonce_host)) return FEDS_ERR_NULL_POINTER;
    if (image_stride < pub_b || private_stride < priv_b || public_stride < pub_b) return FEDS_ERR_BAD_PARAM;
    if (misaligned(d_images) || misaligned(d_private) || misaligned(d_public) || misaligned(d_digests) || misaligned(d_workspace) ||
        misaligned(d_nonces) || (n_images > 1 && ((image_stride | private_stride | public_stride) & 15u)))
        return FEDS_ERR_MISALIGNED;
    const DctPlan pl = dct_plan(w, h, c);
    if (workspace_bytes < feds_dct_packed_workspace_bytes(w, h, c, k, ac_bits) * (size_t)n_images) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    DctParams p;
    fill_dct_params(p, n_images, w, h, c, k, key, d_nonces, nonce_host, true);
    fill_packed_params(p, w, k, ac_bits);
    p.images = d_images; p.image_stride = image_stride;
    p.priv = d_private; p.priv_stride = private_stride;
    p.pub = d_public; p.pub_stride = public_stride;
    uint8_t *ws = static_cast<uint8_t *>(d_workspace);
    p.leaves = (pl.nl > 1) ? ws : d_digests;
    st = launch_fragment_packed(p, c, stream, false);
    if (st != FEDS_OK) return st;
    st = launch_aes_ctr(d_private, private_stride, d_private, private_stride, priv_b, (unsigned)n_images, key, nonce_host, d_nonces, stream);
    if (st != FEDS_OK) return st;
    st = launch_leaves_hash(p, c, stream, true);       // public leaves (16 words per block)
    if (st != FEDS_OK) return st;
    st = launch_packed_private_leaves(p, c, stream);   // private leaves (the groups' bytes, as stored: ciphertext)
    if (st != FEDS_OK) return st;
    if (pl.nl > 1) return run_tree(ws, pl.nl, 2u * n_images, ws + pl.level0_bytes * n_images, d_digests, 32, 0, stream);
    return FEDS_OK;
}

feds_status defragment_packed_impl(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                   int n_images, int w, int h, int c, int k, int ac_bits, const uint8_t key[16], const uint8_t *nonce_host,
                                   const uint8_t *d_nonces, const uint8_t *d_expected, uint8_t *d_images_out, size_t image_stride,
                                   uint32_t *d_flags, void *d_workspace, size_t workspace_bytes, cudaStream_t stream) {
    feds_status st = check_dct_args(n_images, w, h, c, k);
    if (st != FEDS_OK) return st;
    if (!packed_args_ok(ac_bits)) return FEDS_ERR_BAD_PARAM;
    const size_t priv_b = feds_dct_packed_private_bytes(w, h, c, k, ac_bits), pub_b = (size_t)w * h * c;
    if (!d_private || !d_public || !key || !d_images_out || !d_workspace || (!d_nonces && !nonce_host) || (d_expected && !d_flags))
        return FEDS_ERR_NULL_POINTER;
    if (image_stride < pub_b || private_stride < priv_b || public_stride < pub_b) return FEDS_ERR_BAD_PARAM;
    if (misaligned(d_images_out) || misaligned(d_private) || misaligned(d_public) || misaligned(d_expected) || misaligned(d_workspace) ||
        misaligned(d_nonces) || (n_images > 1 && ((image_stride | private_stride | public_stride) & 15u)))
        return FEDS_ERR_MISALIGNED;
    const DctPlan pl = dct_plan(w, h, c);
    if (workspace_bytes < feds_dct_packed_workspace_bytes(w, h, c, k, ac_bits) * (size_t)n_images) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    DctParams p;
    fill_dct_params(p, n_images, w, h, c, k, key, d_nonces, nonce_host, d_expected != nullptr);
    fill_packed_params(p, w, k, ac_bits);
    p.images_out = d_images_out; p.image_stride = image_stride;
    p.priv = const_cast<uint8_t *>(d_private); p.priv_stride = private_stride;
    p.pub = const_cast<uint8_t *>(d_public); p.pub_stride = public_stride;
    uint8_t *ws = static_cast<uint8_t *>(d_workspace);
    if (d_expected) {
        p.leaves = verification_leaves(pl, n_images, ws);
        st = launch_leaves_hash(p, c, stream, true);
        if (st != FEDS_OK) return st;
        st = launch_packed_private_leaves(p, c, stream);
        if (st != FEDS_OK) return st;
        st = finish_verification(p, pl, n_images, k, ws, d_expected, d_flags, stream);
        if (st != FEDS_OK) return st;
    }
    // the decrypted private fragments live behind the digest workspace of the whole batch
    const size_t plain_stride = round_up(priv_b, 256);
    uint8_t *plain = ws + pl.per_image * (size_t)n_images;
    st = launch_aes_ctr(d_private, private_stride, plain, plain_stride, priv_b, (unsigned)n_images, key, nonce_host, d_nonces, stream);
    if (st != FEDS_OK) return st;
    return launch_defragment_packed(p, c, plain, plain_stride, stream, d_expected == nullptr);
}

// ---------------------------------------------------------------------------------------------- tiled DWT design
DwtPlan tiles_plan(int w, int h, int c) {
    DwtPlan pl{};
    const size_t T = (size_t)(w / 8) * (h / 8) * c;
    pl.priv_b = 21 * T;
    pl.pub_b = 60 * T;
    pl.priv_nl = (unsigned)((pl.priv_b + DWT_LEAF_BYTES - 1) / DWT_LEAF_BYTES);
    pl.pub_nl = (unsigned)((pl.pub_b + DWT_LEAF_BYTES - 1) / DWT_LEAF_BYTES);
    pl.planes_bytes = 0;
    pl.priv_tree = std::max<size_t>(tree_bytes(pl.priv_nl), 32);
    pl.pub_tree = std::max<size_t>(tree_bytes(pl.pub_nl), 32);
    pl.per_image = round_up(round_up(pl.priv_tree, 256) + round_up(pl.pub_tree, 256) + 64, 256);
    return pl;
}
feds_status check_tiles_args(int n_images, int w, int h, int c) {
    if (!dct_dims_ok(w, h)) return FEDS_ERR_BAD_DIMS;
    if (!chan_ok(c) || n_images < 1) return FEDS_ERR_BAD_PARAM;
    return FEDS_OK;
}
void fill_tiles_params(DctParams &p, int n_images, int w, int h, const uint8_t key[16], const uint8_t *d_nonces, const uint8_t *nonce_host) {
    memset(&p, 0, sizeof p);
    p.n_images = n_images; p.w = w; p.h = h;
    p.nbr = h / 8; p.nbc = w / 8;
    p.one = 1u;
    p.d_nonces = d_nonces;
    if (nonce_host) nonce_to_be(nonce_host, p.nonce_be);
    aes128_expand_key_host(key, p.rk, h_aes);
}

feds_status fragment_tiles_impl(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c, const uint8_t key[16],
                                const uint8_t *nonce_host, const uint8_t *d_nonces, uint8_t *d_private, size_t private_stride,
                                uint8_t *d_public, size_t public_stride, uint8_t *d_digests, void *d_workspace, size_t workspace_bytes,
                                cudaStream_t stream) {
    feds_status st = check_tiles_args(n_images, w, h, c);
    if (st != FEDS_OK) return st;
    if (!d_images || !key || (!nonce_host && !d_nonces) || !d_private || !d_public || !d_digests || !d_workspace) return FEDS_ERR_NULL_POINTER;
    const DwtPlan pl = tiles_plan(w, h, c);
    if (image_stride < (size_t)w * h * c || private_stride < pl.priv_b || public_stride < pl.pub_b) return FEDS_ERR_BAD_PARAM;
    if (misaligned(d_images) || misaligned(d_private) || misaligned(d_public) || misaligned(d_digests) || misaligned(d_workspace) ||
        misaligned(d_nonces) || (n_images > 1 && ((image_stride | private_stride | public_stride) & 15u)))
        return FEDS_ERR_MISALIGNED;
    if (workspace_bytes < pl.per_image * (size_t)n_images) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    DctParams p;
    fill_tiles_params(p, n_images, w, h, key, d_nonces, nonce_host);
    p.images = d_images; p.image_stride = image_stride;
    p.priv = d_private; p.priv_stride = private_stride;
    p.pub = d_public; p.pub_stride = public_stride;
    st = launch_fragment_dwt_tiles(p, c, stream);
    if (st != FEDS_OK) return st;
    return dwt_digests(d_private, private_stride, d_public, public_stride, n_images, pl, static_cast<uint8_t *>(d_workspace), d_digests, stream);
}

feds_status defragment_tiles_impl(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride, int n_images,
                                  int w, int h, int c, const uint8_t key[16], const uint8_t *nonce_host, const uint8_t *d_nonces,
                                  const uint8_t *d_expected, uint8_t *d_images_out, size_t image_stride, uint32_t *d_flags, void *d_workspace,
                                  size_t workspace_bytes, cudaStream_t stream) {
    feds_status st = check_tiles_args(n_images, w, h, c);
    if (st != FEDS_OK) return st;
    if (!d_private || !d_public || !key || (!nonce_host && !d_nonces) || !d_images_out || (d_expected && (!d_flags || !d_workspace)))
        return FEDS_ERR_NULL_POINTER;
    const DwtPlan pl = tiles_plan(w, h, c);
    if (image_stride < (size_t)w * h * c || private_stride < pl.priv_b || public_stride < pl.pub_b) return FEDS_ERR_BAD_PARAM;
    if (misaligned(d_images_out) || misaligned(d_private) || misaligned(d_public) || misaligned(d_expected) || misaligned(d_workspace) ||
        misaligned(d_nonces) || (n_images > 1 && ((image_stride | private_stride | public_stride) & 15u)))
        return FEDS_ERR_MISALIGNED;
    if (d_expected) {
        if (workspace_bytes < pl.per_image * (size_t)n_images) return FEDS_ERR_WORKSPACE_TOO_SMALL;
        uint8_t *ws = static_cast<uint8_t *>(d_workspace);
        uint8_t *roots = ws + pl.per_image * (size_t)n_images - 64 * (size_t)n_images;
        st = dwt_digests(d_private, private_stride, d_public, public_stride, n_images, pl, ws, roots, stream);
        if (st != FEDS_OK) return st;
        st = launch_compare_digests(roots, d_expected, d_flags, n_images, stream);
        if (st != FEDS_OK) return st;
    }
    DctParams p;
    fill_tiles_params(p, n_images, w, h, key, d_nonces, nonce_host);
    p.images_out = d_images_out; p.image_stride = image_stride;
    p.priv = const_cast<uint8_t *>(d_private); p.priv_stride = private_stride;
    p.pub = const_cast<uint8_t *>(d_public); p.pub_stride = public_stride;
    return launch_defragment_dwt_tiles(p, c, stream);
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

// ------------------------------------------------------------------------------------------------ strong level
size_t feds_dct_strong_public_bytes(int w, int h, int c) {
    if (!dct_dims_ok(w, h) || !chan_ok(c)) return 0;
    return (size_t)w * h * c;
}

feds_status feds_fragment_dct_strong(const uint8_t *d_image, int w, int h, int c, int k, const uint8_t key[16], const uint8_t nonce[16],
                                     uint8_t *d_private, uint8_t *d_public, uint8_t *d_digests, void *d_workspace, size_t workspace_bytes,
                                     feds_stream_t stream) {
    if (!nonce) return FEDS_ERR_NULL_POINTER;
    return fragment_dct_impl(d_image, 1, (size_t)(w > 0 ? w : 0) * (h > 0 ? h : 0) * (c > 0 ? c : 0), w, h, c, k, key, nullptr, nonce,
                             d_private, feds_dct_private_bytes(w, h, c, k), d_public, feds_dct_strong_public_bytes(w, h, c), d_digests,
                             d_workspace, workspace_bytes, FEDS_FLAG_NONE, stream, true);
}

feds_status feds_fragment_dct_strong_batch(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c, int k,
                                           const uint8_t key[16], const uint8_t *d_nonces, uint8_t *d_private, size_t private_stride,
                                           uint8_t *d_public, size_t public_stride, uint8_t *d_digests, void *d_workspace,
                                           size_t workspace_bytes, unsigned flags, feds_stream_t stream) {
    if (!d_nonces) return FEDS_ERR_NULL_POINTER;
    return fragment_dct_impl(d_images, n_images, image_stride, w, h, c, k, key, d_nonces, nullptr, d_private, private_stride, d_public,
                             public_stride, d_digests, d_workspace, workspace_bytes, flags, stream, true);
}

feds_status feds_defragment_dct_strong(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int k, const uint8_t key[16],
                                       const uint8_t nonce[16], const uint8_t *d_expected_digests, uint8_t *d_image_out,
                                       uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes, feds_stream_t stream) {
    if (!nonce) return FEDS_ERR_NULL_POINTER;
    return defragment_dct_impl(d_private, feds_dct_private_bytes(w, h, c, k), d_public, feds_dct_strong_public_bytes(w, h, c), 1, w, h, c, k,
                               key, nullptr, nonce, d_expected_digests, d_image_out,
                               (size_t)(w > 0 ? w : 0) * (h > 0 ? h : 0) * (c > 0 ? c : 0), d_verify_flags, d_workspace, workspace_bytes,
                               FEDS_FLAG_NONE, stream, true);
}

feds_status feds_defragment_dct_strong_batch(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                             int n_images, int w, int h, int c, int k, const uint8_t key[16], const uint8_t *d_nonces,
                                             const uint8_t *d_expected_digests, uint8_t *d_images_out, size_t image_stride,
                                             uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes, unsigned flags,
                                             feds_stream_t stream) {
    if (!d_nonces) return FEDS_ERR_NULL_POINTER;
    return defragment_dct_impl(d_private, private_stride, d_public, public_stride, n_images, w, h, c, k, key, d_nonces, nullptr,
                               d_expected_digests, d_images_out, image_stride, d_verify_flags, d_workspace, workspace_bytes, flags,
                               stream, true);
}

// ------------------------------------------------------------------------------------------------ packed storage
size_t feds_dct_packed_private_bytes(int w, int h, int c, int k, int ac_bits) {
    if (!dct_dims_ok(w, h) || !chan_ok(c) || k < 0 || k > 63 || !packed_args_ok(ac_bits)) return 0;
    return (size_t)c * (h / 8) * packed_row_bytes(w, k, ac_bits);
}
size_t feds_dct_packed_workspace_bytes(int w, int h, int c, int k, int ac_bits) {
    const size_t pb = feds_dct_packed_private_bytes(w, h, c, k, ac_bits);
    if (pb == 0) return 0;
    return dct_plan(w, h, c).per_image + round_up(pb, 256);
}
feds_status feds_fragment_dct_packed(const uint8_t *d_image, int w, int h, int c, int k, int ac_bits, const uint8_t key[16],
                                     const uint8_t nonce[16], uint8_t *d_private, uint8_t *d_public, uint8_t *d_digests,
                                     void *d_workspace, size_t workspace_bytes, feds_stream_t stream) {
    if (!nonce) return FEDS_ERR_NULL_POINTER;
    return fragment_packed_impl(d_image, 1, (size_t)(w > 0 ? w : 0) * (h > 0 ? h : 0) * (c > 0 ? c : 0), w, h, c, k, ac_bits, key, nonce, nullptr,
                                d_private, feds_dct_packed_private_bytes(w, h, c, k, ac_bits), d_public,
                                (size_t)(w > 0 ? w : 0) * (h > 0 ? h : 0) * (c > 0 ? c : 0), d_digests, d_workspace, workspace_bytes, stream);
}
feds_status feds_fragment_dct_packed_batch(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c, int k,
                                           int ac_bits, const uint8_t key[16], const uint8_t *d_nonces, uint8_t *d_private,
                                           size_t private_stride, uint8_t *d_public, size_t public_stride, uint8_t *d_digests,
                                           void *d_workspace, size_t workspace_bytes, feds_stream_t stream) {
    if (!d_nonces) return FEDS_ERR_NULL_POINTER;
    return fragment_packed_impl(d_images, n_images, image_stride, w, h, c, k, ac_bits, key, nullptr, d_nonces, d_private, private_stride,
                                d_public, public_stride, d_digests, d_workspace, workspace_bytes, stream);
}
feds_status feds_defragment_dct_packed(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int k, int ac_bits,
                                       const uint8_t key[16], const uint8_t nonce[16], const uint8_t *d_expected_digests,
                                       uint8_t *d_image_out, uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes,
                                       feds_stream_t stream) {
    if (!nonce) return FEDS_ERR_NULL_POINTER;
    const size_t img_b = (size_t)(w > 0 ? w : 0) * (h > 0 ? h : 0) * (c > 0 ? c : 0);
    return defragment_packed_impl(d_private, feds_dct_packed_private_bytes(w, h, c, k, ac_bits), d_public, img_b, 1, w, h, c, k, ac_bits, key,
                                  nonce, nullptr, d_expected_digests, d_image_out, img_b, d_verify_flags, d_workspace, workspace_bytes, stream);
}
feds_status feds_defragment_dct_packed_batch(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                             int n_images, int w, int h, int c, int k, int ac_bits, const uint8_t key[16],
                                             const uint8_t *d_nonces, const uint8_t *d_expected_digests, uint8_t *d_images_out,
                                             size_t image_stride, uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes,
                                             feds_stream_t stream) {
    if (!d_nonces) return FEDS_ERR_NULL_POINTER;
    return defragment_packed_impl(d_private, private_stride, d_public, public_stride, n_images, w, h, c, k, ac_bits, key, nullptr, d_nonces,
                                  d_expected_digests, d_images_out, image_stride, d_verify_flags, d_workspace, workspace_bytes, stream);
}

// ------------------------------------------------------------------------------------------------ DWT
feds_status feds_fragment_dwt(const uint8_t *d_image, int w, int h, int c, int levels, const uint8_t key[16], const uint8_t nonce[16],
                              uint8_t *d_private, uint8_t *d_public, uint8_t *d_digests, void *d_workspace, size_t workspace_bytes,
                              feds_stream_t stream) {
    if (!nonce) return check_dwt_args(1, w, h, c, levels) != FEDS_OK ? check_dwt_args(1, w, h, c, levels) : FEDS_ERR_NULL_POINTER;
    return fragment_dwt_impl(d_image, 1, (size_t)(w > 0 ? w : 0) * (h > 0 ? h : 0) * (c > 0 ? c : 0), w, h, c, levels, key, nonce, nullptr,
                             d_private, feds_dwt_private_bytes(w, h, c, levels), d_public, feds_dwt_public_bytes(w, h, c, levels), d_digests,
                             d_workspace, workspace_bytes, FEDS_FLAG_NONE, stream);
}

feds_status feds_fragment_dwt_batch(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c, int levels,
                                    const uint8_t key[16], const uint8_t *d_nonces, uint8_t *d_private, size_t private_stride,
                                    uint8_t *d_public, size_t public_stride, uint8_t *d_digests, void *d_workspace,
                                    size_t workspace_bytes, unsigned flags, feds_stream_t stream) {
    if (!d_nonces) return check_dwt_args(n_images, w, h, c, levels) != FEDS_OK ? check_dwt_args(n_images, w, h, c, levels) : FEDS_ERR_NULL_POINTER;
    return fragment_dwt_impl(d_images, n_images, image_stride, w, h, c, levels, key, nullptr, d_nonces, d_private, private_stride, d_public,
                             public_stride, d_digests, d_workspace, workspace_bytes, flags, stream);
}

feds_status feds_defragment_dwt(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int levels,
                                const uint8_t key[16], const uint8_t nonce[16], const uint8_t *d_expected_digests,
                                uint8_t *d_image_out, uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes,
                                feds_stream_t stream) {
    if (!nonce) return check_dwt_args(1, w, h, c, levels) != FEDS_OK ? check_dwt_args(1, w, h, c, levels) : FEDS_ERR_NULL_POINTER;
    return defragment_dwt_impl(d_private, feds_dwt_private_bytes(w, h, c, levels), d_public, feds_dwt_public_bytes(w, h, c, levels), 1, w, h,
                               c, levels, key, nonce, nullptr, d_expected_digests, d_image_out,
                               (size_t)(w > 0 ? w : 0) * (h > 0 ? h : 0) * (c > 0 ? c : 0), d_verify_flags, d_workspace, workspace_bytes,
                               FEDS_FLAG_NONE, stream);
}

feds_status feds_defragment_dwt_batch(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                      int n_images, int w, int h, int c, int levels, const uint8_t key[16], const uint8_t *d_nonces,
                                      const uint8_t *d_expected_digests, uint8_t *d_images_out, size_t image_stride,
                                      uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes, unsigned flags,
                                      feds_stream_t stream) {
    if (!d_nonces) return check_dwt_args(n_images, w, h, c, levels) != FEDS_OK ? check_dwt_args(n_images, w, h, c, levels) : FEDS_ERR_NULL_POINTER;
    return defragment_dwt_impl(d_private, private_stride, d_public, public_stride, n_images, w, h, c, levels, key, nullptr, d_nonces,
                               d_expected_digests, d_images_out, image_stride, d_verify_flags, d_workspace, workspace_bytes, flags, stream);
}

feds_status feds_defragment_dwt_batch_2s(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                         int n_images, int w, int h, int c, int levels, const uint8_t key[16], const uint8_t *d_nonces,
                                         const uint8_t *d_expected_digests, uint8_t *d_images_out, size_t image_stride,
                                         uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes, unsigned flags,
                                         feds_stream_t stream, feds_stream_t aux_stream, feds_event_t fork_event, feds_event_t join_event) {
    const feds_status st = check_dwt_args(n_images, w, h, c, levels);
    if (st != FEDS_OK) return st;
    if (!d_nonces || !d_expected_digests || !d_verify_flags || !aux_stream || !fork_event || !join_event) return FEDS_ERR_NULL_POINTER;
    if (aux_stream == stream) return FEDS_ERR_BAD_PARAM;
    return defragment_dwt_impl(d_private, private_stride, d_public, public_stride, n_images, w, h, c, levels, key, nullptr, d_nonces,
                               d_expected_digests, d_images_out, image_stride, d_verify_flags, d_workspace, workspace_bytes, flags, stream,
                               aux_stream, fork_event, join_event);
}

feds_status feds_verify_dwt(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int levels,
                            const uint8_t *d_expected_digests, uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes,
                            feds_stream_t stream) {
    const feds_status a0 = check_dwt_args(1, w, h, c, levels);
    if (a0 != FEDS_OK) return a0;
    if (!d_private || !d_public || !d_expected_digests || !d_verify_flags || !d_workspace) return FEDS_ERR_NULL_POINTER;
    if (misaligned(d_private) || misaligned(d_public) || misaligned(d_expected_digests) || misaligned(d_workspace)) return FEDS_ERR_MISALIGNED;
    const DwtPlan pl = dwt_plan(w, h, c, levels);
    if (workspace_bytes < pl.per_image) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    uint8_t *ws = static_cast<uint8_t *>(d_workspace);
    uint8_t *roots = ws + pl.per_image - 64;
    const feds_status st = dwt_digests(d_private, pl.priv_b, d_public, pl.pub_b, 1, pl, ws + pl.planes_bytes, roots, stream);
    if (st != FEDS_OK) return st;
    return launch_compare_digests(roots, d_expected_digests, d_verify_flags, 1, stream);
}

// ------------------------------------------------------------------------------------------------ tiled DWT design
size_t feds_dwt_tiles_private_bytes(int w, int h, int c) { return (dct_dims_ok(w, h) && chan_ok(c)) ? tiles_plan(w, h, c).priv_b : 0; }
size_t feds_dwt_tiles_public_bytes(int w, int h, int c) { return (dct_dims_ok(w, h) && chan_ok(c)) ? tiles_plan(w, h, c).pub_b : 0; }
size_t feds_dwt_tiles_workspace_bytes(int w, int h, int c) { return (dct_dims_ok(w, h) && chan_ok(c)) ? tiles_plan(w, h, c).per_image : 0; }

feds_status feds_fragment_dwt_tiles(const uint8_t *d_image, int w, int h, int c, const uint8_t key[16], const uint8_t nonce[16],
                                    uint8_t *d_private, uint8_t *d_public, uint8_t *d_digests, void *d_workspace, size_t workspace_bytes,
                                    feds_stream_t stream) {
    if (!nonce) return check_tiles_args(1, w, h, c) != FEDS_OK ? check_tiles_args(1, w, h, c) : FEDS_ERR_NULL_POINTER;
    return fragment_tiles_impl(d_image, 1, (size_t)(w > 0 ? w : 0) * (h > 0 ? h : 0) * (c > 0 ? c : 0), w, h, c, key, nonce, nullptr, d_private,
                               feds_dwt_tiles_private_bytes(w, h, c), d_public, feds_dwt_tiles_public_bytes(w, h, c), d_digests, d_workspace,
                               workspace_bytes, stream);
}
feds_status feds_fragment_dwt_tiles_batch(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c,
                                          const uint8_t key[16], const uint8_t *d_nonces, uint8_t *d_private, size_t private_stride,
                                          uint8_t *d_public, size_t public_stride, uint8_t *d_digests, void *d_workspace,
                                          size_t workspace_bytes, feds_stream_t stream) {
    if (!d_nonces) return check_tiles_args(n_images, w, h, c) != FEDS_OK ? check_tiles_args(n_images, w, h, c) : FEDS_ERR_NULL_POINTER;
    return fragment_tiles_impl(d_images, n_images, image_stride, w, h, c, key, nullptr, d_nonces, d_private, private_stride, d_public,
                               public_stride, d_digests, d_workspace, workspace_bytes, stream);
}
feds_status feds_defragment_dwt_tiles(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, const uint8_t key[16],
                                      const uint8_t nonce[16], const uint8_t *d_expected_digests, uint8_t *d_image_out,
                                      uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes, feds_stream_t stream) {
    if (!nonce) return check_tiles_args(1, w, h, c) != FEDS_OK ? check_tiles_args(1, w, h, c) : FEDS_ERR_NULL_POINTER;
    return defragment_tiles_impl(d_private, feds_dwt_tiles_private_bytes(w, h, c), d_public, feds_dwt_tiles_public_bytes(w, h, c), 1, w, h, c, key,
                                 nonce, nullptr, d_expected_digests, d_image_out, (size_t)(w > 0 ? w : 0) * (h > 0 ? h : 0) * (c > 0 ? c : 0),
                                 d_verify_flags, d_workspace, workspace_bytes, stream);
}
feds_status feds_defragment_dwt_tiles_batch(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                            int n_images, int w, int h, int c, const uint8_t key[16], const uint8_t *d_nonces,
                                            const uint8_t *d_expected_digests, uint8_t *d_images_out, size_t image_stride,
                                            uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes, feds_stream_t stream) {
    if (!d_nonces) return check_tiles_args(n_images, w, h, c) != FEDS_OK ? check_tiles_args(n_images, w, h, c) : FEDS_ERR_NULL_POINTER;
    return defragment_tiles_impl(d_private, private_stride, d_public, public_stride, n_images, w, h, c, key, nullptr, d_nonces,
                                 d_expected_digests, d_images_out, image_stride, d_verify_flags, d_workspace, workspace_bytes, stream);
}

// ------------------------------------------------------------------------------------------------ stream primitives
feds_status feds_aes128_ctr(const uint8_t *d_in, uint8_t *d_out, size_t n_bytes, const uint8_t key[16], const uint8_t nonce[16],
                            feds_stream_t stream) {
    if (!key || !nonce || (n_bytes && (!d_in || !d_out))) return FEDS_ERR_NULL_POINTER;
    if (misaligned(d_in) || misaligned(d_out)) return FEDS_ERR_MISALIGNED;
    return launch_aes_ctr(d_in, 0, d_out, 0, n_bytes, 1, key, nonce, nullptr, stream);
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
    if (nl == 0) return launch_empty_root(d_root, stream);  // SHA-256("")
    uint8_t *ws = static_cast<uint8_t *>(d_workspace);
    const uint8_t *const data[2] = {d_data, nullptr};
    const size_t strides[2] = {0, 0};
    const unsigned long long nbytes[2] = {n_bytes, 0};
    const unsigned nls[2] = {nl, 0};
    uint8_t *const out[2] = {nl > 1 ? ws : d_root, nullptr};
    const feds_status st = launch_stream_leaves(data, strides, nbytes, nls, out, 1, false, stream);
    if (st != FEDS_OK) return st;
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
    if (images_per_chunk < 1 || n_streams < 1 || (flags & ~DCT_FLAGS)) return FEDS_ERR_BAD_PARAM;
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
    if (images_per_chunk < 1 || n_streams < 1 || (flags & ~DCT_FLAGS)) return FEDS_ERR_BAD_PARAM;
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
unsigned long long feds_debug_launch_count(void) { return t_launches; }

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

void feds_debug_strong_basis_host(int32_t out[64 * 64]) { strong_basis_host(out); }

void feds_debug_zigzag_host(int out[64]) {
    for (int z = 0; z < 64; ++z) out[z] = h_zigzag.pos[z];
}

}  // extern "C"
