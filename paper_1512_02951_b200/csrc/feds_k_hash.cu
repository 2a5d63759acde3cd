// feds_k_hash.cu — launchers of the stream-level kernels (feds_hash.cuh): Merkle upper levels, SHA-256 of fixed-size
// stream leaves, AES-128-CTR over a byte stream, digest compare.
#include <algorithm>

#include "feds_hash.cuh"
#include "feds_host.h"

namespace feds {

namespace {
constexpr AesTables h_aes = make_aes_tables();

void nonce_to_be(const uint8_t nonce[16], uint32_t out[4]) {
    for (int i = 0; i < 4; ++i)
        out[i] = ((uint32_t)nonce[4 * i] << 24) | ((uint32_t)nonce[4 * i + 1] << 16) | ((uint32_t)nonce[4 * i + 2] << 8) | nonce[4 * i + 3];
}

feds_status tail_smem_once() {
    static size_t smem_set = 0;
    return set_smem_once(merkle_tail_kernel, TAIL_SMEM_BYTES, smem_set);
}

// the top of a few trees spread over the chip (merkle_top_kernel): pays when merkle_tail_kernel would hash TWO levels one node per
// thread, i.e. more than 64 nodes in the first (measured: 8192^2 DWT, 256 nodes, 56 -> 44 us; 512^2 DCT, 32 nodes, 33 -> 37 + the
// memset). `spare` = the end of the primary family's level storage (tree_bytes keeps TOP_CTRL_BYTES per tree)
bool top_pays(unsigned total_trees, unsigned na, unsigned nb) {
    const unsigned ma = (na + FANOUT - 1) / FANOUT, mb = (nb + FANOUT - 1) / FANOUT;
    return total_trees <= (unsigned)TOP_MAX_TREES && std::max(ma, mb) > 4u * FANOUT;
}
size_t top_levels_bytes(unsigned n, unsigned n_trees) {
    const unsigned m1 = (n + FANOUT - 1) / FANOUT, m2 = (m1 + FANOUT - 1) / FANOUT;
    return (size_t)n_trees * ((m1 > 1 ? m1 : 0) + (m2 > 1 ? m2 : 0)) * 32;
}
feds_status launch_top(MerkleLevelParams &mp, unsigned total_trees, uint8_t *spare, cudaStream_t stream) {
    static_assert(TOP_CTRL_BYTES >= 2 * TOP_CTRL_WORDS * 4, "the primary family's spare bytes hold the counters of both families");
    mp.ctrl = reinterpret_cast<unsigned *>(spare);
    FEDS_CUDA(cudaMemsetAsync(spare, 0, (size_t)total_trees * TOP_CTRL_WORDS * 4, stream));
    merkle_top_kernel<<<dim3(TOP_CTAS_PER_TREE, total_trees), TOP_THREADS, 0, stream>>>(mp);
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

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
}  // namespace

// Reduce level-0 digests [tree][n0][32] (tree stride = n0*32) to roots written at roots + tree*root_stride.
// `scratch` holds the intermediate levels. n_trees trees of identical shape.
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
        if (top_pays(n_trees, n, 0)) {
            mp.scratch = sc;
            return launch_top(mp, n_trees, sc + top_levels_bytes(n, n_trees), stream);
        }
        feds_status ts = tail_smem_once();
        if (ts != FEDS_OK) return ts;
        merkle_tail_kernel<<<n_trees, TAIL_THREADS, TAIL_SMEM_BYTES, stream>>>(mp);
        FEDS_LAUNCH_CHECK();
    }
    return FEDS_OK;
}

// two families of n_trees trees each, of different shapes (DWT private / public): wide levels separately, all tops in one
// launch. Level-0 digests [tree][n][32]; roots of family a at roota + tree * root_stride, of family b at rootb + tree * root_stride.
feds_status run_two_trees(const uint8_t *l0a, unsigned na, uint8_t *sca, uint8_t *roota, const uint8_t *l0b, unsigned nb, uint8_t *scb,
                          uint8_t *rootb, unsigned n_trees, size_t root_stride, cudaStream_t stream) {
    const uint8_t *ina = l0a, *inb = l0b;
    feds_status st = reduce_wide(ina, na, n_trees, sca, 0, stream);
    if (st != FEDS_OK) return st;
    st = reduce_wide(inb, nb, n_trees, scb, 0, stream);
    if (st != FEDS_OK) return st;
    if (na <= 1 && nb <= 1) return FEDS_OK;  // one-leaf trees: the leaf kernel already wrote the roots
    MerkleLevelParams mp{};
    mp.one = 1u; mp.n_out = 1;
    unsigned ctas = 0;
    uint8_t *spare = nullptr;
    if (na > 1) {
        mp.n_trees = n_trees; mp.in = ina; mp.n_in = na; mp.in_tree_stride = (size_t)na * 32; mp.out = roota; mp.out_tree_stride = root_stride;
        mp.scratch = sca; spare = sca + top_levels_bytes(na, n_trees);
        ctas = n_trees;
    }
    if (nb > 1) {
        if (ctas == 0) {
            mp.n_trees = n_trees; mp.in = inb; mp.n_in = nb; mp.in_tree_stride = (size_t)nb * 32; mp.out = rootb; mp.out_tree_stride = root_stride;
            mp.scratch = scb; spare = scb + top_levels_bytes(nb, n_trees);
        } else {
            mp.in2 = inb; mp.n_in2 = nb; mp.n_trees2 = n_trees; mp.in2_tree_stride = (size_t)nb * 32; mp.out2 = rootb; mp.out2_tree_stride = root_stride;
            mp.scratch2 = scb;
        }
        ctas += n_trees;
    }
    if (top_pays(ctas, na > 1 ? na : 0, nb > 1 ? nb : 0)) return launch_top(mp, ctas, spare, stream);
    feds_status ts = tail_smem_once();
    if (ts != FEDS_OK) return ts;
    merkle_tail_kernel<<<ctas, TAIL_THREADS, TAIL_SMEM_BYTES, stream>>>(mp);
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

// leaf digests of the two streams (private, public) of n_images images in one launch; a stream may be empty (nl == 0)
feds_status launch_stream_leaves(const uint8_t *const d[2], const size_t stride[2], const unsigned long long n_bytes[2], const unsigned nl[2],
                                 uint8_t *const out[2], unsigned n_images, bool profile, cudaStream_t stream) {
    StreamLeavesParams sp{};
    for (int f = 0; f < 2; ++f) {
        sp.data[f] = d[f]; sp.n_bytes[f] = n_bytes[f]; sp.n_leaves[f] = nl[f]; sp.out[f] = out[f]; sp.data_stride[f] = stride[f];
    }
    sp.n_images = n_images;
    sp.one = 1u;
    const unsigned long long total = (unsigned long long)(nl[0] + nl[1]) * n_images;
    if (total == 0) return FEDS_OK;
    if (profile && prof_start_event()) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    if (total <= STREAM_COOP_MAX) {   // few leaves: a warp per leaf shortens the chain of dependent compressions
        static size_t smem_set = 0;
        feds_status s = set_smem_once(stream_leaves_coop_kernel, STREAM_COOP_SMEM_BYTES, smem_set);
        if (s != FEDS_OK) return s;
        stream_leaves_coop_kernel<<<(unsigned)((total + STREAM_COOP_WARPS - 1) / STREAM_COOP_WARPS), STREAM_COOP_WARPS * 32, STREAM_COOP_SMEM_BYTES, stream>>>(sp);
    } else
    stream_leaves_kernel<<<(unsigned)((total + LEAF_THREADS - 1) / LEAF_THREADS), LEAF_THREADS, 0, stream>>>(sp);
    if (profile && prof_stop_event()) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

// AES-128-CTR of byte streams: the conflict-free 128 KB table layout pays once there are a few MB to encrypt
feds_status launch_aes_ctr(const uint8_t *d_in, size_t in_stride, uint8_t *d_out, size_t out_stride, size_t n_bytes, unsigned n_msgs,
                           const uint8_t key[16], const uint8_t *nonce_host, const uint8_t *d_nonces, cudaStream_t stream) {
    if (n_bytes == 0 || n_msgs == 0) return FEDS_OK;
    CtrParams cp{};
    cp.in = d_in; cp.out = d_out; cp.n_bytes = n_bytes; cp.in_stride = in_stride; cp.out_stride = out_stride; cp.n_msgs = n_msgs;
    cp.d_nonces = d_nonces;
    cp.c128 = 128u;
    if (nonce_host) nonce_to_be(nonce_host, cp.nonce_be);
    aes128_expand_key_host(key, cp.rk, h_aes);
    const unsigned long long nblk = ((n_bytes + 15) / 16) * n_msgs;
    const unsigned sms = (unsigned)sm_count();
    if ((unsigned long long)n_bytes * n_msgs >= ((size_t)4 << 20)) {
        const size_t smem = (size_t)AES_TABLE_WORDS * 32 * 4;
        static size_t smem_set = 0;
        feds_status st = set_smem_once(aes_ctr_stream_kernel<32>, smem, smem_set);
        if (st != FEDS_OK) return st;
        aes_ctr_stream_kernel<32><<<sms, AES_THREADS, smem, stream>>>(cp);
    } else {
        const unsigned want = (unsigned)((nblk + AES_THREADS - 1) / AES_THREADS);
        aes_ctr_stream_kernel<1><<<std::min(want, 2 * sms), AES_THREADS, (size_t)AES_TABLE_WORDS * 4, stream>>>(cp);
    }
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

feds_status launch_compare_digests(const uint8_t *computed, const uint8_t *expected, uint32_t *flags, int n_images, cudaStream_t stream) {
    compare_digests_kernel<<<(n_images + 127) / 128, 128, 0, stream>>>(computed, expected, flags, n_images);
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}
feds_status launch_empty_public_roots(uint8_t *digests, int n_images, cudaStream_t stream) {
    write_empty_public_root_kernel<<<(n_images + 127) / 128, 128, 0, stream>>>(digests, n_images);
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}
feds_status launch_empty_root(uint8_t *root, cudaStream_t stream) {
    write_empty_root_kernel<<<1, 32, 0, stream>>>(root);
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

}  // namespace feds
