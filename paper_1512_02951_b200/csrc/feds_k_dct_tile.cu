// feds_k_dct_tile.cu — launchers of the digest-free tile kernels and the registers-only leaf-hash kernel (feds_dct_tile.cuh).
#include <algorithm>

#include "feds_dct_tile.cuh"
#include "feds_host.h"

namespace feds {

namespace {
// digest-free path: one persistent CTA per SM, GROUPS tile groups inside it
template <int C, typename Kernel>
feds_status launch_dct_tile(Kernel kernel, const DctParams &p, cudaStream_t stream, bool profile, size_t &smem_set) {
    constexpr int TB = TileShape<C>::TB, GROUPS = TileShape<C>::GROUPS;
    const size_t smem = tile_smem_bytes<C>(p.k);
    feds_status s = set_smem_once(kernel, smem, smem_set);
    if (s != FEDS_OK) return s;
    const unsigned long long tiles = (unsigned long long)p.n_images * p.nbr * ((p.nbc + TB - 1) / TB);
    const unsigned grid = (unsigned)std::min<unsigned long long>((tiles + GROUPS - 1) / GROUPS, (unsigned long long)sm_count());
    if (prof_start_event() && profile) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    kernel<<<grid, TileShape<C>::CTA, smem, stream>>>(p);
    if (prof_stop_event() && profile) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}
template <int C, int V> feds_status frag(const DctParams &p, cudaStream_t s, bool profile) {
    static size_t smem_set = 0;
    return launch_dct_tile<C>(fragment_dct_tile_kernel<C, V>, p, s, profile, smem_set);
}
template <int C, int V> feds_status defrag(const DctParams &p, cudaStream_t s, bool profile) {
    static size_t smem_set = 0;
    return launch_dct_tile<C>(defragment_dct_tile_kernel<C, V>, p, s, profile, smem_set);
}
}  // namespace

feds_status launch_fragment_tile(const DctParams &p, int c, cudaStream_t stream, bool profile) {
    if (!p.generic_tiles && dct_tma_supported(p, c)) return launch_fragment_tma(p, c, stream, profile);
    const int V = dct_vec_width(p.k);
#define FEDS_V(CC) (V == 4 ? frag<CC, 4>(p, stream, profile) : V == 2 ? frag<CC, 2>(p, stream, profile) : frag<CC, 1>(p, stream, profile))
    return c == 1 ? FEDS_V(1) : c == 3 ? FEDS_V(3) : FEDS_V(4);
#undef FEDS_V
}
feds_status launch_defragment_tile(const DctParams &p, int c, cudaStream_t stream, bool profile) {
    if (!p.generic_tiles && dct_tma_supported(p, c)) return launch_defragment_tma(p, c, stream, profile);
    const int V = dct_vec_width(p.k);
#define FEDS_V(CC) (V == 4 ? defrag<CC, 4>(p, stream, profile) : V == 2 ? defrag<CC, 2>(p, stream, profile) : defrag<CC, 1>(p, stream, profile))
    return c == 1 ? FEDS_V(1) : c == 3 ? FEDS_V(3) : FEDS_V(4);
#undef FEDS_V
}

// leaf digests of fragments as they lie in memory: the verification half of a verified defragment
feds_status launch_leaves_hash(const DctParams &p, int c, cudaStream_t stream, bool profile) {
    const unsigned long long threads = 2 * p.total_leaves;
    if (prof_start_event() && profile) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    if (p.total_leaves <= COOP_MAX_LEAVES) {   // few leaves: a warp per public leaf shortens the chain of dependent compressions
        static size_t smem_set[3] = {0, 0, 0};
        const unsigned long long cwarps = p.total_leaves + (p.total_leaves + 31) / 32;   // public leaves + private leaves by 32
        const unsigned cgrid = (unsigned)((cwarps + COOP_WARPS - 1) / COOP_WARPS);
        feds_status s = FEDS_OK;
        if (c == 1) { s = set_smem_once(dct_leaves_hash_coop_kernel<1>, COOP_SMEM_BYTES, smem_set[0]); if (s == FEDS_OK) dct_leaves_hash_coop_kernel<1><<<cgrid, COOP_WARPS * 32, COOP_SMEM_BYTES, stream>>>(p); }
        else if (c == 3) { s = set_smem_once(dct_leaves_hash_coop_kernel<3>, COOP_SMEM_BYTES, smem_set[1]); if (s == FEDS_OK) dct_leaves_hash_coop_kernel<3><<<cgrid, COOP_WARPS * 32, COOP_SMEM_BYTES, stream>>>(p); }
        else { s = set_smem_once(dct_leaves_hash_coop_kernel<4>, COOP_SMEM_BYTES, smem_set[2]); if (s == FEDS_OK) dct_leaves_hash_coop_kernel<4><<<cgrid, COOP_WARPS * 32, COOP_SMEM_BYTES, stream>>>(p); }
        if (s != FEDS_OK) return s;
        if (prof_stop_event() && profile) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
        FEDS_LAUNCH_CHECK();
        return FEDS_OK;
    }
    const unsigned grid = (unsigned)((threads + LEAFHASH_THREADS - 1) / LEAFHASH_THREADS);
    if (c == 1) dct_leaves_hash_kernel<1><<<grid, LEAFHASH_THREADS, 0, stream>>>(p);
    else if (c == 3) dct_leaves_hash_kernel<3><<<grid, LEAFHASH_THREADS, 0, stream>>>(p);
    else dct_leaves_hash_kernel<4><<<grid, LEAFHASH_THREADS, 0, stream>>>(p);
    if (prof_stop_event() && profile) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

}  // namespace feds
