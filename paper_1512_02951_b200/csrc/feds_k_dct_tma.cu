// feds_k_dct_tma.cu — launchers of the bulk-copy (TMA) tile kernels of the digest-free DCT path (feds_dct_tma.cuh).
#include <algorithm>

#include "feds_dct_tma.cuh"
#include "feds_host.h"

namespace feds {

// all runs and pixel-row segments 16-byte multiples at 16-byte aligned addresses; a tile spans at most two block rows
bool dct_tma_supported(const DctParams &p, int c) {
    return c == 1 ? tma_shape_ok<1>(p.w) : c == 3 ? tma_shape_ok<3>(p.w) : tma_shape_ok<4>(p.w);
}

namespace {
template <int C, typename Kernel>
feds_status launch_tma(Kernel kernel, const DctParams &p, cudaStream_t stream, bool profile, size_t &smem_set) {
    using S = TmaShape<C>;
    const size_t smem = tma_smem_bytes<C>(p.k, S::GROUPS);
    feds_status s = set_smem_once(kernel, smem, smem_set);
    if (s != FEDS_OK) return s;
    const unsigned long long tiles = (unsigned long long)p.n_images * (((unsigned long long)p.nbr * p.nbc + S::TB - 1) / S::TB);
    const unsigned grid = (unsigned)std::min<unsigned long long>((tiles + S::GROUPS - 1) / S::GROUPS, (unsigned long long)sm_count());
    if (prof_start_event() && profile) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    kernel<<<grid, S::CTA, smem, stream>>>(p);
    if (prof_stop_event() && profile) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}
template <int C, int V> feds_status frag(const DctParams &p, cudaStream_t s, bool profile) {
    static size_t smem_set = 0;
    return launch_tma<C>(fragment_dct_tma_kernel<C, V>, p, s, profile, smem_set);
}
template <int C, int V> feds_status defrag(const DctParams &p, cudaStream_t s, bool profile) {
    static size_t smem_set = 0;
    return launch_tma<C>(defragment_dct_tma_kernel<C, V>, p, s, profile, smem_set);
}
}  // namespace

feds_status launch_fragment_tma(const DctParams &p, int c, cudaStream_t stream, bool profile) {
    const int V = dct_vec_width(p.k);
#define FEDS_V(CC) (V == 4 ? frag<CC, 4>(p, stream, profile) : V == 2 ? frag<CC, 2>(p, stream, profile) : frag<CC, 1>(p, stream, profile))
    return c == 1 ? FEDS_V(1) : c == 3 ? FEDS_V(3) : FEDS_V(4);
#undef FEDS_V
}
feds_status launch_defragment_tma(const DctParams &p, int c, cudaStream_t stream, bool profile) {
    const int V = dct_vec_width(p.k);
#define FEDS_V(CC) (V == 4 ? defrag<CC, 4>(p, stream, profile) : V == 2 ? defrag<CC, 2>(p, stream, profile) : defrag<CC, 1>(p, stream, profile))
    return c == 1 ? FEDS_V(1) : c == 3 ? FEDS_V(3) : FEDS_V(4);
#undef FEDS_V
}

}  // namespace feds
