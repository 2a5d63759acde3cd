// feds_k_dct_fused.cu — launchers of the warp-specialised fused DCT kernels with digests (feds_dct_fused.cuh).
#include <algorithm>

#include "feds_dct_fused.cuh"
#include "feds_host.h"

#ifndef FU_HW
#define FU_HW 16   // hash warps per CTA (tile warps: 8)
#endif

namespace feds {

bool dct_fused_supported(const DctParams &p, int c) {
    return c == 1 ? fu_shape_ok<1>(p.w) : c == 3 ? fu_shape_ok<3>(p.w) : fu_shape_ok<4>(p.w);
}

namespace {
template <int C, int V, bool FRAGMENT>
feds_status go(const DctParams &p, cudaStream_t stream) {
    using F = FuShape<C, FU_HW>;
    static size_t smem_set = 0;
    auto kernel = dct_fused_kernel<C, V, FU_HW, FRAGMENT>;
    const size_t smem = fu_smem_bytes<C>(p.k, F::NP);
    feds_status s = set_smem_once(kernel, smem, smem_set);
    if (s != FEDS_OK) return s;
    const unsigned long long plane = (unsigned long long)p.nbr * p.nbc;
    const unsigned long long units = (unsigned long long)p.n_images * ((plane + FU_UNIT_BLOCKS - 1) / FU_UNIT_BLOCKS);
    const unsigned grid = (unsigned)std::min<unsigned long long>(units, (unsigned long long)sm_count());
    if (prof_start_event()) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    kernel<<<grid, F::THREADS, smem, stream>>>(p);
    if (prof_stop_event()) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}
template <bool FRAGMENT>
feds_status dispatch(const DctParams &p, int c, cudaStream_t stream) {
    if (!dct_fused_supported(p, c)) return FEDS_ERR_BAD_PARAM;
    const int V = dct_vec_width(p.k);
#define FEDS_V(CC) (V == 4 ? go<CC, 4, FRAGMENT>(p, stream) : V == 2 ? go<CC, 2, FRAGMENT>(p, stream) : go<CC, 1, FRAGMENT>(p, stream))
    return c == 1 ? FEDS_V(1) : c == 3 ? FEDS_V(3) : FEDS_V(4);
#undef FEDS_V
}
}  // namespace

feds_status launch_fragment_fused(const DctParams &p, int c, cudaStream_t stream) { return dispatch<true>(p, c, stream); }
feds_status launch_defragment_fused(const DctParams &p, int c, cudaStream_t stream) { return dispatch<false>(p, c, stream); }

}  // namespace feds
