// feds_k_dct_fused.cu — launcher of the thread-per-leaf fused fragment kernel (feds_dct.cuh; steps 1-5, V in {2, 4}).
#include <algorithm>

#include "feds_dct.cuh"
#include "feds_host.h"

namespace feds {

namespace {
template <typename Kernel>
feds_status launch_dct(Kernel kernel, const DctParams &p, cudaStream_t stream, size_t &smem_set) {
    // persistent: one CTA per SM, its warps stride over the leaf groups. 16 warps unless their slots exceed the SM's
    // shared memory (k >= 32: the padding slack grows), then 8.
    int threads = DCT_THREADS;
    size_t smem = (size_t)(AES_TABLE_WORDS + threads * p.slot_stride) * 4;
    if (smem > DCT_SMEM_MAX) { threads = 256; smem = (size_t)(AES_TABLE_WORDS + threads * p.slot_stride) * 4; }
    const unsigned grid = std::min<unsigned>(p.n_groups, (unsigned)sm_count());
    feds_status s = set_smem_once(kernel, DCT_SMEM_MAX, smem_set);
    if (s != FEDS_OK) return s;
    if (prof_start_event()) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    kernel<<<grid, threads, smem, stream>>>(p);
    if (prof_stop_event()) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}
template <int C, int V>
feds_status go(const DctParams &p, cudaStream_t s) {
    static size_t smem_set = 0;
    return launch_dct(fragment_dct_kernel<C, V>, p, s, smem_set);
}
}  // namespace

// the fused kernel exists for V = 4 and V = 2 only
feds_status launch_fragment_fused(const DctParams &p, int c, cudaStream_t stream) {
    const int V = dct_vec_width(p.k);
#define FEDS_V(CC) (V == 4 ? go<CC, 4>(p, stream) : go<CC, 2>(p, stream))
    return c == 1 ? FEDS_V(1) : c == 3 ? FEDS_V(3) : FEDS_V(4);
#undef FEDS_V
}

}  // namespace feds
