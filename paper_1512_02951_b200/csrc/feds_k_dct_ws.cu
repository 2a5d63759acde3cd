// feds_k_dct_ws.cu — launchers of the warp-specialised fused DCT kernels (feds_dct_ws.cuh).
#include <algorithm>

#include "feds_dct_ws.cuh"
#include "feds_host.h"

namespace feds {

// whole 8-block leaves (every stream is a whole number of 64-byte chunks) and 8/16-byte runs
bool dct_ws_supported(const DctParams &p, int c) {
    (void)c;
    return (p.nbc % G_BLOCKS) == 0 && dct_vec_width(p.k) >= 2;
}

namespace {
template <int C, int V, bool FRAGMENT>
feds_status go(const DctParams &p, cudaStream_t stream) {
    static size_t smem_set = 0;
    auto kernel = dct_ws_kernel<C, V, FRAGMENT>;
    const size_t smem = ws_smem_bytes();
    feds_status s = set_smem_once(kernel, smem, smem_set);
    if (s != FEDS_OK) return s;
    const unsigned units = (unsigned)WsShape<C>::UNITS;
    const unsigned grid = std::min<unsigned>((p.ws_n_sg + units - 1) / units, (unsigned)sm_count());
    if (prof_start_event()) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    kernel<<<grid, WS_THREADS, smem, stream>>>(p);
    if (prof_stop_event()) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}
template <bool FRAGMENT>
feds_status dispatch(const DctParams &p, int c, cudaStream_t stream) {
    if (!dct_ws_supported(p, c)) return FEDS_ERR_BAD_PARAM;
    const int V = dct_vec_width(p.k);
#define FEDS_V(CC) (V == 4 ? go<CC, 4, FRAGMENT>(p, stream) : go<CC, 2, FRAGMENT>(p, stream))
    return c == 1 ? FEDS_V(1) : c == 3 ? FEDS_V(3) : FEDS_V(4);
#undef FEDS_V
}
}  // namespace

feds_status launch_fragment_ws(const DctParams &p, int c, cudaStream_t stream) { return dispatch<true>(p, c, stream); }
feds_status launch_defragment_ws(const DctParams &p, int c, cudaStream_t stream) { return dispatch<false>(p, c, stream); }

}  // namespace feds
