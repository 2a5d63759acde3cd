// feds_k_dwt_tiles.cu — launchers of the tiled DWT design's kernels (feds_dwt_tiles.cuh; PAPER.md 6.9.3-6.9.4).
#include "feds_dwt_tiles.cuh"
#include "feds_host.h"

namespace feds {

feds_status launch_fragment_dwt_tiles(const DctParams &p, int c, cudaStream_t stream) {
    const unsigned long long threads = (unsigned long long)p.n_images * c * p.nbr * p.nbc;
    const unsigned grid = (unsigned)((threads + TILES_THREADS - 1) / TILES_THREADS);
    if (prof_start_event()) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    if (c == 1) fragment_dwt_tiles_kernel<1><<<grid, TILES_THREADS, 0, stream>>>(p);
    else if (c == 3) fragment_dwt_tiles_kernel<3><<<grid, TILES_THREADS, 0, stream>>>(p);
    else fragment_dwt_tiles_kernel<4><<<grid, TILES_THREADS, 0, stream>>>(p);
    if (prof_stop_event()) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}
feds_status launch_defragment_dwt_tiles(const DctParams &p, int c, cudaStream_t stream) {
    const unsigned long long threads = (unsigned long long)p.n_images * c * p.nbr * p.nbc;
    const unsigned grid = (unsigned)((threads + TILES_THREADS - 1) / TILES_THREADS);
    if (prof_start_event()) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    if (c == 1) defragment_dwt_tiles_kernel<1><<<grid, TILES_THREADS, 0, stream>>>(p);
    else if (c == 3) defragment_dwt_tiles_kernel<3><<<grid, TILES_THREADS, 0, stream>>>(p);
    else defragment_dwt_tiles_kernel<4><<<grid, TILES_THREADS, 0, stream>>>(p);
    if (prof_stop_event()) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

}  // namespace feds
