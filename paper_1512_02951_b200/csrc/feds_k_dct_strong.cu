// feds_k_dct_strong.cu — launchers of the strong-level kernels (feds_dct_strong.cuh; PAPER.md 6.3.2) and of the packed-storage kernels
// (feds_dct_packed.cuh and, on bulk-copy tile groups, feds_dct_packed_tile.cuh; PAPER.md 6.4.3), which share the fixed-point basis table.
#include <algorithm>

#include "feds_dct_packed_tile.cuh"
#include "feds_host.h"

namespace feds {

namespace {
constexpr size_t STRONG_SMEM = (size_t)(AES_TABLE_WORDS + 64 * STRONG_THREADS) * 4;
constexpr StrongBasis h_strong_basis = make_strong_basis();
}  // namespace

void strong_basis_host(int32_t out[64 * 64]) {
    for (int i = 0; i < 64 * 64; ++i) out[i] = h_strong_basis.B[i];
}

feds_status launch_fragment_strong(const DctParams &p, int c, cudaStream_t stream, bool profile) {
    const unsigned long long threads = (unsigned long long)p.n_images * c * p.nbr * p.nbc;
    const unsigned grid = (unsigned)((threads + STRONG_THREADS - 1) / STRONG_THREADS);
    if (prof_start_event() && profile) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    // measured on the cfg3 batch: the pruned-transform form wins up to k = 7 (k = 3: 8.12 -> 7.37 ms, k = 5: 8.89 -> 8.14), is level at k = 9
#define FEDS_S(CC) { if (p.k < 4) fragment_dct_strong_kernel<CC, 4><<<grid, STRONG_THREADS, STRONG_SMEM, stream>>>(p); \
                     else if (p.k < 8) fragment_dct_strong_kernel<CC, 8><<<grid, STRONG_THREADS, STRONG_SMEM, stream>>>(p); \
                     else fragment_dct_strong_kernel<CC, 64><<<grid, STRONG_THREADS, STRONG_SMEM, stream>>>(p); }
    if (c == 1) FEDS_S(1) else if (c == 3) FEDS_S(3) else FEDS_S(4)
#undef FEDS_S
    if (prof_stop_event() && profile) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

feds_status launch_defragment_strong(const DctParams &p, int c, cudaStream_t stream, bool profile) {
    const unsigned long long threads = (unsigned long long)p.n_images * c * p.nbr * p.nbc;
    const unsigned grid = (unsigned)((threads + STRONG_THREADS - 1) / STRONG_THREADS);
    if (prof_start_event() && profile) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    // the inverse has no transform to prune: the unrolled accumulators win only for k <= 3 (7.58 -> 7.37 ms; k = 5: 8.37 -> 8.58)
#define FEDS_S(CC) { if (p.k < 4) defragment_dct_strong_kernel<CC, 4><<<grid, STRONG_THREADS, STRONG_SMEM, stream>>>(p); \
                     else defragment_dct_strong_kernel<CC, 64><<<grid, STRONG_THREADS, STRONG_SMEM, stream>>>(p); }
    if (c == 1) FEDS_S(1) else if (c == 3) FEDS_S(3) else FEDS_S(4)
#undef FEDS_S
    if (prof_stop_event() && profile) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

// ---- packed integer storage: bulk-copy tile groups (feds_dct_packed_tile.cuh) where the shape allows, else one thread per
// (leaf group, channel)
namespace {
template <int C, typename Kernel, typename... Extra>
feds_status launch_packed_tile(Kernel kernel, size_t &smem_set, const DctParams &p, cudaStream_t stream, bool profile, Extra... extra) {
    using S = TmaShape<C>;
    using PS = PackedTileShape<C>;
    const size_t smem = packed_tile_smem_bytes<C>();
    feds_status s = set_smem_once(kernel, smem, smem_set);
    if (s != FEDS_OK) return s;
    const unsigned long long tiles = (unsigned long long)p.n_images * (((unsigned long long)p.nbr * p.nbc + S::TB - 1) / S::TB);
    const unsigned grid = (unsigned)std::min<unsigned long long>((tiles + PS::GROUPS - 1) / PS::GROUPS, (unsigned long long)sm_count());
    if (prof_start_event() && profile) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    kernel<<<grid, PS::CTA, smem, stream>>>(p, extra...);
    if (prof_stop_event() && profile) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}
bool packed_tile_supported(const DctParams &p, int c) {
    if (p.generic_tiles) return false;
    return c == 1 ? packed_tile_ok<1>(p.w, p.k) : c == 3 ? packed_tile_ok<3>(p.w, p.k) : packed_tile_ok<4>(p.w, p.k);
}
}  // namespace

feds_status launch_fragment_packed(const DctParams &p, int c, cudaStream_t stream, bool profile) {
    if (packed_tile_supported(p, c)) {
#define FEDS_PT(CC, PM) { static size_t set = 0; return launch_packed_tile<CC>(fragment_dct_packed_tile_kernel<CC, PM>, set, p, stream, profile); }
#define FEDS_PT_P(CC) { if (p.k < 4) FEDS_PT(CC, 4) else if (p.k < 6) FEDS_PT(CC, 6) else if (p.k < 8) FEDS_PT(CC, 8) else FEDS_PT(CC, 16) }
        if (c == 1) FEDS_PT_P(1) else if (c == 3) FEDS_PT_P(3) else FEDS_PT_P(4)
#undef FEDS_PT_P
#undef FEDS_PT
    }
    const unsigned long long threads = (unsigned long long)p.n_images * c * p.nbr * p.nlr;
    const unsigned grid = (unsigned)((threads + PACKED_THREADS - 1) / PACKED_THREADS);
    const size_t smem = (size_t)64 * PACKED_THREADS * 4;
    if (prof_start_event() && profile) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    if (c == 1) fragment_dct_packed_kernel<1><<<grid, PACKED_THREADS, smem, stream>>>(p);
    else if (c == 3) fragment_dct_packed_kernel<3><<<grid, PACKED_THREADS, smem, stream>>>(p);
    else fragment_dct_packed_kernel<4><<<grid, PACKED_THREADS, smem, stream>>>(p);
    if (prof_stop_event() && profile) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}
feds_status launch_defragment_packed(const DctParams &p, int c, const uint8_t *plain, size_t plain_stride, cudaStream_t stream, bool profile) {
    if (packed_tile_supported(p, c)) {
#define FEDS_PT(CC, PM) { static size_t set = 0; return launch_packed_tile<CC>(defragment_dct_packed_tile_kernel<CC, PM>, set, p, stream, profile, plain, plain_stride); }
#define FEDS_PT_P(CC) { if (p.k < 4) FEDS_PT(CC, 4) else if (p.k < 6) FEDS_PT(CC, 6) else if (p.k < 8) FEDS_PT(CC, 8) else FEDS_PT(CC, 16) }
        if (c == 1) FEDS_PT_P(1) else if (c == 3) FEDS_PT_P(3) else FEDS_PT_P(4)
#undef FEDS_PT_P
#undef FEDS_PT
    }
    const unsigned long long threads = (unsigned long long)p.n_images * c * p.nbr * p.nlr;
    const unsigned grid = (unsigned)((threads + PACKED_THREADS - 1) / PACKED_THREADS);
    const size_t smem = (size_t)64 * PACKED_THREADS * 4;
    if (prof_start_event() && profile) FEDS_CUDA(cudaEventRecord(prof_start_event(), stream));
    if (c == 1) defragment_dct_packed_kernel<1><<<grid, PACKED_THREADS, smem, stream>>>(p, plain, plain_stride);
    else if (c == 3) defragment_dct_packed_kernel<3><<<grid, PACKED_THREADS, smem, stream>>>(p, plain, plain_stride);
    else defragment_dct_packed_kernel<4><<<grid, PACKED_THREADS, smem, stream>>>(p, plain, plain_stride);
    if (prof_stop_event() && profile) FEDS_CUDA(cudaEventRecord(prof_stop_event(), stream));
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}
feds_status launch_packed_private_leaves(const DctParams &p, int c, cudaStream_t stream) {
    const unsigned long long threads = (unsigned long long)p.n_images * c * p.nbr * p.nlr;
    packed_private_leaves_kernel<<<(unsigned)((threads + PACKED_THREADS - 1) / PACKED_THREADS), PACKED_THREADS, 0, stream>>>(p, c);
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

}  // namespace feds
