// feds_host.h — host-side glue shared by the translation units of libfeds: the error macros, the per-thread profiling
// events, and the launchers each kernel file exports to feds_api.cu (which holds the C ABI, the argument checks and the
// workspace plans, and no kernel). One .cu per kernel family so that nvcc compiles them in parallel (build.py).
#pragma once
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

#include "../../include/feds.h"

namespace feds {

struct DctParams;
struct DwtLevelParams;

// defined in feds_api.cu
feds_status cuda_fail(cudaError_t e);
int sm_count();                       // SMs of the current device (the persistent kernels launch one CTA per SM)
cudaEvent_t prof_start_event();       // thread-local profiling hook (feds_profile_events), or nullptr
cudaEvent_t prof_stop_event();
void count_launch();                  // + 1 on the calling thread's launch counter

#define FEDS_CUDA(call)                                        \
    do {                                                       \
        cudaError_t e__ = (call);                              \
        if (e__ != cudaSuccess) return ::feds::cuda_fail(e__); \
    } while (0)
// every kernel launch of the library goes through this: error check + the per-thread launch counter (feds_debug_launch_count)
#define FEDS_LAUNCH_CHECK()             \
    do {                                \
        ::feds::count_launch();         \
        FEDS_CUDA(cudaGetLastError()); \
    } while (0)

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per process and kernel instantiation: the attribute is a property of
// the loaded function, not data state of a call (a `static bool` per instantiation; racing first calls set the same value).
template <typename K>
inline feds_status set_smem_once(K kernel, size_t bytes, size_t &done_bytes) {
    if (done_bytes >= bytes) return FEDS_OK;
    FEDS_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    done_bytes = bytes;
    return FEDS_OK;
}

// ---- feds_k_dct_fused.cu: warp-specialised fused kernels (steps 1-5 / 6-8 with verification): bulk-copy tile groups + hash warps
bool dct_fused_supported(const DctParams &p, int c);
feds_status launch_fragment_fused(const DctParams &p, int c, cudaStream_t stream);
feds_status launch_defragment_fused(const DctParams &p, int c, cudaStream_t stream);
// ---- feds_k_dct_tma.cu: the digest-free tile kernels on bulk asynchronous copies (w % 32 == 0 and at least one tile per block row)
bool dct_tma_supported(const DctParams &p, int c);
feds_status launch_fragment_tma(const DctParams &p, int c, cudaStream_t stream, bool profile);
feds_status launch_defragment_tma(const DctParams &p, int c, cudaStream_t stream, bool profile);
// ---- feds_k_dct_tile.cu: digest-free tile kernels and the registers-only leaf-hash kernel
// (`profile`: record the thread's profiling events, if any, around this kernel -- the caller sets it for the dominant kernel of the call)
feds_status launch_fragment_tile(const DctParams &p, int c, cudaStream_t stream, bool profile);
feds_status launch_defragment_tile(const DctParams &p, int c, cudaStream_t stream, bool profile);
feds_status launch_leaves_hash(const DctParams &p, int c, cudaStream_t stream, bool profile);
// ---- feds_k_dct_strong.cu: the report's strong level of protection (one thread per block; any image size)
feds_status launch_fragment_strong(const DctParams &p, int c, cudaStream_t stream, bool profile);
feds_status launch_defragment_strong(const DctParams &p, int c, cudaStream_t stream, bool profile);
void strong_basis_host(int32_t out[64 * 64]);
// packed integer storage (same translation unit): one thread per (leaf group, channel); `plain` = decrypted private fragments
feds_status launch_fragment_packed(const DctParams &p, int c, cudaStream_t stream, bool profile);
feds_status launch_defragment_packed(const DctParams &p, int c, const uint8_t *plain, size_t plain_stride, cudaStream_t stream, bool profile);
feds_status launch_packed_private_leaves(const DctParams &p, int c, cudaStream_t stream);
// ---- feds_k_dwt_tiles.cu: the report's tiled DWT design (one thread per 8x8 tile; the profiling events bracket the kernel)
feds_status launch_fragment_dwt_tiles(const DctParams &p, int c, cudaStream_t stream);
feds_status launch_defragment_dwt_tiles(const DctParams &p, int c, cudaStream_t stream);
// ---- feds_k_hash.cu: Merkle upper levels, stream leaves, AES-CTR stream, digest compare
// Every tree's scratch (all levels with more than one node above level 0) ends with TOP_CTRL_BYTES for merkle_top_kernel's counters.
constexpr size_t TOP_CTRL_BYTES = 256;
feds_status run_tree(const uint8_t *level0, unsigned n0, unsigned n_trees, uint8_t *scratch, uint8_t *roots, size_t root_stride,
                     int skip_odd, cudaStream_t stream);
feds_status run_two_trees(const uint8_t *l0a, unsigned na, uint8_t *sca, uint8_t *roota, const uint8_t *l0b, unsigned nb, uint8_t *scb,
                          uint8_t *rootb, unsigned n_trees, size_t root_stride, cudaStream_t stream);
// leaf digests of the two streams of n_images images: stream f of image i at d[f] + i * stride[f], digests at out[f] + (i * nl[f] + j) * 32
feds_status launch_stream_leaves(const uint8_t *const d[2], const size_t stride[2], const unsigned long long n_bytes[2], const unsigned nl[2],
                                 uint8_t *const out[2], unsigned n_images, bool profile, cudaStream_t stream);
// n_msgs independent CTR messages of n_bytes each (strides in bytes); nonce: host (single message) or device uint8[n_msgs][16]
feds_status launch_aes_ctr(const uint8_t *d_in, size_t in_stride, uint8_t *d_out, size_t out_stride, size_t n_bytes, unsigned n_msgs,
                           const uint8_t key[16], const uint8_t *nonce_host, const uint8_t *d_nonces, cudaStream_t stream);
feds_status launch_compare_digests(const uint8_t *computed, const uint8_t *expected, uint32_t *flags, int n_images, cudaStream_t stream);
feds_status launch_empty_public_roots(uint8_t *digests, int n_images, cudaStream_t stream);
feds_status launch_empty_root(uint8_t *root, cudaStream_t stream);
// ---- feds_k_dwt.cu: one 5/3 level per launch; `tiled` forces the shared-memory tile kernels (FEDS_FLAG_DWT_TILED)
feds_status launch_dwt_fwd_level(DwtLevelParams &p, bool first, int c_img, int n_images, bool tiled, cudaStream_t stream);
feds_status launch_dwt_inv_level(DwtLevelParams &p, bool last, int c_img, int n_images, bool tiled, cudaStream_t stream);

}  // namespace feds
