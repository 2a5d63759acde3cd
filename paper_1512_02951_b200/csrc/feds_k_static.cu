// feds_k_static.cu — feds_sha256_merkle_static: the stream Merkle digest (step 5 on a byte stream) for callers
// that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).
//
// feds_sha256_merkle needs a caller-provided workspace for the leaf digests and the inner levels of the tree. Here that
// workspace is a file-scope array in device memory: every GPU that loads the library holds FEDS_STATIC_SCRATCH_BYTES (1.125 MiB)
// of it until the process exits, and streams of up to FEDS_SHA256_MERKLE_STATIC_MAX_BYTES (64 MiB = 32,768 leaves) fit. The
// kernels are the ones feds_sha256_merkle launches (stream_leaves_kernel / its cooperative form, merkle_level_kernel, the tree
// top): the call only supplies the scratch pointer, so the root is the same 32 bytes.
//
// In host code the NAME of a __device__ array is a host-side stand-in, not a device address (a kernel given it would fault, or on
// a system where the GPU reaches host memory, quietly use the wrong bytes): the address comes from cudaGetSymbolAddress, asked
// once per device with that device current, in this translation unit, and is what the kernels receive.
//
// All calls on one device share the array and it keeps the last call's contents. Nothing in it needs to start at zero except
// the arrival counters of the spread-out tree top, which that path clears with a memset node in front of its kernel on every call
// (feds_k_hash.cu); every digest slot a call reads it has written first. Two calls that overlap on the GPU (different streams
// without an ordering between them) race on the array: order them, or use feds_sha256_merkle with a workspace per call.
#include <atomic>

#include "feds_host.h"

namespace feds {
namespace {

constexpr size_t FEDS_STATIC_SCRATCH_BYTES = (size_t)1152 << 10;
static __device__ __align__(256) uint8_t g_static_scratch[FEDS_STATIC_SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;
std::atomic<uint8_t *> g_scratch_ptr[MAX_DEVICES];   // device address of g_static_scratch per device (racing first calls store the same value)

// the array's address on the CURRENT device
feds_status static_scratch(uint8_t **out) {
    int dev = 0;
    FEDS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return FEDS_ERR_BAD_PARAM;
    uint8_t *p = g_scratch_ptr[dev].load(std::memory_order_acquire);
    if (!p) {
        FEDS_CUDA(cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_static_scratch));
        if (!p) return FEDS_ERR_CUDA;
        g_scratch_ptr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return FEDS_OK;
}

}  // namespace
}  // namespace feds

extern "C" {

size_t feds_sha256_merkle_static_max_bytes(void) { return (size_t)64 << 20; }

feds_status feds_sha256_merkle_static(const uint8_t *d_data, size_t n_bytes, uint8_t *d_root, feds_stream_t stream) {
    if (!d_root || (n_bytes && !d_data)) return FEDS_ERR_NULL_POINTER;
    if (n_bytes > feds_sha256_merkle_static_max_bytes()) return FEDS_ERR_BAD_PARAM;   // beyond the static scratch: use feds_sha256_merkle
    if (feds_sha256_merkle_workspace_bytes(n_bytes) > feds::FEDS_STATIC_SCRATCH_BYTES) return FEDS_ERR_WORKSPACE_TOO_SMALL;
    uint8_t *scratch = nullptr;
    const feds_status st = feds::static_scratch(&scratch);
    if (st != FEDS_OK) return st;
    return feds_sha256_merkle(d_data, n_bytes, d_root, scratch, feds::FEDS_STATIC_SCRATCH_BYTES, stream);
}

}  // extern "C"
