/*
 * feds.h — C ABI of libfeds: selective-encryption fragmentation of 8-bit images on one B200 (sm_100a).
 *
 * Method: arXiv 1512.02951 section 6 ("P:n" = PAPER.md line n); byte format: DESIGN.md section 2.
 *
 * Conventions (all entry points)
 *   - `d_*` pointers are DEVICE pointers, 16-byte aligned; `key`/`nonce` (16 bytes each) are HOST pointers and are
 *     read before the call returns. `h_*` pointers (host-staged entry points only) are HOST pointers.
 *   - The caller owns every buffer. The library allocates nothing, keeps no global state, logs nothing.
 *   - All work is enqueued on `stream`; no call synchronises the device. Argument errors are returned before
 *     anything is enqueued; a failed launch returns FEDS_ERR_CUDA (see feds_last_cuda_error); asynchronous faults
 *     surface at the caller's next synchronisation, as with any CUDA library.
 *   - Input, fragments, workspace and output must not alias.
 *   - Image layout: uint8[H][W][C], interleaved, tight pitch, C in {1,3,4}; the transform runs per channel plane.
 *   - There is no CPU fallback anywhere in this library.
 */
#ifndef FEDS_H
#define FEDS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__CUDACC__) || defined(__CUDA_RUNTIME_API_H__) || defined(__DRIVER_TYPES_H__)
#include <cuda_runtime_api.h>
typedef cudaStream_t feds_stream_t;
typedef cudaEvent_t feds_event_t;
#else
typedef struct CUstream_st *feds_stream_t; /* identical to cudaStream_t */
typedef struct CUevent_st *feds_event_t;   /* identical to cudaEvent_t */
#endif

typedef enum {
    FEDS_OK = 0,
    FEDS_ERR_NULL_POINTER = 1,
    FEDS_ERR_BAD_DIMS = 2,            /* w,h <= 0; not a multiple of 8 (DCT) / of 2^levels (DWT) */
    FEDS_ERR_BAD_PARAM = 3,           /* k not in [0,63]; levels not in [1,6]; channels not in {1,3,4}; n_images < 1; bad stride/flags */
    FEDS_ERR_WORKSPACE_TOO_SMALL = 4,
    FEDS_ERR_CUDA = 5,                /* a launch or copy failed; cudaError_t kept for feds_last_cuda_error() */
    FEDS_ERR_MISALIGNED = 6           /* a device pointer or stride is not 16-byte aligned */
} feds_status;

/* Flags for the *_batch entry points. */
#define FEDS_FLAG_NONE 0u
#define FEDS_FLAG_NO_DIGEST 1u /* skip step 5 (SHA-256 Merkle digests): the report's own selective encryption (DCT + select + AES,
                                  P:488-494), HBM-bound. d_digests is not written; defragment does not verify. */
/* Route overrides (tests and profiling; results are byte-identical on every route). Without them the library picks the
 * route from the shape alone. A forced route that does not support the shape returns FEDS_ERR_BAD_PARAM. */
#define FEDS_FLAG_FORCE_FUSED 2u /* DCT with digests: the warp-specialised fused kernel (needs w % 64 == 0 and w >= 256, gray: w >= 512) */
#define FEDS_FLAG_FORCE_SPLIT 4u /* DCT with digests: digest-free tile kernel + leaf-hash kernel (what the library picks by itself) */
#define FEDS_FLAG_DWT_TILED 8u   /* DWT: the tiled shared-memory level kernels instead of the register-streaming ones */
#define FEDS_FLAG_GENERIC_TILES 16u /* DCT: the generic tile kernels (any w) even where the bulk-copy (TMA) tile kernels apply (w % 32 == 0) */

const char *feds_status_string(feds_status s);
int feds_last_cuda_error(void); /* cudaError_t of the most recent FEDS_ERR_CUDA on this thread, else 0 */

/* Frozen format constants: blocks per DCT leaf G, Merkle fan-out F, bytes per DWT leaf. */
void feds_merkle_params(int *g_blocks, int *fanout, int *dwt_leaf_bytes);

/* Fragment sizes in bytes for ONE image (DC + first k zigzag AC -> private; LL_L -> private).
 * Return 0 for invalid arguments. */
size_t feds_dct_private_bytes(int w, int h, int c, int k);       /* (w/8)(h/8) c (k+1) 4  */
size_t feds_dct_public_bytes(int w, int h, int c, int k);        /* (w/8)(h/8) c (63-k) 4 */
size_t feds_dwt_private_bytes(int w, int h, int c, int levels);  /* (w>>L)(h>>L) c 2      */
size_t feds_dwt_public_bytes(int w, int h, int c, int levels);   /* (w h - (w>>L)(h>>L)) c 2 */
/* Workspace bytes for ONE image (leaf digests + tree levels; DWT: also the intermediate LL planes).
 * A batch of n images needs n times this. */
size_t feds_workspace_bytes(int w, int h, int c, int k_or_levels, int is_dwt);

/*
 * feds_fragment_dct — steps 1-5 of the path (P:541-545 DCT 8x8, P:488-494 selection,
 * P:607 + P:1018 AES-128-CTR on the private part, BASELINE north_star SHA-256 digests).
 *   d_image    in : uint8[h][w][c]
 *   k          in : number of AC coefficients (zigzag order) that join the DC in the private fragment, 0..63
 *   key, nonce in : HOST, 16 bytes each; nonce = initial counter block T_0, T_i = (T_0 + i) mod 2^128 big-endian
 *   d_private  out: feds_dct_private_bytes() bytes: float32 LE [block][z = 0..k], AES-128-CTR ciphertext
 *   d_public   out: feds_dct_public_bytes() bytes: float32 LE [block][z = k+1..63], plaintext
 *   d_digests  out: 64 bytes: Merkle root of the private fragment (as stored) || root of the public fragment
 *   d_workspace   : >= feds_workspace_bytes(w,h,c,k,0) bytes of scratch
 */
feds_status feds_fragment_dct(const uint8_t *d_image, int w, int h, int c, int k, const uint8_t key[16],
                              const uint8_t nonce[16], uint8_t *d_private, uint8_t *d_public, uint8_t *d_digests,
                              void *d_workspace, size_t workspace_bytes, feds_stream_t stream);

/*
 * feds_defragment_dct — steps 6-8 (decrypt, reassemble, inverse transform; round to nearest, clamp).
 *   d_expected_digests in : 64 bytes or NULL. Non-NULL: the digests of the fragments as received are recomputed
 *                           and compared; d_verify_flags[0] = bit0 (private mismatch) | bit1 (public mismatch).
 *                           NULL: no verification, d_verify_flags is not written.
 *   d_image_out       out: uint8[h][w][c]; written regardless of the verification result.
 */
feds_status feds_defragment_dct(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int k,
                                const uint8_t key[16], const uint8_t nonce[16], const uint8_t *d_expected_digests,
                                uint8_t *d_image_out, uint32_t *d_verify_flags, void *d_workspace,
                                size_t workspace_bytes, feds_stream_t stream);

/*
 * feds_verify_dct — the integrity half of step 6 alone ("integrity requirement"; A8, A10): recomputes the
 * Merkle roots of the two fragments as they lie in memory and compares them with d_expected_digests (64 bytes per image).
 * Needs no key: the digests cover the stored bytes (ciphertext / plaintext coefficients), so whoever holds a fragment
 * can check it. d_verify_flags[i] = bit0 (private mismatch) | bit1 (public mismatch). Workspace as for feds_defragment_dct.
 * feds_verify_dct_batch: n_images fragments at the given byte strides (as feds_defragment_dct_batch).
 */
feds_status feds_verify_dct(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int k,
                            const uint8_t *d_expected_digests, uint32_t *d_verify_flags, void *d_workspace,
                            size_t workspace_bytes, feds_stream_t stream);
feds_status feds_verify_dct_batch(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public,
                                  size_t public_stride, int n_images, int w, int h, int c, int k,
                                  const uint8_t *d_expected_digests, uint32_t *d_verify_flags, void *d_workspace,
                                  size_t workspace_bytes, feds_stream_t stream);

/*
 * Strong level of protection (PAPER.md 6.3.2, Figure 8; byte format: DESIGN.md 2.3). Part 1 of every 8x8 block (DC +
 * first k zigzag AC, float32) is encrypted with AES-128-CTR exactly as by feds_fragment_dct; the public part of a block is its
 * 64 remainder pixels -- "the reverse DCT result of the rest DCT coefficients padded with zero", i.e. x minus the low-pass
 * image of Part 1, evaluated in exact fixed-point arithmetic and stored modulo 256 -- XORed with SHA-512(Part 1 of the block)
 * (one 512-bit string per block). Digests: the Merkle roots of the two fragments as stored, as everywhere else.
 *   d_public: feds_dct_strong_public_bytes(w,h,c) = w*h*c bytes, uint8 [block][64], blocks in the order of feds_fragment_dct.
 *   d_private, d_digests, workspace (feds_workspace_bytes(w,h,c,k,0)), key, nonce, errors: as feds_fragment_dct.
 * The inverse rebuilds the low-pass image and the keystream from the decrypted Part 1 and is exact (uint8 for uint8) by
 * construction. *_batch: n_images images at the given byte strides, per-image nonces on the device; flags: FEDS_FLAG_NO_DIGEST.
 */
size_t feds_dct_strong_public_bytes(int w, int h, int c);
feds_status feds_fragment_dct_strong(const uint8_t *d_image, int w, int h, int c, int k, const uint8_t key[16],
                                     const uint8_t nonce[16], uint8_t *d_private, uint8_t *d_public, uint8_t *d_digests,
                                     void *d_workspace, size_t workspace_bytes, feds_stream_t stream);
feds_status feds_defragment_dct_strong(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int k,
                                       const uint8_t key[16], const uint8_t nonce[16], const uint8_t *d_expected_digests,
                                       uint8_t *d_image_out, uint32_t *d_verify_flags, void *d_workspace,
                                       size_t workspace_bytes, feds_stream_t stream);
feds_status feds_fragment_dct_strong_batch(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c,
                                           int k, const uint8_t key[16], const uint8_t *d_nonces, uint8_t *d_private,
                                           size_t private_stride, uint8_t *d_public, size_t public_stride,
                                           uint8_t *d_digests, void *d_workspace, size_t workspace_bytes, unsigned flags,
                                           feds_stream_t stream);
feds_status feds_defragment_dct_strong_batch(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public,
                                             size_t public_stride, int n_images, int w, int h, int c, int k,
                                             const uint8_t key[16], const uint8_t *d_nonces,
                                             const uint8_t *d_expected_digests, uint8_t *d_images_out, size_t image_stride,
                                             uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes,
                                             unsigned flags, feds_stream_t stream);

/*
 * Packed integer coefficient storage (PAPER.md 6.4.3, Table 5; byte format: DESIGN.md 2.4). Part 1 of every block is
 * stored as integers: DC rounded into 11 bits ("DC coefficients are bounded by 2040"), every AC rounded into a sign-magnitude
 * field of ac_bits = 11 or 8 bits, clamped to its range; the fields of the (up to) 8 blocks of a leaf group form one little-endian
 * bit stream, so a full group takes exactly 11 + k*ac_bits bytes: 12.9 % (11-bit) or 9.96 % (8-bit) of a gray image at k = 5, as
 * P:599 prints. The private fragment is that stream under AES-128-CTR; the public fragment is w*h*c bytes, uint8 [block][64]: the
 * remainder pixels x - L modulo 256 ("IDCT of the rest"), taken against the quantised Part 1 in exact fixed-point arithmetic,
 * so that the inverse reproduces every pixel exactly with either storage. Digests: Merkle roots of the stored bytes (private leaf =
 * one group's bytes, public leaf = 8 blocks x 64 bytes).
 *   workspace: feds_dct_packed_workspace_bytes() per image (digest levels + room for the decrypted private fragment).
 *   errors as feds_fragment_dct; ac_bits other than 11 or 8: FEDS_ERR_BAD_PARAM. d_digests and the workspace are required.
 */
size_t feds_dct_packed_private_bytes(int w, int h, int c, int k, int ac_bits);
size_t feds_dct_packed_workspace_bytes(int w, int h, int c, int k, int ac_bits);
feds_status feds_fragment_dct_packed(const uint8_t *d_image, int w, int h, int c, int k, int ac_bits, const uint8_t key[16],
                                     const uint8_t nonce[16], uint8_t *d_private, uint8_t *d_public, uint8_t *d_digests,
                                     void *d_workspace, size_t workspace_bytes, feds_stream_t stream);
feds_status feds_defragment_dct_packed(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int k, int ac_bits,
                                       const uint8_t key[16], const uint8_t nonce[16], const uint8_t *d_expected_digests,
                                       uint8_t *d_image_out, uint32_t *d_verify_flags, void *d_workspace,
                                       size_t workspace_bytes, feds_stream_t stream);
feds_status feds_fragment_dct_packed_batch(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c,
                                           int k, int ac_bits, const uint8_t key[16], const uint8_t *d_nonces,
                                           uint8_t *d_private, size_t private_stride, uint8_t *d_public, size_t public_stride,
                                           uint8_t *d_digests, void *d_workspace, size_t workspace_bytes,
                                           feds_stream_t stream);
feds_status feds_defragment_dct_packed_batch(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public,
                                             size_t public_stride, int n_images, int w, int h, int c, int k, int ac_bits,
                                             const uint8_t key[16], const uint8_t *d_nonces,
                                             const uint8_t *d_expected_digests, uint8_t *d_images_out, size_t image_stride,
                                             uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes,
                                             feds_stream_t stream);

/*
 * feds_fragment_dwt / feds_defragment_dwt — rows D1-D8: level shift -128, `levels`-level whole-image
 * Le Gall 5/3 integer lifting, rows then columns, LL_levels -> private under AES-128-CTR,
 * the other subbands -> public (order: channel, level L..1, HL, LH, HH, row-major int16 LE), SHA-256 Merkle
 * digests over 2048-byte leaves of each fragment stream; the inverse is exact.
 */
feds_status feds_fragment_dwt(const uint8_t *d_image, int w, int h, int c, int levels, const uint8_t key[16],
                              const uint8_t nonce[16], uint8_t *d_private, uint8_t *d_public, uint8_t *d_digests,
                              void *d_workspace, size_t workspace_bytes, feds_stream_t stream);

feds_status feds_defragment_dwt(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int levels,
                                const uint8_t key[16], const uint8_t nonce[16], const uint8_t *d_expected_digests,
                                uint8_t *d_image_out, uint32_t *d_verify_flags, void *d_workspace,
                                size_t workspace_bytes, feds_stream_t stream);

/* feds_verify_dwt — as feds_verify_dct for the DWT path's fragments (2048-byte leaves of each fragment stream); no key needed.
 * Workspace as for feds_defragment_dwt. */
feds_status feds_verify_dwt(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c, int levels,
                            const uint8_t *d_expected_digests, uint32_t *d_verify_flags, void *d_workspace,
                            size_t workspace_bytes, feds_stream_t stream);

/*
 * Batched DWT entry points: n_images images of identical shape at the given byte strides (multiples of 16), one nonce per image
 * in the DEVICE array d_nonces (uint8[n_images][16], non-overlapping counter ranges as for the DCT batch), digests at
 * d_digests + 64 i, verify flags at d_verify_flags + i. Every level kernel, the AES-CTR pass and the leaf hashing span the
 * whole batch in one launch each. Workspace: n_images * feds_workspace_bytes(w, h, c, levels, 1).
 * flags: FEDS_FLAG_NONE or FEDS_FLAG_DWT_TILED.
 */
feds_status feds_fragment_dwt_batch(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c, int levels,
                                    const uint8_t key[16], const uint8_t *d_nonces, uint8_t *d_private, size_t private_stride,
                                    uint8_t *d_public, size_t public_stride, uint8_t *d_digests, void *d_workspace,
                                    size_t workspace_bytes, unsigned flags, feds_stream_t stream);
feds_status feds_defragment_dwt_batch(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                      int n_images, int w, int h, int c, int levels, const uint8_t key[16], const uint8_t *d_nonces,
                                      const uint8_t *d_expected_digests, uint8_t *d_images_out, size_t image_stride,
                                      uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes, unsigned flags,
                                      feds_stream_t stream);

/*
 * feds_defragment_dwt_batch with the verification on a second stream. Recomputing the digests of the received fragments (leaf
 * hashing, tree, compare: A10 "recompute + compare before use") and rebuilding the image from them (AES-CTR, inverse levels) read
 * the same bytes and write disjoint parts of the workspace; on a single image the first is a chain of dependent hash launches
 * that leaves the chip half empty and the second is bound by memory. This form enqueues the verification on aux_stream and the
 * reconstruction on stream: fork_event is recorded on stream and waited for by aux_stream before its first kernel, join_event
 * is recorded on aux_stream after the compare kernel and waited for by stream after the last level -- work enqueued on stream
 * after the call sees both the image and the flags; nothing synchronises with the host; both streams may be under capture into
 * one CUDA graph. The caller owns both streams and both events (any flags; cudaEventDisableTiming recommended) and must not
 * reuse the events before the call's work has completed. d_expected_digests and d_verify_flags must not be NULL (without
 * verification there is nothing to overlap: use feds_defragment_dwt_batch). Same results as feds_defragment_dwt_batch.
 * (There is no such form for the DCT path: its reconstruction kernel is one persistent CTA per SM, and sharing the chip with
 * the hash kernel leaves some of those CTAs without an SM until the hashing is over -- measured: up to 1.9x slower at 2048^2.)
 */
feds_status feds_defragment_dwt_batch_2s(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public, size_t public_stride,
                                         int n_images, int w, int h, int c, int levels, const uint8_t key[16], const uint8_t *d_nonces,
                                         const uint8_t *d_expected_digests, uint8_t *d_images_out, size_t image_stride,
                                         uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes, unsigned flags,
                                         feds_stream_t stream, feds_stream_t aux_stream, feds_event_t fork_event, feds_event_t join_event);
/*
 * Batched DCT entry points ("series of images"): n_images images of identical shape, image i at
 * d_images + i*image_stride, fragments at d_private + i*private_stride / d_public + i*public_stride, digests at
 * d_digests + 64 i, verify flags at d_verify_flags + i. Every image is an independent CTR message with its own
 * nonce ("different IV for each input matrix"): d_nonces is a DEVICE array uint8[n_images][16].
 * The counter ranges must not overlap: every image uses the counter blocks [nonce_i, nonce_i + ceil(private_bytes / 16)) mod 2^128
 * under the one key, so any two nonces of a batch (and of every other batch under that key) must differ by at least that many
 * blocks -- overlapping ranges reuse keystream (a two-time pad). The library cannot check this across calls; it is the caller's duty.
 * One launch per stage spans the whole batch. Strides are in bytes, multiples of 16, >= the per-image size.
 * Workspace: n_images * feds_workspace_bytes(...).
 */
feds_status feds_fragment_dct_batch(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c,
                                    int k, const uint8_t key[16], const uint8_t *d_nonces, uint8_t *d_private,
                                    size_t private_stride, uint8_t *d_public, size_t public_stride, uint8_t *d_digests,
                                    void *d_workspace, size_t workspace_bytes, unsigned flags, feds_stream_t stream);

feds_status feds_defragment_dct_batch(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public,
                                      size_t public_stride, int n_images, int w, int h, int c, int k,
                                      const uint8_t key[16], const uint8_t *d_nonces,
                                      const uint8_t *d_expected_digests, uint8_t *d_images_out, size_t image_stride,
                                      uint32_t *d_verify_flags, void *d_workspace, size_t workspace_bytes,
                                      unsigned flags, feds_stream_t stream);

/*
 * Host-staged batch fragment (BASELINE north_star "stream-overlapped host<->device staging"; the paper's
 * Fig. 11 overlay, moved to PCIe): images, fragments and digests live in HOST memory (pinned for
 * the copies to overlap); the batch is cut into n_streams chunks-in-flight, each chunk doing H2D -> fragment
 * -> D2H on its own stream. The caller supplies the streams and one device scratch area of
 * feds_fragment_dct_host_scratch_bytes() bytes. h_nonces is uint8[n_images][16] on the HOST.
 * Returns after enqueuing; synchronise the given streams before reading the outputs.
 */
size_t feds_fragment_dct_host_scratch_bytes(int images_per_chunk, int n_streams, int w, int h, int c, int k);
feds_status feds_fragment_dct_host(const uint8_t *h_images, int n_images, int w, int h, int c, int k,
                                   const uint8_t key[16], const uint8_t *h_nonces, uint8_t *h_private,
                                   uint8_t *h_public, uint8_t *h_digests, int images_per_chunk, void *d_scratch,
                                   size_t scratch_bytes, feds_stream_t *streams, int n_streams, unsigned flags);

/*
 * Host-staged batch defragment: the mirror image (H2D fragments + nonces [+ expected digests] -> defragment -> D2H
 * images [+ verify flags]). h_expected_digests may be NULL (no verification; h_verify_flags untouched).
 * Uses the same chunk -> stream mapping and the same scratch slot per stream as feds_fragment_dct_host (the two scratch
 * sizes are equal), so the two may be enqueued back to back -- or alternately, sub-batch by sub-batch, which keeps both PCIe
 * directions busy -- on the same streams and scratch without a synchronisation in between.
 */
size_t feds_defragment_dct_host_scratch_bytes(int images_per_chunk, int n_streams, int w, int h, int c, int k);
feds_status feds_defragment_dct_host(const uint8_t *h_private, const uint8_t *h_public, int n_images, int w, int h, int c, int k,
                                     const uint8_t key[16], const uint8_t *h_nonces, const uint8_t *h_expected_digests,
                                     uint8_t *h_images_out, uint32_t *h_verify_flags, int images_per_chunk, void *d_scratch,
                                     size_t scratch_bytes, feds_stream_t *streams, int n_streams, unsigned flags);

/*
 * The report's own DWT design (PAPER.md 6.9.3-6.9.4, Figure 18; byte format: DESIGN.md 2.5): every 8x8 tile of every
 * channel plane gets two levels of the integer Le Gall 5/3 transform. "Level 1" (the four LL2 coefficients, 40 bits) is protected by
 * AES-128-CTR; "level 2" (HL2, LH2, HH2: 124 bits) is XORed with SHA-256(level 1 || key || nonce); "level 3" (HL1, LH1, HH1: 480 bits)
 * with SHA-512(level 2 || key || nonce); fields of 10 bits, 11 for HH2.
 *   d_private: feds_dwt_tiles_private_bytes() = 21 bytes per tile: [16 bytes of protected level 2 per tile] then [5 bytes of level 1
 *              per tile, all tiles as one AES-128-CTR message]
 *   d_public : feds_dwt_tiles_public_bytes() = 60 bytes per tile (protected level 3); tiles in the order channel, tile row, tile column
 *   d_digests: 64 bytes, stream Merkle roots of the two fragments as stored (2048-byte leaves, as the DWT path)
 *   workspace: feds_dwt_tiles_workspace_bytes() per image. w, h multiples of 8. The inverse is exact.
 */
size_t feds_dwt_tiles_private_bytes(int w, int h, int c);
size_t feds_dwt_tiles_public_bytes(int w, int h, int c);
size_t feds_dwt_tiles_workspace_bytes(int w, int h, int c);
feds_status feds_fragment_dwt_tiles(const uint8_t *d_image, int w, int h, int c, const uint8_t key[16], const uint8_t nonce[16],
                                    uint8_t *d_private, uint8_t *d_public, uint8_t *d_digests, void *d_workspace,
                                    size_t workspace_bytes, feds_stream_t stream);
feds_status feds_defragment_dwt_tiles(const uint8_t *d_private, const uint8_t *d_public, int w, int h, int c,
                                      const uint8_t key[16], const uint8_t nonce[16], const uint8_t *d_expected_digests,
                                      uint8_t *d_image_out, uint32_t *d_verify_flags, void *d_workspace,
                                      size_t workspace_bytes, feds_stream_t stream);
feds_status feds_fragment_dwt_tiles_batch(const uint8_t *d_images, int n_images, size_t image_stride, int w, int h, int c,
                                          const uint8_t key[16], const uint8_t *d_nonces, uint8_t *d_private,
                                          size_t private_stride, uint8_t *d_public, size_t public_stride, uint8_t *d_digests,
                                          void *d_workspace, size_t workspace_bytes, feds_stream_t stream);
feds_status feds_defragment_dwt_tiles_batch(const uint8_t *d_private, size_t private_stride, const uint8_t *d_public,
                                            size_t public_stride, int n_images, int w, int h, int c, const uint8_t key[16],
                                            const uint8_t *d_nonces, const uint8_t *d_expected_digests, uint8_t *d_images_out,
                                            size_t image_stride, uint32_t *d_verify_flags, void *d_workspace,
                                            size_t workspace_bytes, feds_stream_t stream);

/*
 * Stream primitives: the two cryptographic steps of the path on a plain byte stream in device memory.
 *
 * feds_aes128_ctr — step 4 alone: d_out[i] = d_in[i] XOR keystream[i] over n_bytes bytes, counter block of the j-th
 * 16-byte block = (nonce + j) mod 2^128 big-endian (SP 800-38A 6.5, A6); the keystream of a partial last block
 * is truncated. d_out == d_in (in place) is allowed, partial overlap is not. This is also the report's comparison
 * baseline "AES over the whole image" when given the image bytes.
 * key, nonce: HOST pointers. n_bytes == 0 is a no-op.
 *
 * feds_sha256_merkle — step 5 alone on a stream: leaf j = SHA-256(bytes [2048 j, min(2048 (j+1), n))), upper levels with
 * fan-out 16; a one-leaf stream's root is its leaf digest, an empty stream's root is SHA-256("").
 * d_root: 32 bytes, device. Workspace: feds_sha256_merkle_workspace_bytes(n_bytes) (leaf and inner digests); may be
 * NULL when the stream has at most one leaf.
 *
 * Errors as for the other entry points: NULL_POINTER, MISALIGNED (16-byte alignment of every device pointer),
 * WORKSPACE_TOO_SMALL, BAD_PARAM (more than 2^32 - 1 leaves), CUDA. Nothing is enqueued when an error is returned.
 */
feds_status feds_aes128_ctr(const uint8_t *d_in, uint8_t *d_out, size_t n_bytes, const uint8_t key[16],
                            const uint8_t nonce[16], feds_stream_t stream);
size_t feds_sha256_merkle_workspace_bytes(size_t n_bytes);
feds_status feds_sha256_merkle(const uint8_t *d_data, size_t n_bytes, uint8_t *d_root, void *d_workspace,
                               size_t workspace_bytes, feds_stream_t stream);

/*
 * feds_sha256_merkle_static — feds_sha256_merkle for callers that cannot allocate device memory (code under CUDA graph
 * capture, serving loops, harnesses that forbid cudaMalloc): the same digest (step 5 on a stream), the same
 * kernels, but the workspace is a static array in device memory inside the library, 1.125 MiB on every GPU that loads the
 * library, held until the process exits. The call allocates and frees nothing (no cudaMalloc / cudaFree, no allocating
 * library routine) and does not synchronise. d_data: n_bytes bytes, device; d_root: 32 bytes, device; both 16-byte aligned.
 * Limit: n_bytes <= feds_sha256_merkle_static_max_bytes() = 64 MiB (32,768 leaves); a longer stream returns
 * FEDS_ERR_BAD_PARAM and enqueues nothing -- use feds_sha256_merkle with a workspace of your own. Other errors as for
 * feds_sha256_merkle.
 * All calls on one device share the array, and it keeps the last call's contents (each call writes every slot it reads and
 * clears the counters it needs at zero): calls that may overlap on the GPU -- different streams with no ordering between
 * them -- race on it and must be ordered by the caller; calls on one stream, or on different devices, are safe.
 */
size_t feds_sha256_merkle_static_max_bytes(void);
feds_status feds_sha256_merkle_static(const uint8_t *d_data, size_t n_bytes, uint8_t *d_root, feds_stream_t stream);

/*
 * Profiling hook (not part of the data path; thread-local): while set, every fragment/defragment call made on this
 * thread records ev_start immediately before and ev_stop immediately after its dominant kernel(s), on the call's stream:
 * DCT calls with digests (fragment, verified defragment, feds_verify_dct): the leaf-hash kernel, or the fused kernel on the
 * FEDS_FLAG_FORCE_FUSED route; digest-free DCT calls: the tile kernel; DWT path: the leaf-hashing kernel.
 * Both are cudaEvent_t handles owned by the caller. Pass NULL, NULL to clear.
 */
void feds_profile_events(void *ev_start, void *ev_stop);

#ifdef __cplusplus
}
#endif
#endif /* FEDS_H */
