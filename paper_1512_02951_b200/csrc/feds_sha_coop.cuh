// feds_sha_coop.cuh — SHA-256 of ONE message by a whole warp, for latency (sm_100a).
//
// A thread that hashes a leaf alone walks a chain of dependent compressions; with a lone warp on an SM one compression takes
// ~3,900 cycles (every instruction waits for the one before it), so the 34 compressions of a DCT leaf cost 68 us and the three
// top levels of a tree 54 us however small the image is. But only the 64 ROUNDS of a compression depend on the chaining value:
// the message schedule W_0..W_63 of every 64-byte block of the message is a function of the data alone. So:
//   phase 1: lane b expands the schedule of block b (up to 32 blocks at a time) and parks W_t + K_t in shared memory;
//   phase 2: the rounds of those blocks run one after the other (every lane computes the same values: no divergence, broadcast
//            loads), each round a chain of three dependent instructions: e' = (d + h + K_t + W_t) + Sigma1(e) + Ch(e, f, g)
//            with the bracket formed off the critical path.
// ~2,900 cycles per block instead of ~3,900 (a lone warp cannot issue the ~16 instructions of a round in less than ~45 cycles). Throughput is a 32nd of a thread-per-message kernel's, so the host uses these kernels
// only while there are fewer messages than the chip has warp schedulers to spare (small images, tree tops).
#pragma once
#include "feds_device.cuh"

namespace feds {

// per warp: W_t + K_t of STRIDE blocks at a time, t-major (word t of block b at t * STRIDE + b): conflict-free stores
template <int STRIDE> constexpr int coop_ws_words() { return 64 * STRIDE; }

// big-endian message word j of 64-byte block b of a message of nbytes bytes at msg (4-byte aligned), with the FIPS 180-4 5.1.1
// padding: 0x80, zeros, 64-bit bit length in the last block
__device__ __forceinline__ uint32_t coop_message_word(const uint8_t *msg, unsigned nbytes, unsigned nblocks, unsigned b, int j) {
    const unsigned off = 64u * b + 4u * j;
    if (off + 4u <= nbytes) return bswap32(*reinterpret_cast<const uint32_t *>(msg + off));
    if (b == nblocks - 1 && j == 15) return nbytes * 8u;   // messages here are shorter than 2^29 bytes
    if (b == nblocks - 1 && j == 14) return 0u;
    uint32_t word = 0u;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const unsigned pos = off + q;
        const uint32_t byte = pos < nbytes ? msg[pos] : (pos == nbytes ? 0x80u : 0u);
        word = (word << 8) | byte;
    }
    return word;
}

// additions as IMAD on the FMA pipe (add_fma): the ten shift / logic operations of a round keep the ALU pipe to themselves
#define FEDS_COOP_ROUND(a, b, c, d, e, f, g, h, kw)                                   \
    {                                                                                 \
        const uint32_t x = add_fma(h, kw, one), y = add_fma(x, d, one);               \
        const uint32_t S1 = rotr32(e, 6) ^ rotr32(e, 11) ^ rotr32(e, 25);             \
        const uint32_t ch = (e & f) ^ (~e & g);                                       \
        const uint32_t S0 = rotr32(a, 2) ^ rotr32(a, 13) ^ rotr32(a, 22);             \
        const uint32_t maj = (a & b) ^ (a & c) ^ (b & c);                             \
        const uint32_t sc = add_fma(S1, ch, one);                                     \
        d = add_fma(y, sc, one);                                                      \
        h = add_fma(add_fma(x, sc, one), add_fma(S0, maj, one), one);                 \
    }

// All 32 lanes of a warp call this with the same arguments; every lane ends with the digest state in H. `ws` = this warp's
// coop_ws_words<STRIDE>() words of shared memory; STRIDE (<= 32) blocks are expanded at a time. msg may be global or shared
// (generic pointer), 4-byte aligned. `one` = 1, opaque to the compiler (add_fma).
template <int STRIDE>
__device__ __forceinline__ void sha256_warp_coop(const uint8_t *msg, unsigned nbytes, uint32_t *ws, int lane, const uint32_t one, uint32_t (&H)[8]) {
    sha256_init(H);
    const unsigned nblocks = (nbytes + 9u + 63u) / 64u;
#pragma unroll 1
    for (unsigned base = 0; base < nblocks; base += STRIDE) {
        const unsigned b = base + lane;
        if (lane < STRIDE && b < nblocks) {
            uint32_t w[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) w[j] = coop_message_word(msg, nbytes, nblocks, b, j);
#pragma unroll
            for (int t = 0; t < 16; ++t) ws[t * STRIDE + lane] = w[t] + c_sha256_k[t];
#pragma unroll 1
            for (int i = 1; i < 4; ++i) {
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const uint32_t w15 = w[(j + 1) & 15], w2 = w[(j + 14) & 15];
                    const uint32_t s0 = rotr32(w15, 7) ^ rotr32(w15, 18) ^ (w15 >> 3);
                    const uint32_t s1 = rotr32(w2, 17) ^ rotr32(w2, 19) ^ (w2 >> 10);
                    w[j] = w[j] + s0 + w[(j + 9) & 15] + s1;
                    ws[(16 * i + j) * STRIDE + lane] = w[j] + c_sha256_k[16 * i + j];
                }
            }
        }
        __syncwarp();
        const unsigned nb = min((unsigned)STRIDE, nblocks - base);
#pragma unroll 1
        for (unsigned bb = 0; bb < nb; ++bb) {
            uint32_t a = H[0], b2 = H[1], c = H[2], d = H[3], e = H[4], f = H[5], g = H[6], h = H[7];
            const uint32_t *wk = ws + bb;
            uint32_t kw[8], kn[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) kw[q] = wk[q * STRIDE];
#pragma unroll 1
            for (int t = 0; t < 64; t += 8) {
#pragma unroll
                for (int q = 0; q < 8; ++q) kn[q] = wk[((t + 8 + q) & 63) * STRIDE];   // the next eight, in flight under these rounds
                FEDS_COOP_ROUND(a, b2, c, d, e, f, g, h, kw[0])
                FEDS_COOP_ROUND(h, a, b2, c, d, e, f, g, kw[1])
                FEDS_COOP_ROUND(g, h, a, b2, c, d, e, f, kw[2])
                FEDS_COOP_ROUND(f, g, h, a, b2, c, d, e, kw[3])
                FEDS_COOP_ROUND(e, f, g, h, a, b2, c, d, kw[4])
                FEDS_COOP_ROUND(d, e, f, g, h, a, b2, c, kw[5])
                FEDS_COOP_ROUND(c, d, e, f, g, h, a, b2, kw[6])
                FEDS_COOP_ROUND(b2, c, d, e, f, g, h, a, kw[7])
#pragma unroll
                for (int q = 0; q < 8; ++q) kw[q] = kn[q];
            }
            H[0] += a; H[1] += b2; H[2] += c; H[3] += d; H[4] += e; H[5] += f; H[6] += g; H[7] += h;
        }
        __syncwarp();
    }
}

}  // namespace feds
