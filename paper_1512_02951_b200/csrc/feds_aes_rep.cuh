// feds_aes_rep.cuh — AES-128 rounds on the 32-fold replicated FOUR-table layout (128 KB of shared memory), shared by the AES-CTR
// stream kernel (feds_hash.cuh) and the tile role of the fused DCT kernels (feds_dct_fused.cuh).
#pragma once
#include "feds_device.cuh"

namespace feds {

constexpr int REP4_TABLE_WORDS = 4 * 256 * 32;   // entry x of table t, copy l at word (t * 256 + x) * 32 + l

// The ten rounds on the 32-fold replicated four-table layout (entry x of table t, copy l at byte t * 32768 + x * 128 + l * 4;
// lane l reads copy l, which lies in bank l: every lookup is one wavefront). A lookup costs ONE ALU-pipe instruction (PRMT: the
// byte, zero-extended), one IMAD on the FMA pipe (byte * 128 + lane base; the multiplier is a run-time 128 so that ptxas keeps it a
// multiply-add instead of a shift and an add on the ALU pipe) and the LDS, whose immediate offset selects the table: 24 ALU-pipe
// instructions per round against 40 for shift + mask-or-lane. Same arithmetic as aes128_encrypt (FIPS-197 5.1, T-table form).
struct RepAes {
    uint32_t base;   // shared-memory byte address of the tables + 4 * lane
    uint32_t c128;   // = 128, opaque to the compiler
};
template <int BYTE, int TABLE>
__device__ __forceinline__ uint32_t rep_lookup(const RepAes &A, uint32_t word) {
    const uint32_t b = __byte_perm(word, 0u, 0x4440 + BYTE);
    uint32_t addr, v;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(addr) : "r"(b), "r"(A.c128), "r"(A.base));
    asm("ld.shared.u32 %0, [%1 + %2];" : "=r"(v) : "r"(addr), "n"(TABLE * 32768));
    return v;
}
// ROLLED: the nine middle rounds as a loop (a tenth of the code; see aes128_encrypt in feds_dct_tile.cuh)
template <bool ROLLED = false, typename RkPtr>
__device__ __forceinline__ void aes128_encrypt_rep32(const RepAes &A, const RkPtr rk, uint32_t (&s)[4]) {
    uint32_t s0 = s[0] ^ rk[0], s1 = s[1] ^ rk[1], s2 = s[2] ^ rk[2], s3 = s[3] ^ rk[3];
#define FEDS_REP_ROUND(r)                                                                                                              \
    {                                                                                                                                  \
        const uint32_t t0 = rep_lookup<0, 0>(A, s0) ^ rep_lookup<1, 1>(A, s1) ^ rep_lookup<2, 2>(A, s2) ^ rep_lookup<3, 3>(A, s3) ^ rk[4 * (r) + 0]; \
        const uint32_t t1 = rep_lookup<0, 0>(A, s1) ^ rep_lookup<1, 1>(A, s2) ^ rep_lookup<2, 2>(A, s3) ^ rep_lookup<3, 3>(A, s0) ^ rk[4 * (r) + 1]; \
        const uint32_t t2 = rep_lookup<0, 0>(A, s2) ^ rep_lookup<1, 1>(A, s3) ^ rep_lookup<2, 2>(A, s0) ^ rep_lookup<3, 3>(A, s1) ^ rk[4 * (r) + 2]; \
        const uint32_t t3 = rep_lookup<0, 0>(A, s3) ^ rep_lookup<1, 1>(A, s0) ^ rep_lookup<2, 2>(A, s1) ^ rep_lookup<3, 3>(A, s2) ^ rk[4 * (r) + 3]; \
        s0 = t0; s1 = t1; s2 = t2; s3 = t3;                                                                                            \
    }
    if (ROLLED) {
#pragma unroll 1
        for (int r = 1; r < 10; ++r) FEDS_REP_ROUND(r)
    } else {
#pragma unroll
        for (int r = 1; r < 10; ++r) FEDS_REP_ROUND(r)
    }
#undef FEDS_REP_ROUND
    // final round: SubBytes + ShiftRows. S sits in byte 0 of T2, bytes 1 and 2 of T0 and byte 3 of T1 (T0 = (2S, S, S, 3S)).
#define FEDS_LAST(a, b, c, d)                                                                       \
    __byte_perm(__byte_perm(rep_lookup<0, 2>(A, a), rep_lookup<1, 0>(A, b), 0x3250),                 \
                __byte_perm(rep_lookup<2, 0>(A, c), rep_lookup<3, 1>(A, d), 0x7210), 0x7610)
    const uint32_t u0 = FEDS_LAST(s0, s1, s2, s3), u1 = FEDS_LAST(s1, s2, s3, s0), u2 = FEDS_LAST(s2, s3, s0, s1), u3 = FEDS_LAST(s3, s0, s1, s2);
#undef FEDS_LAST
    s[0] = u0 ^ rk[40]; s[1] = u1 ^ rk[41]; s[2] = u2 ^ rk[42]; s[3] = u3 ^ rk[43];
}

}  // namespace feds
