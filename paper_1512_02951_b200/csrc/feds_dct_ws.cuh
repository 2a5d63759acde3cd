// feds_dct_ws.cuh — warp-specialised fused kernels of the DCT path with digests, sm_100a.
//
// The digest path is bound by the integer (ALU) pipe: one SHA-256 compression per 64 stored bytes is ~1040 shift / logic /
// byte-permute operations that only that pipe executes, against 5 bytes of HBM traffic per pixel. A thread can
// only hash a leaf serially, so the chip is kept busy by having ~600 leaves per SM in flight; what decides the speed is that the
// threads walking those SHA chains do nothing else. Hence two kinds of warps in one persistent CTA per SM:
//
//   * HASH warps (20, 72 registers each): lane l owns one Merkle leaf (8 consecutive 8x8 blocks of one block row of one
//     channel) and streams its bytes, 64 at a time, straight from the fragment buffers into the message registers:
//     the registers-only loop of dct_leaves_hash_kernel (no shared-memory slots, no carry copies).
//   * WORKER warps (4, 128 registers; the highest warp ids, which the issue arbiter prefers): lane l owns one 8-block pixel
//     strip, ALL channels. Fragment: per 8x8 block load pixels, DCT, zigzag split, AES-128-CTR on the private words, store both
//     runs. Defragment: load both runs, decrypt, merge, IDCT, round, interleave the channels, store pixel rows.
//
// A worker produces (or consumes) "slab" s = block s of each of the 32 strips of a unit, s = 0..7; the C hash warps of that unit
// (one per channel) follow one slab behind. The fragment buffers in HBM / L2 ARE the stage between the two: the worker's stores
// are made visible with a CTA-scope fence and a counter in shared memory, the hash warps poll that counter before they fetch
// the next 64 bytes, and the workers stay at most `ahead` slabs in front of the slowest hash warp, so that what is hashed (or,
// when defragmenting, read a second time) is still in L2: fragments cross the HBM interface once.
//
// Requirements (the host routes everything else to the tile kernel + leaf-hash kernel): (w/8) % 8 == 0, so that every leaf has
// exactly 8 blocks and its streams are whole 64-byte chunks; k + 1 even (V = 2 or 4: runs are 8/16-byte multiples).
#pragma once
#include "feds_dct.cuh"

namespace feds {

constexpr int WS_HASH_WARPS = 20;   // five warpgroups (setmaxnreg acts on warpgroups of 4 warps)
constexpr int WS_WORK_WARPS = 4;    // one warpgroup, the last one
constexpr int WS_THREADS = (WS_HASH_WARPS + WS_WORK_WARPS) * 32;
constexpr int WS_HASH_REGS = 72, WS_WORK_REGS = 120;   // 20 * 72 + 4 * 120 = 24 * 80: setmaxnreg only moves registers inside the CTA's own pool
constexpr int WS_TABLE_WORDS = 4 * 256 * 32;   // T0..T3, every entry replicated 32 times (lane l reads copy l in bank l)
constexpr int WS_KB_STRIDE = 68;               // words of keystream scratch per worker lane (<= 64 + 3), 4 mod 32
constexpr int WS_PB_STRIDE = 68;               // words of packed-pixel scratch per worker lane (C * 16 <= 64), 4 mod 32

template <int C> struct WsShape {
    static constexpr int UNITS = WS_HASH_WARPS / C;                               // units in flight per CTA: 20 / 6 / 5
    static constexpr int PER_WORKER = (UNITS + WS_WORK_WARPS - 1) / WS_WORK_WARPS;
};
__host__ __device__ inline size_t ws_smem_bytes() {
    return (size_t)(WS_TABLE_WORDS + WS_WORK_WARPS * 32 * (WS_KB_STRIDE + WS_PB_STRIDE) + 64) * 4;
}

__device__ __forceinline__ void ws_fence_cta() { asm volatile("fence.acq_rel.cta;" ::: "memory"); }
__device__ __forceinline__ int ld_volatile_s32(const int *p) {
    int v;
    asm volatile("ld.volatile.shared.s32 %0, [%1];" : "=r"(v) : "r"((uint32_t)__cvta_generic_to_shared(p)) : "memory");
    return v;
}
__device__ __forceinline__ void st_volatile_s32(int *p, int v) {
    asm volatile("st.volatile.shared.s32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(p)), "r"(v) : "memory");
}

// ------------------------------------------------------------------------------------------------------------
// AES-128 on the 32-fold replicated four-table layout (entry x of table t, copy l at byte t * 32768 + x * 128 + l * 4).
// A lookup costs ONE ALU-pipe instruction (PRMT: the byte, zero-extended), one IMAD on the FMA pipe (byte * 128 + lane base; the
// multiplier is a run-time 128 so that ptxas keeps it a multiply-add) and the LDS, whose immediate offset selects the table:
// 24 ALU-pipe instructions per round against 52 for the shift-mask-or form on a single table. Same arithmetic as aes128_encrypt.
// ------------------------------------------------------------------------------------------------------------
struct WsAes {
    uint32_t base;   // shared-memory byte address of the tables + 4 * lane
    uint32_t c128;   // = 128, opaque to the compiler
};
template <int BYTE, int TABLE>
__device__ __forceinline__ uint32_t ws_lookup(const WsAes &A, uint32_t word) {
    const uint32_t b = __byte_perm(word, 0u, 0x4440 + BYTE);
    uint32_t addr, v;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(addr) : "r"(b), "r"(A.c128), "r"(A.base));
    asm("ld.shared.u32 %0, [%1 + %2];" : "=r"(v) : "r"(addr), "n"(TABLE * 32768));
    return v;
}
template <typename RkPtr>
__device__ __forceinline__ void ws_aes128_encrypt(const WsAes &A, const RkPtr rk, uint32_t (&s)[4]) {
    uint32_t s0 = s[0] ^ rk[0], s1 = s[1] ^ rk[1], s2 = s[2] ^ rk[2], s3 = s[3] ^ rk[3];
#pragma unroll
    for (int r = 1; r < 10; ++r) {
        const uint32_t t0 = ws_lookup<0, 0>(A, s0) ^ ws_lookup<1, 1>(A, s1) ^ ws_lookup<2, 2>(A, s2) ^ ws_lookup<3, 3>(A, s3) ^ rk[4 * r + 0];
        const uint32_t t1 = ws_lookup<0, 0>(A, s1) ^ ws_lookup<1, 1>(A, s2) ^ ws_lookup<2, 2>(A, s3) ^ ws_lookup<3, 3>(A, s0) ^ rk[4 * r + 1];
        const uint32_t t2 = ws_lookup<0, 0>(A, s2) ^ ws_lookup<1, 1>(A, s3) ^ ws_lookup<2, 2>(A, s0) ^ ws_lookup<3, 3>(A, s1) ^ rk[4 * r + 2];
        const uint32_t t3 = ws_lookup<0, 0>(A, s3) ^ ws_lookup<1, 1>(A, s0) ^ ws_lookup<2, 2>(A, s1) ^ ws_lookup<3, 3>(A, s2) ^ rk[4 * r + 3];
        s0 = t0; s1 = t1; s2 = t2; s3 = t3;
    }
    // final round: SubBytes + ShiftRows. S sits in byte 0 of T2, bytes 1 and 2 of T0 and byte 3 of T1 (T0 = (2S, S, S, 3S)).
#define FEDS_WS_LAST(a, b, c, d)                                                                              \
    __byte_perm(__byte_perm(ws_lookup<0, 2>(A, a), ws_lookup<1, 0>(A, b), 0x3250),                            \
                __byte_perm(ws_lookup<2, 0>(A, c), ws_lookup<3, 1>(A, d), 0x7210), 0x7610)
    const uint32_t u0 = FEDS_WS_LAST(s0, s1, s2, s3), u1 = FEDS_WS_LAST(s1, s2, s3, s0), u2 = FEDS_WS_LAST(s2, s3, s0, s1), u3 = FEDS_WS_LAST(s3, s0, s1, s2);
#undef FEDS_WS_LAST
    s[0] = u0 ^ rk[40]; s[1] = u1 ^ rk[41]; s[2] = u2 ^ rk[42]; s[3] = u3 ^ rk[43];
}

// ------------------------------------------------------------------------------------------------------------
// geometry shared by both roles
// ------------------------------------------------------------------------------------------------------------
struct WsStrip {
    bool valid;
    int n, br, g;   // image, block row, strip (= leaf column) in the row
};
__device__ __forceinline__ WsStrip ws_decode_strip(const DctParams &p, unsigned sg, int lane) {
    WsStrip S;
    const unsigned long long total = (unsigned long long)p.n_images * p.nbr * p.nlr;
    unsigned long long idx = (unsigned long long)sg * 32 + lane;
    S.valid = idx < total;
    if (!S.valid) idx = total - 1;   // lanes past the end repeat the last strip and store nothing
    const unsigned per_image = (unsigned)p.nbr * p.nlr;
    S.n = (int)(idx / per_image);
    const unsigned rem = (unsigned)(idx % per_image);
    S.br = (int)(rem / (unsigned)p.nlr);
    S.g = (int)(rem % (unsigned)p.nlr);
    return S;
}

struct WsCtrl {
    int *ready;      // [UNITS]  slabs finished by the unit's worker (running count over the unit's strip groups)
    int *consumed;   // [WS_HASH_WARPS] slabs whose bytes the hash warp has fetched completely
};

// ------------------------------------------------------------------------------------------------------------
// HASH role. Warp hw serves unit u = hw / C, channel ch = hw % C; lane = strip of the unit's current strip group.
// ------------------------------------------------------------------------------------------------------------
template <int C>
__device__ __forceinline__ void ws_hash_role(const DctParams &p, const WsCtrl &ctl, int hw, int lane) {
    constexpr int UNITS = WsShape<C>::UNITS;
    const int u = hw / C, ch = hw % C;
    const int P = p.k + 1, Q = 63 - p.k;
    const int pace = Q > 0 ? 0 : 1;   // the stream whose progress paces the worker: the first non-empty one
    const unsigned n_sg = p.ws_n_sg;
    int ready_seen = 0;
#pragma unroll 1
    for (unsigned it = 0;; ++it) {
        const unsigned sg = (unsigned)(u * (int)gridDim.x + (int)blockIdx.x) + it * (unsigned)(UNITS * (int)gridDim.x);
        if (sg >= n_sg) break;
        const int base_n = 8 * (int)it;
        const WsStrip S = ws_decode_strip(p, sg, lane);
        const unsigned row = (unsigned)(ch * p.nbr + S.br);
        const unsigned li = row * (unsigned)p.nlr + (unsigned)S.g;
        const size_t b0 = (size_t)row * p.nbc + (size_t)S.g * G_BLOCKS;
#pragma unroll 1
        for (int f = 0; f < 2; ++f) {   // 0: public stream (Q words per block), 1: private stream (ciphertext, P words per block)
            const int W = f ? P : Q;
            if (W == 0) continue;       // k = 63: the public fragment is empty, its root is written elsewhere
            const uint32_t *src = reinterpret_cast<const uint32_t *>(f ? p.priv + (size_t)S.n * p.priv_stride : p.pub + (size_t)S.n * p.pub_stride) +
                                  b0 * (size_t)W;
            const int full = W >> 1;    // 8 W words = W / 2 chunks of 16 words (W is even here)
            int cons = 0;               // slabs of this leaf group fetched completely
            uint32_t H[8], w[16];
            uint4 nx[4];
            sha256_init(H);
            auto fetch = [&](int blk) {
                const int words_end = 16 * (blk + 1);
                if ((ready_seen - base_n) * W < words_end) {
                    while (true) {
                        ready_seen = ld_volatile_s32(ctl.ready + u);
                        if ((ready_seen - base_n) * W >= words_end) break;
                        __nanosleep(64);
                    }
                    ws_fence_cta();   // acquire: the worker's stores of those slabs are visible to the loads below
                }
                const uint4 *q = reinterpret_cast<const uint4 *>(src + 16 * (size_t)blk);
#pragma unroll
                for (int i = 0; i < 4; ++i) nx[i] = __ldcg(q + i);   // every byte is hashed once: no use for L1
                if (f == pace) {
                    const int c0 = cons;
                    while (words_end >= (cons + 1) * W) ++cons;
                    if (cons != c0 && lane == 0) st_volatile_s32(ctl.consumed + hw, base_n + cons);
                }
            };
            fetch(0);
#pragma unroll 1
            for (int blk = 0; blk <= full; ++blk) {
                if (blk < full) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        w[4 * i] = bswap32(nx[i].x); w[4 * i + 1] = bswap32(nx[i].y); w[4 * i + 2] = bswap32(nx[i].z); w[4 * i + 3] = bswap32(nx[i].w);
                    }
                    if (blk + 1 < full) fetch(blk + 1);
                } else {   // padding block (FIPS 180-4 5.1.1): the message is a whole number of 64-byte chunks
#pragma unroll
                    for (int i = 0; i < 16; ++i) w[i] = 0u;
                    w[0] = 0x80000000u;
                    w[15] = (uint32_t)(8 * W) * 32u;   // message length in bits
                }
                sha256_compress_rolled_fma(H, w, p.one);
            }
            if (S.valid) store_digest(p.leaves + (((size_t)S.n * 2 + (f ? 0 : 1)) * p.leaves_per_image + li) * 32, H);
        }
        if (lane == 0) st_volatile_s32(ctl.consumed + hw, base_n + 8);
    }
}

// ------------------------------------------------------------------------------------------------------------
// WORKER role, shared scheduling: worker `pw` serves units pw, pw + 4, ...; for each it runs slab after slab of the unit's
// strip groups, never more than p.ws_ahead slabs in front of the slowest of the unit's C hash warps.
// ------------------------------------------------------------------------------------------------------------
template <int C, typename SlabFn>
__device__ __forceinline__ void ws_worker_schedule(const DctParams &p, const WsCtrl &ctl, int pw, int lane, SlabFn &&slab) {
    constexpr int UNITS = WsShape<C>::UNITS, PER = WsShape<C>::PER_WORKER;
    int issued[PER];
#pragma unroll
    for (int j = 0; j < PER; ++j) issued[j] = 0;
    const unsigned n_sg = p.ws_n_sg;
#pragma unroll 1
    while (true) {
        // the unit whose hash warps are closest to running dry goes next (one call site of the slab code)
        int pick = -1, pick_n = 0, pick_lead = 0x7fffffff;
        unsigned pick_sg = 0;
        bool more = false;
#pragma unroll
        for (int j = 0; j < PER; ++j) {
            const int u = pw + j * WS_WORK_WARPS;
            if (u >= UNITS) continue;
            const int n = issued[j];
            const unsigned sg = (unsigned)(u * (int)gridDim.x + (int)blockIdx.x) + (unsigned)(n >> 3) * (unsigned)(UNITS * (int)gridDim.x);
            if (sg >= n_sg) continue;
            more = true;
            int cons = ld_volatile_s32(ctl.consumed + u * C);
#pragma unroll
            for (int c = 1; c < C; ++c) cons = min(cons, ld_volatile_s32(ctl.consumed + u * C + c));
            const int lead = n - cons;
            if (lead < p.ws_ahead && lead < pick_lead) { pick = j; pick_n = n; pick_lead = lead; pick_sg = sg; }
        }
        if (!more) break;
        if (pick < 0) { __nanosleep(128); continue; }
        slab(pick_sg, pick_n & 7);
        ws_fence_cta();   // release: this lane's stores before the counter
        __syncwarp();
        if (lane == 0) st_volatile_s32(ctl.ready + pw + pick * WS_WORK_WARPS, pick_n + 1);
#pragma unroll
        for (int j = 0; j < PER; ++j)
            if (j == pick) issued[j] = pick_n + 1;
    }
}

// keystream of the private words [w0, w0 + P) of one block -> kb[(w0 & 3) + j], j = 0..P-1 (whole counter blocks are computed)
__device__ __forceinline__ void ws_keystream(const DctParams &p, const WsAes &A, const uint32_t (&nonce)[4], unsigned long long w0, int P,
                                             uint32_t *kb) {
    const unsigned long long blk0 = w0 >> 2;
    const int nks = ((int)(w0 & 3) + P + 3) >> 2;
#pragma unroll 1
    for (int j = 0; j < nks; ++j) {
        uint32_t ks[4];
        ctr_block(nonce, blk0 + j, ks);
        ws_aes128_encrypt(A, p.rk, ks);
        *reinterpret_cast<uint4 *>(kb + 4 * j) = make_uint4(ks[0], ks[1], ks[2], ks[3]);
    }
}

template <int C, int V>
__device__ __forceinline__ void ws_fragment_slab(const DctParams &p, const WsAes &A, uint32_t *kb, unsigned sg, int s, int lane) {
    constexpr ZigzagTable ZZ = make_zigzag();
    const WsStrip S = ws_decode_strip(p, sg, lane);
    if (!S.valid) return;
    const int P = p.k + 1, Q = 63 - p.k;
    const uint8_t *img = p.images + (size_t)S.n * p.image_stride;
    uint32_t *priv = reinterpret_cast<uint32_t *>(p.priv + (size_t)S.n * p.priv_stride);
    uint32_t *pub = reinterpret_cast<uint32_t *>(p.pub + (size_t)S.n * p.pub_stride);
    uint32_t nonce[4];
    load_nonce(p, S.n, nonce);
#pragma unroll 1
    for (int ch = 0; ch < C; ++ch) {
        const size_t blk = ((size_t)(ch * p.nbr + S.br) * p.nbc) + (size_t)S.g * G_BLOCKS + s;
        const unsigned long long w0 = (unsigned long long)blk * P;
        ws_keystream(p, A, nonce, w0, P, kb);
        const uint32_t *kv = kb + (int)(w0 & 3);
        float v[64];
        load_block<C>(img, p.w, 8 * S.br, 8 * (S.g * G_BLOCKS + s), ch, v);
        dct8x8(v);
        uint32_t *pv = priv + w0;                 // private run of this block, indexed by z
        uint32_t *pq = pub + blk * (size_t)Q - P;  // public run of this block, indexed by z (z >= P)
#pragma unroll
        for (int g = 0; g < 64; g += V) {
            uint32_t x[V];
#pragma unroll
            for (int t = 0; t < V; ++t) x[t] = __float_as_uint(v[ZZ.pos[g + t]]);
            if (g < P) {
                uint32_t ks[V];
                vec_load<V>(kv + g, ks);
#pragma unroll
                for (int t = 0; t < V; ++t) x[t] ^= ks[t];
                vec_store<V>(pv + g, x);
            } else {
                vec_store<V>(pq + g, x);
            }
        }
    }
}

// interleave the packed rows of C channel planes (2 words = 8 pixels each) into 2 C words of pixel-interleaved bytes
template <int C>
__device__ __forceinline__ void ws_store_row(uint8_t *row, const uint32_t *pb, int r) {
    if (C == 1) {
        *reinterpret_cast<uint2 *>(row) = *reinterpret_cast<const uint2 *>(pb + 2 * r);
    } else if (C == 3) {
        const uint2 R = *reinterpret_cast<const uint2 *>(pb + 2 * r), G = *reinterpret_cast<const uint2 *>(pb + 16 + 2 * r),
                    B = *reinterpret_cast<const uint2 *>(pb + 32 + 2 * r);
        const uint32_t rg0 = __byte_perm(R.x, G.x, 0x5140), rg1 = __byte_perm(R.x, G.x, 0x7362);   // R0 G0 R1 G1 | R2 G2 R3 G3
        const uint32_t rg2 = __byte_perm(R.y, G.y, 0x5140), rg3 = __byte_perm(R.y, G.y, 0x7362);
        const uint32_t w0 = __byte_perm(rg0, B.x, 0x2410);                                           // R0 G0 B0 R1
        const uint32_t w1 = __byte_perm(__byte_perm(rg0, B.x, 0x0053), rg1, 0x5410);                 // G1 B1 R2 G2
        const uint32_t w2 = __byte_perm(rg1, B.x, 0x7326);                                           // B2 R3 G3 B3
        const uint32_t w3 = __byte_perm(rg2, B.y, 0x2410);
        const uint32_t w4 = __byte_perm(__byte_perm(rg2, B.y, 0x0053), rg3, 0x5410);
        const uint32_t w5 = __byte_perm(rg3, B.y, 0x7326);
        uint2 *o = reinterpret_cast<uint2 *>(row);
        o[0] = make_uint2(w0, w1);
        o[1] = make_uint2(w2, w3);
        o[2] = make_uint2(w4, w5);
    } else {
        const uint2 R = *reinterpret_cast<const uint2 *>(pb + 2 * r), G = *reinterpret_cast<const uint2 *>(pb + 16 + 2 * r),
                    B = *reinterpret_cast<const uint2 *>(pb + 32 + 2 * r), Al = *reinterpret_cast<const uint2 *>(pb + 48 + 2 * r);
        const uint32_t rg0 = __byte_perm(R.x, G.x, 0x5140), rg1 = __byte_perm(R.x, G.x, 0x7362);
        const uint32_t ba0 = __byte_perm(B.x, Al.x, 0x5140), ba1 = __byte_perm(B.x, Al.x, 0x7362);
        const uint32_t rg2 = __byte_perm(R.y, G.y, 0x5140), rg3 = __byte_perm(R.y, G.y, 0x7362);
        const uint32_t ba2 = __byte_perm(B.y, Al.y, 0x5140), ba3 = __byte_perm(B.y, Al.y, 0x7362);
        uint4 *o = reinterpret_cast<uint4 *>(row);
        o[0] = make_uint4(__byte_perm(rg0, ba0, 0x5410), __byte_perm(rg0, ba0, 0x7632), __byte_perm(rg1, ba1, 0x5410), __byte_perm(rg1, ba1, 0x7632));
        o[1] = make_uint4(__byte_perm(rg2, ba2, 0x5410), __byte_perm(rg2, ba2, 0x7632), __byte_perm(rg3, ba3, 0x5410), __byte_perm(rg3, ba3, 0x7632));
    }
}

template <int C, int V>
__device__ __forceinline__ void ws_defragment_slab(const DctParams &p, const WsAes &A, uint32_t *kb, uint32_t *pb, unsigned sg, int s, int lane) {
    constexpr ZigzagTable ZZ = make_zigzag();
    const WsStrip S = ws_decode_strip(p, sg, lane);
    if (!S.valid) return;
    const int P = p.k + 1, Q = 63 - p.k;
    const uint32_t *priv = reinterpret_cast<const uint32_t *>(p.priv + (size_t)S.n * p.priv_stride);
    const uint32_t *pub = reinterpret_cast<const uint32_t *>(p.pub + (size_t)S.n * p.pub_stride);
    uint32_t nonce[4];
    load_nonce(p, S.n, nonce);
#pragma unroll 1
    for (int ch = 0; ch < C; ++ch) {
        const size_t blk = ((size_t)(ch * p.nbr + S.br) * p.nbc) + (size_t)S.g * G_BLOCKS + s;
        const unsigned long long w0 = (unsigned long long)blk * P;
        ws_keystream(p, A, nonce, w0, P, kb);
        const uint32_t *kv = kb + (int)(w0 & 3);
        const uint32_t *pv = priv + w0;
        const uint32_t *pq = pub + blk * (size_t)Q - P;
        float v[64];
#pragma unroll
        for (int g = 0; g < 64; g += V) {
            uint32_t x[V];
            if (g < P) {
                uint32_t ks[V];
                vec_load_global<V>(pv + g, x);
                vec_load<V>(kv + g, ks);
#pragma unroll
                for (int t = 0; t < V; ++t) x[t] ^= ks[t];
            } else {
                vec_load_global<V>(pq + g, x);
            }
#pragma unroll
            for (int t = 0; t < V; ++t) v[ZZ.pos[g + t]] = __uint_as_float(x[t]);
        }
        idct8x8(v);
#pragma unroll
        for (int r = 0; r < 8; r += 2) {   // rounded, saturated, packed: two words per row (A5)
            const uint4 q = make_uint4(pack4_u8(v[8 * r], v[8 * r + 1], v[8 * r + 2], v[8 * r + 3]),
                                       pack4_u8(v[8 * r + 4], v[8 * r + 5], v[8 * r + 6], v[8 * r + 7]),
                                       pack4_u8(v[8 * r + 8], v[8 * r + 9], v[8 * r + 10], v[8 * r + 11]),
                                       pack4_u8(v[8 * r + 12], v[8 * r + 13], v[8 * r + 14], v[8 * r + 15]));
            *reinterpret_cast<uint4 *>(pb + 16 * ch + 2 * r) = q;
        }
    }
    uint8_t *img = p.images_out + (size_t)S.n * p.image_stride;
    const int x0 = 8 * (S.g * G_BLOCKS + s);
#pragma unroll
    for (int r = 0; r < 8; ++r) ws_store_row<C>(img + ((size_t)(8 * S.br + r) * p.w + x0) * C, pb, r);
}

// ------------------------------------------------------------------------------------------------------------
// kernels
// ------------------------------------------------------------------------------------------------------------
template <int C, int V, bool FRAGMENT>
__global__ void __launch_bounds__(WS_THREADS, 1) dct_ws_kernel(const __grid_constant__ DctParams p) {
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *s_kb = smem + WS_TABLE_WORDS;
    uint32_t *s_pb = s_kb + WS_WORK_WARPS * 32 * WS_KB_STRIDE;
    int *s_ctl = reinterpret_cast<int *>(s_pb + WS_WORK_WARPS * 32 * WS_PB_STRIDE);
    {
        const uint32_t *src = &g_aes.T[0][0];
        for (int i = threadIdx.x; i < WS_TABLE_WORDS; i += WS_THREADS) smem[i] = src[i >> 5];
        if (threadIdx.x < 64) s_ctl[threadIdx.x] = 0;
        __syncthreads();
    }
    WsCtrl ctl;
    ctl.ready = s_ctl;
    ctl.consumed = s_ctl + 32;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp < WS_HASH_WARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(WS_HASH_REGS));
        if (warp < WsShape<C>::UNITS * C) ws_hash_role<C>(p, ctl, warp, lane);
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(WS_WORK_REGS));
        const int pw = warp - WS_HASH_WARPS;
        WsAes A;
        A.base = (uint32_t)__cvta_generic_to_shared(smem) + 4u * lane;
        A.c128 = p.c128;
        uint32_t *kb = s_kb + (pw * 32 + lane) * WS_KB_STRIDE;
        uint32_t *pb = s_pb + (pw * 32 + lane) * WS_PB_STRIDE;
        if (FRAGMENT) {
            ws_worker_schedule<C>(p, ctl, pw, lane, [&](unsigned sg, int s) { ws_fragment_slab<C, V>(p, A, kb, sg, s, lane); });
        } else {
            ws_worker_schedule<C>(p, ctl, pw, lane, [&](unsigned sg, int s) { ws_defragment_slab<C, V>(p, A, kb, pb, sg, s, lane); });
        }
    }
}

}  // namespace feds
