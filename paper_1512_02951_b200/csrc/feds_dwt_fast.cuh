// feds_dwt_fast.cuh — register-streaming Le Gall 5/3 level kernels for levels whose
// width is a multiple of the per-thread pixel run and whose buffers are 16-byte aligned; everything else takes the tiled
// shared-memory kernels of feds_dwt.cuh. Same arithmetic, so the result is bit-identical.
//
// A thread owns PX adjacent pixels (all C channels when the data is the interleaved uint8 image, one plane otherwise) and
// walks down R subband rows. Horizontal lifting takes its two neighbour values from the adjacent lanes with shuffles;
// lanes 0 and 31 of every warp are halo lanes (warps overlap by one lane on each side), so no shared memory and no
// barrier is needed. Vertical lifting is a running recurrence down the rows: the thread keeps the previous even row and
// the previous high-pass row in registers. Every global access is a 64/128-bit access of one lane's contiguous run.
#pragma once
#include "feds_dwt.cuh"

namespace feds {

constexpr int DWTF_WARPS = 4;         // warps per CTA, stacked vertically (consecutive row tiles of one column strip)
constexpr int DWTF_ROWS = 16;         // subband rows per warp tile on large levels; DwtLevelParams::rows (16, 8 or 4) is what a launch uses:
                                      // small levels take shorter tiles so that the grid still fills the SMs (each tile re-reads 3 halo rows)
constexpr int DWTF_LANES_OUT = 30;    // lanes 1..30 write; 0 and 31 are halo

template <int N>
__device__ __forceinline__ void load_bytes(const uint8_t *src, uint32_t (&w)[N / 4]) {
    if (N == 16) {
        const uint4 q = __ldg(reinterpret_cast<const uint4 *>(src));
        w[0] = q.x; w[1 % (N / 4)] = q.y; w[2 % (N / 4)] = q.z; w[3 % (N / 4)] = q.w;
    } else {
#pragma unroll
        for (int i = 0; i < N / 8; ++i) {
            const uint2 q = __ldg(reinterpret_cast<const uint2 *>(src) + i);
            w[2 * i] = q.x; w[2 * i + 1] = q.y;
        }
    }
}
template <int N>
__device__ __forceinline__ void store_bytes(uint8_t *dst, const uint32_t (&w)[N / 4]) {
    if (N == 16) {
        *reinterpret_cast<uint4 *>(dst) = make_uint4(w[0], w[1 % (N / 4)], w[2 % (N / 4)], w[3 % (N / 4)]);
    } else {
#pragma unroll
        for (int i = 0; i < N / 8; ++i) reinterpret_cast<uint2 *>(dst)[i] = make_uint2(w[2 * i], w[2 * i + 1]);
    }
}
// N int16 values <-> N ints; N = 4 (one 64-bit access), 8 (one 128-bit access) or 16 (two)
template <int N>
__device__ __forceinline__ void load_i16(const int16_t *src, int (&v)[N]) {
    uint32_t w[N / 2];
    if (N == 4) {
        const uint2 q = __ldg(reinterpret_cast<const uint2 *>(src));
        w[0] = q.x; w[1] = q.y;
    } else {
#pragma unroll
        for (int i = 0; i < N / 8; ++i) {
            const uint4 q = __ldg(reinterpret_cast<const uint4 *>(src) + i);
            w[4 * i] = q.x; w[4 * i + 1] = q.y; w[4 * i + 2] = q.z; w[4 * i + 3] = q.w;
        }
    }
#pragma unroll
    for (int i = 0; i < N / 2; ++i) { v[2 * i] = (int)(int16_t)(w[i] & 0xffffu); v[2 * i + 1] = (int)w[i] >> 16; }
}
template <int N>
__device__ __forceinline__ void store_i16(int16_t *dst, const int (&v)[N]) {
    uint32_t w[N / 2];
#pragma unroll
    for (int i = 0; i < N / 2; ++i) w[i] = __byte_perm((uint32_t)v[2 * i], (uint32_t)v[2 * i + 1], 0x5410);
    if (N == 4) {
        *reinterpret_cast<uint2 *>(dst) = make_uint2(w[0], w[1]);
    } else {
#pragma unroll
        for (int i = 0; i < N / 8; ++i) reinterpret_cast<uint4 *>(dst)[i] = make_uint4(w[4 * i], w[4 * i + 1], w[4 * i + 2], w[4 * i + 3]);
    }
}

// ------------------------------------------------------------------------------------------------------------
// forward level. U8: input is the interleaved uint8 image (level 1), C channels per pixel; else one int16 plane (C = 1 here,
// the plane index comes from blockIdx.z). A row of a thread is NV = PX*C values v[p*C + ch].
// After horizontal lifting the row is h[half][q][ch], q = 0..HP-1 (half 0: low-pass s, half 1: high-pass d).
// ------------------------------------------------------------------------------------------------------------
template <int C, int PX, bool U8>
struct FwdRow {
    static constexpr int NV = PX * C, HP = PX / 2;
    static constexpr int RAW = U8 ? NV / 4 : NV / 2;   // 32-bit words of one row of this lane's run as loaded
    // image / plane row y of the lane's run starting at pixel px0, as loaded (the loop keeps the next two rows in flight)
    static __device__ __forceinline__ void load(const DwtLevelParams &p, const void *base, int y, int px0, bool in_range, uint32_t (&w)[RAW]) {
        if (in_range) {
            if (U8) {
                load_bytes<NV>(static_cast<const uint8_t *>(base) + ((size_t)y * p.img_w + px0) * C, reinterpret_cast<uint32_t(&)[NV / 4]>(w));
            } else {
                const uint4 *src = reinterpret_cast<const uint4 *>(static_cast<const int16_t *>(base) + (size_t)y * p.cw + px0);
                if (NV == 4) {
                    const uint2 q = __ldg(reinterpret_cast<const uint2 *>(src));
                    w[0] = q.x; w[1 % RAW] = q.y;
                } else {
#pragma unroll
                    for (int i = 0; i < NV / 8; ++i) {
                        const uint4 q = __ldg(src + i);
                        w[(4 * i) % RAW] = q.x; w[(4 * i + 1) % RAW] = q.y; w[(4 * i + 2) % RAW] = q.z; w[(4 * i + 3) % RAW] = q.w;
                    }
                }
            }
        } else {
#pragma unroll
            for (int i = 0; i < RAW; ++i) w[i] = U8 ? 0x80808080u : 0u;   // lifts to zeros
        }
    }
    static __device__ __forceinline__ void get(const DwtLevelParams &p, const void *base, int y, int px0, bool in_range, bool first_run,
                                               bool last_run, int (&lo)[HP * C], int (&hi)[HP * C]) {
        uint32_t w[RAW];
        load(p, base, y, px0, in_range, w);
        lift(w, first_run, last_run, lo, hi);
    }
    // horizontal lifting of a loaded row
    static __device__ __forceinline__ void lift(const uint32_t (&w)[RAW], bool first_run, bool last_run, int (&lo)[HP * C], int (&hi)[HP * C]) {
        int v[NV];
        if (U8) {
#pragma unroll
            for (int i = 0; i < NV; ++i) v[i] = (int)((w[i >> 2] >> (8 * (i & 3))) & 0xffu) - 128;
        } else {
#pragma unroll
            for (int i = 0; i < NV / 2; ++i) { v[2 * i] = (int)(int16_t)(w[i % RAW] & 0xffffu); v[2 * i + 1] = (int)w[i % RAW] >> 16; }
        }
        int rn[C];  // x[PX] of this run = the right neighbour's first pixel; x[cw] = x[cw-2] at the image border
#pragma unroll
        for (int ch = 0; ch < C; ++ch) {
            rn[ch] = __shfl_down_sync(0xffffffffu, v[ch], 1);
            if (last_run) rn[ch] = v[(PX - 2) * C + ch];
        }
#pragma unroll
        for (int q = 0; q < HP; ++q)
#pragma unroll
            for (int ch = 0; ch < C; ++ch) {
                const int a = v[2 * q * C + ch], b = (q < HP - 1) ? v[(2 * q + 2) * C + ch] : rn[ch];
                hi[q * C + ch] = v[(2 * q + 1) * C + ch] - ((a + b) >> 1);
            }
#pragma unroll
        for (int ch = 0; ch < C; ++ch) {
            int ln = __shfl_up_sync(0xffffffffu, hi[(HP - 1) * C + ch], 1);  // d[-1] of this run; d[-1] = d[0] at the border
            if (first_run) ln = hi[ch];
#pragma unroll
            for (int q = 0; q < HP; ++q) {
                const int dp = (q > 0) ? hi[(q - 1) * C + ch] : ln;
                lo[q * C + ch] = v[2 * q * C + ch] + ((dp + hi[q * C + ch] + 2) >> 2);
            }
        }
    }
};

template <int C, int PX, bool U8>
__global__ void __launch_bounds__(DWTF_WARPS * 32) dwt_fwd_fast_kernel(const __grid_constant__ DwtLevelParams p) {
    constexpr int HP = PX / 2, NH = HP * C;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int bw = p.cw >> 1, bh = p.ch >> 1;
    const int px0 = ((int)blockIdx.x * DWTF_LANES_OUT + lane - 1) * PX;
    const bool in_range = px0 >= 0 && px0 < p.cw;
    const bool writer = in_range && lane >= 1 && lane <= DWTF_LANES_OUT;
    const bool first_run = px0 == 0, last_run = px0 + PX == p.cw;
    const int m0 = ((int)blockIdx.y * DWTF_WARPS + warp) * p.rows;
    if (m0 >= bh) return;  // whole warp
    const int m1 = min(m0 + p.rows, bh);
    // plane bookkeeping: U8 -> blockIdx.z = image n, all C channels here; else blockIdx.z = plane index n*Cimg + c
    const int n = U8 ? (int)blockIdx.z : (int)blockIdx.z / p.C, c0 = U8 ? 0 : (int)blockIdx.z % p.C;
    const void *base = U8 ? static_cast<const void *>(p.img_in + (size_t)n * p.image_stride)
                          : static_cast<const void *>(p.ll_in + (size_t)blockIdx.z * p.ll_in_plane_stride);
    const size_t band = (size_t)bw * bh;
    const int bc0 = px0 >> 1;
    using Row = FwdRow<C, PX, U8>;

    int Elo[NH], Ehi[NH], Plo[NH], Phi[NH];  // even row h[2m]; previous vertical high-pass d[m-1] (both halves)
    if (m0 > 0) {
        int Olo[NH], Ohi[NH], Nlo[NH], Nhi[NH];
        Row::get(p, base, 2 * m0 - 2, px0, in_range, first_run, last_run, Elo, Ehi);
        Row::get(p, base, 2 * m0 - 1, px0, in_range, first_run, last_run, Olo, Ohi);
        Row::get(p, base, 2 * m0, px0, in_range, first_run, last_run, Nlo, Nhi);
#pragma unroll
        for (int i = 0; i < NH; ++i) {
            Plo[i] = Olo[i] - ((Elo[i] + Nlo[i]) >> 1);
            Phi[i] = Ohi[i] - ((Ehi[i] + Nhi[i]) >> 1);
            Elo[i] = Nlo[i]; Ehi[i] = Nhi[i];
        }
    } else {
        Row::get(p, base, 0, px0, in_range, first_run, last_run, Elo, Ehi);
#pragma unroll
        for (int i = 0; i < NH; ++i) { Plo[i] = 0; Phi[i] = 0; }
    }
    uint32_t rO[Row::RAW], rN[Row::RAW];   // rows 2m+1 and 2m+2 as loaded, one iteration ahead of their use (two ahead gained nothing)
    Row::load(p, base, 2 * m0 + 1, px0, in_range, rO);
    Row::load(p, base, min(2 * m0 + 2, p.ch - 1), px0, in_range, rN);
#pragma unroll 1
    for (int m = m0; m < m1; ++m) {
        uint32_t nO[Row::RAW], nN[Row::RAW];
        if (m + 1 < m1) {
            Row::load(p, base, 2 * m + 3, px0, in_range, nO);
            Row::load(p, base, min(2 * m + 4, p.ch - 1), px0, in_range, nN);
        }
        int Olo[NH], Ohi[NH], Nlo[NH], Nhi[NH];
        Row::lift(rO, first_run, last_run, Olo, Ohi);
        if (2 * m + 2 < p.ch) {
            Row::lift(rN, first_run, last_run, Nlo, Nhi);
        } else {  // h[ch] = h[ch-2]
#pragma unroll
            for (int i = 0; i < NH; ++i) { Nlo[i] = Elo[i]; Nhi[i] = Ehi[i]; }
        }
#pragma unroll
        for (int i = 0; i < Row::RAW; ++i) { rO[i] = nO[i]; rN[i] = nN[i]; }
        int Slo[NH], Shi[NH];
#pragma unroll
        for (int i = 0; i < NH; ++i) {
            const int dl = Olo[i] - ((Elo[i] + Nlo[i]) >> 1), dh = Ohi[i] - ((Ehi[i] + Nhi[i]) >> 1);
            const int pl = (m == 0) ? dl : Plo[i], ph = (m == 0) ? dh : Phi[i];  // d[-1] = d[0]
            Slo[i] = Elo[i] + ((pl + dl + 2) >> 2);
            Shi[i] = Ehi[i] + ((ph + dh + 2) >> 2);
            Plo[i] = dl; Phi[i] = dh;
            Elo[i] = Nlo[i]; Ehi[i] = Nhi[i];
        }
        if (writer) {
#pragma unroll
            for (int ch = 0; ch < C; ++ch) {
                const int cc = c0 + ch;
                int16_t *llb = p.ll_band + (size_t)n * p.ll_band_image_stride + (size_t)cc * p.ll_band_chan_stride;
                int16_t *pb = p.pub + (size_t)n * p.pub_image_stride + (size_t)cc * p.pub_chan_stride + p.level_off;
                const size_t o = (size_t)m * bw + bc0;
                int t0[HP], t1[HP], t2[HP], t3[HP];
#pragma unroll
                for (int q = 0; q < HP; ++q) { t0[q] = Slo[q * C + ch]; t1[q] = Shi[q * C + ch]; t2[q] = Plo[q * C + ch]; t3[q] = Phi[q * C + ch]; }
                store_i16<HP>(llb + o, t0);             // LL: low-pass both ways
                store_i16<HP>(pb + o, t1);              // HL: high-pass horizontally
                store_i16<HP>(pb + band + o, t2);       // LH: high-pass vertically
                store_i16<HP>(pb + 2 * band + o, t3);   // HH
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// inverse level: vertical synthesis as a running recurrence down the subband rows (both horizontal halves), then
// horizontal synthesis of each finished row with the neighbour values from the adjacent lanes.
// U8: the output is the interleaved uint8 image (level 1): + 128, clamp.
// ------------------------------------------------------------------------------------------------------------
template <int C, int PX, bool U8>
struct InvRow {
    static constexpr int NV = PX * C, HP = PX / 2;
    // row of vertically synthesised values (L = low-horizontal half, H = high-horizontal half) -> PX pixels, stored at row y
    static __device__ __forceinline__ void put(const DwtLevelParams &p, void *base, int y, int px0, bool writer, bool first_run, bool last_run,
                                               const int (&L)[HP * C], const int (&H)[HP * C]) {
        int v[NV];
#pragma unroll
        for (int ch = 0; ch < C; ++ch) {
            int hl = __shfl_up_sync(0xffffffffu, H[(HP - 1) * C + ch], 1);  // d[-1]; = d[0] at the border
            if (first_run) hl = H[ch];
            int e[HP];
#pragma unroll
            for (int q = 0; q < HP; ++q) e[q] = L[q * C + ch] - ((((q > 0) ? H[(q - 1) * C + ch] : hl) + H[q * C + ch] + 2) >> 2);
            int er = __shfl_down_sync(0xffffffffu, e[0], 1);  // x[PX] of this run; x[cw] = x[cw-2] at the border
            if (last_run) er = e[HP - 1];
#pragma unroll
            for (int q = 0; q < HP; ++q) {
                v[2 * q * C + ch] = e[q];
                v[(2 * q + 1) * C + ch] = H[q * C + ch] + ((e[q] + ((q < HP - 1) ? e[q + 1] : er)) >> 1);
            }
        }
        if (!writer) return;
        if (U8) {
            uint32_t w[NV / 4];
#pragma unroll
            for (int i = 0; i < NV / 4; ++i) {
                uint32_t x = 0;
#pragma unroll
                for (int t = 0; t < 4; ++t) x |= (uint32_t)min(max(v[4 * i + t] + 128, 0), 255) << (8 * t);
                w[i] = x;
            }
            store_bytes<NV>(static_cast<uint8_t *>(base) + ((size_t)y * p.img_w + px0) * C, w);
        } else {
            store_i16<NV>(static_cast<int16_t *>(base) + (size_t)y * p.cw + px0, v);
        }
    }
};

template <int C, int PX, bool U8>
__global__ void __launch_bounds__(DWTF_WARPS * 32) dwt_inv_fast_kernel(const __grid_constant__ DwtLevelParams p) {
    constexpr int HP = PX / 2, NH = HP * C;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int bw = p.cw >> 1, bh = p.ch >> 1;
    const int px0 = ((int)blockIdx.x * DWTF_LANES_OUT + lane - 1) * PX;
    const bool in_range = px0 >= 0 && px0 < p.cw;
    const bool writer = in_range && lane >= 1 && lane <= DWTF_LANES_OUT;
    const bool first_run = px0 == 0, last_run = px0 + PX == p.cw;
    const int m0 = ((int)blockIdx.y * DWTF_WARPS + warp) * p.rows;
    if (m0 >= bh) return;
    const int m1 = min(m0 + p.rows, bh);
    const int n = U8 ? (int)blockIdx.z : (int)blockIdx.z / p.C, c0 = U8 ? 0 : (int)blockIdx.z % p.C;
    void *base = U8 ? static_cast<void *>(p.img_out + (size_t)n * p.image_stride)
                    : static_cast<void *>(p.ll_out_plane + (size_t)blockIdx.z * p.ll_out_plane_stride);
    const size_t band = (size_t)bw * bh;
    const int bc0 = px0 >> 1;
    using Row = InvRow<C, PX, U8>;

    // subband row m of this lane's columns: s = (LL | HL), d = (LH | HH), index q*C + ch
    auto load_sd = [&](int m, int (&sl)[NH], int (&sh)[NH], int (&dl)[NH], int (&dh)[NH], bool want_s) {
        if (!in_range) {
#pragma unroll
            for (int i = 0; i < NH; ++i) { sl[i] = 0; sh[i] = 0; dl[i] = 0; dh[i] = 0; }
            return;
        }
#pragma unroll
        for (int ch = 0; ch < C; ++ch) {
            const int cc = c0 + ch;
            const int16_t *llb = p.ll_band + (size_t)n * p.ll_band_image_stride + (size_t)cc * p.ll_band_chan_stride;
            const int16_t *pb = p.pub + (size_t)n * p.pub_image_stride + (size_t)cc * p.pub_chan_stride + p.level_off;
            const size_t o = (size_t)m * bw + bc0;
            int t[HP];
            if (want_s) {
                load_i16<HP>(llb + o, t);
#pragma unroll
                for (int q = 0; q < HP; ++q) sl[q * C + ch] = t[q];
                load_i16<HP>(pb + o, t);
#pragma unroll
                for (int q = 0; q < HP; ++q) sh[q * C + ch] = t[q];
            }
            load_i16<HP>(pb + band + o, t);
#pragma unroll
            for (int q = 0; q < HP; ++q) dl[q * C + ch] = t[q];
            load_i16<HP>(pb + 2 * band + o, t);
#pragma unroll
            for (int q = 0; q < HP; ++q) dh[q * C + ch] = t[q];
        }
    };

    int Xl[NH], Xh[NH], Dl[NH], Dh[NH];  // x[2m] (vertically synthesised even row) and d[m], both halves
    {
        int sl[NH], sh[NH], pl[NH], ph[NH];
        load_sd(m0, sl, sh, Dl, Dh, true);
        if (m0 > 0) {
            int u0[NH], u1[NH];
            load_sd(m0 - 1, u0, u1, pl, ph, false);
        } else {
#pragma unroll
            for (int i = 0; i < NH; ++i) { pl[i] = Dl[i]; ph[i] = Dh[i]; }  // d[-1] = d[0]
        }
#pragma unroll
        for (int i = 0; i < NH; ++i) {
            Xl[i] = sl[i] - ((pl[i] + Dl[i] + 2) >> 2);
            Xh[i] = sh[i] - ((ph[i] + Dh[i] + 2) >> 2);
        }
    }
#pragma unroll 1
    for (int m = m0; m < m1; ++m) {
        int Nl[NH], Nh[NH], El[NH], Eh[NH];  // next even row x[2m+2], next d
        if (m + 1 < bh) {
            int sl[NH], sh[NH];
            load_sd(m + 1, sl, sh, El, Eh, true);
#pragma unroll
            for (int i = 0; i < NH; ++i) {
                Nl[i] = sl[i] - ((Dl[i] + El[i] + 2) >> 2);
                Nh[i] = sh[i] - ((Dh[i] + Eh[i] + 2) >> 2);
            }
        } else {  // x[2bh] = x[2bh-2]
#pragma unroll
            for (int i = 0; i < NH; ++i) { Nl[i] = Xl[i]; Nh[i] = Xh[i]; El[i] = 0; Eh[i] = 0; }
        }
        int Ol[NH], Oh[NH];
#pragma unroll
        for (int i = 0; i < NH; ++i) {
            Ol[i] = Dl[i] + ((Xl[i] + Nl[i]) >> 1);
            Oh[i] = Dh[i] + ((Xh[i] + Nh[i]) >> 1);
        }
        Row::put(p, base, 2 * m, px0, writer, first_run, last_run, Xl, Xh);
        Row::put(p, base, 2 * m + 1, px0, writer, first_run, last_run, Ol, Oh);
#pragma unroll
        for (int i = 0; i < NH; ++i) { Xl[i] = Nl[i]; Xh[i] = Nh[i]; Dl[i] = El[i]; Dh[i] = Eh[i]; }
    }
}

}  // namespace feds
