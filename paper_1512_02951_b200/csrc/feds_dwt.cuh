// feds_dwt.cuh — Le Gall 5/3 integer lifting, one dyadic level per launch.
//   forward : d[n] = x[2n+1] - floor((x[2n] + x[2n+2]) / 2);  s[n] = x[2n] + floor((d[n-1] + d[n] + 2) / 4)
//   inverse : x[2n] = s[n] - floor((d[n-1] + d[n] + 2) / 4);  x[2n+1] = d[n] + floor((x[2n] + x[2n+2]) / 2)
// with x[N] = x[N-2], d[-1] = d[0] (P:755-762 in the DESIGN.md A12/A14 reading); rows then columns forward
// (P:812), columns then rows inverse. A CTA transforms one tile with its halo staged in shared memory; integer
// arithmetic makes the result independent of the tiling. Arithmetic shifts are floors (toward -inf).
// Global traffic is vectorised wherever the addresses allow (aligned 4-byte loads of 4 pixels / 2 coefficients,
// 8/16-byte stores of 4/8/16 outputs); out-of-range or misaligned pieces fall back to mirrored scalar accesses.
#pragma once
#include "feds_device.cuh"

namespace feds {

constexpr int DWT_TW = 64;   // output (subband) columns per tile
constexpr int DWT_TH = 16;   // output (subband) rows per tile
constexpr int DWT_THREADS = 256;

__device__ __forceinline__ int mirror_idx(int i, int n) {  // whole-sample symmetric extension, then clamp
    if (i < 0) i = -i;
    if (i >= n) i = 2 * (n - 1) - i;
    return min(max(i, 0), n - 1);
}

struct DwtLevelParams {
    // forward: input = u8 image (first level) or the previous LL plane; inverse: output likewise
    const uint8_t *img_in;   // [n][h][w][C] uint8 (FIRST only)
    uint8_t *img_out;        // inverse LAST only
    size_t image_stride;
    int C;
    int img_w;               // full image width (pixel pitch of the u8 image)
    const int16_t *ll_in;    // forward (not FIRST): current LL plane of plane p at ll_in + p*ll_in_plane_stride, pitch cw
    int16_t *ll_out_plane;   // inverse (not LAST): reconstructed LL_{l-1} plane, pitch cw
    size_t ll_in_plane_stride, ll_out_plane_stride;  // in elements; plane index = n*C + c
    int cw, ch;              // size of the level's input (forward) / output (inverse): 2*bw x 2*bh
    // subband storage. LL of this level: either a workspace plane or the private fragment (last forward level / first inverse level)
    int16_t *ll_band;        // base for plane (n, c): ll_band + n*ll_band_image_stride + c*ll_band_chan_stride (elements)
    size_t ll_band_image_stride, ll_band_chan_stride;
    int16_t *pub;            // public fragment base; band b (0 HL, 1 LH, 2 HH) of plane (n,c) at
                             // pub + n*pub_image_stride + c*pub_chan_stride + level_off + b*bw*bh (elements)
    size_t pub_image_stride, pub_chan_stride, level_off;
    int rows;                // streaming kernels (feds_dwt_fast.cuh): subband rows per warp tile
};

__device__ __forceinline__ bool aligned8(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 7u) == 0; }
__device__ __forceinline__ uint32_t pack16(int a, int b) { return ((uint32_t)a & 0xffffu) | ((uint32_t)b << 16); }

// ------------------------------------------------------------------------------------------------------------
// forward level
// ------------------------------------------------------------------------------------------------------------
template <bool FIRST>
__global__ void __launch_bounds__(DWT_THREADS) dwt_fwd_level_kernel(const __grid_constant__ DwtLevelParams p) {
    constexpr int IR = 2 * DWT_TH + 3, IC = 2 * DWT_TW + 3;
    __shared__ int16_t sIn[IR][IC + 1];
    __shared__ int16_t sHd[IR][DWT_TW + 2];   // horizontal high-pass, index n - (tx0-1)
    __shared__ int16_t sHs[IR][DWT_TW];       // horizontal low-pass, index n - tx0
    __shared__ int16_t sVd[DWT_TH + 1][2 * DWT_TW];  // vertical high-pass of [sHs | sHd], row index m - (ty0-1)

    const int plane = blockIdx.z;  // n*C + c
    const int n = plane / p.C, c = plane % p.C;
    const int tx0 = blockIdx.x * DWT_TW, ty0 = blockIdx.y * DWT_TH;
    const int bw = p.cw >> 1, bh = p.ch >> 1;
    const int tid = threadIdx.x;

    // stage A: input tile with halo (mirrored at the borders); local column lx <-> x = 2*tx0 - 2 + lx
    if (FIRST) {
        const uint8_t *img = p.img_in + (size_t)n * p.image_stride;
        if (p.C == 1 && (p.img_w & 3) == 0) {
            constexpr int NW = (IC + 2 + 3) / 4 + 1;  // aligned 4-pixel words covering x in [2*tx0 - 4, 2*tx0 + 2*TW + 4)
            for (int i = tid; i < IR * NW; i += DWT_THREADS) {
                const int ly = i / NW, j = i % NW;
                const int y = mirror_idx(2 * ty0 - 2 + ly, p.ch), xw = 2 * tx0 - 4 + 4 * j;
                const uint8_t *row = img + (size_t)y * p.img_w;
                uint32_t q;
                if (xw >= 0 && xw + 3 < p.cw) q = __ldg(reinterpret_cast<const uint32_t *>(row + xw));
                else q = (uint32_t)row[mirror_idx(xw, p.cw)] | ((uint32_t)row[mirror_idx(xw + 1, p.cw)] << 8) |
                         ((uint32_t)row[mirror_idx(xw + 2, p.cw)] << 16) | ((uint32_t)row[mirror_idx(xw + 3, p.cw)] << 24);
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                    const int lx = 4 * j - 2 + t;
                    if (lx >= 0 && lx < IC) sIn[ly][lx] = (int16_t)((int)((q >> (8 * t)) & 0xffu) - 128);
                }
            }
        } else {
            for (int i = tid; i < IR * IC; i += DWT_THREADS) {
                const int ly = i / IC, lx = i % IC;
                const int y = mirror_idx(2 * ty0 - 2 + ly, p.ch), x = mirror_idx(2 * tx0 - 2 + lx, p.cw);
                sIn[ly][lx] = (int16_t)((int)img[((size_t)y * p.img_w + x) * p.C + c] - 128);
            }
        }
    } else {
        const int16_t *pl = p.ll_in + (size_t)plane * p.ll_in_plane_stride;
        constexpr int NP = (IC + 1) / 2;  // aligned coefficient pairs covering x in [2*tx0 - 2, 2*tx0 + 2*TW + 2)
        for (int i = tid; i < IR * NP; i += DWT_THREADS) {
            const int ly = i / NP, j = i % NP;
            const int y = mirror_idx(2 * ty0 - 2 + ly, p.ch), x = 2 * tx0 - 2 + 2 * j;
            const int16_t *row = pl + (size_t)y * p.cw;
            int a, b;
            if (x >= 0 && x + 1 < p.cw) {
                const uint32_t q = __ldg(reinterpret_cast<const uint32_t *>(row + x));
                a = (int16_t)(q & 0xffffu); b = (int16_t)(q >> 16);
            } else {
                a = row[mirror_idx(x, p.cw)]; b = row[mirror_idx(x + 1, p.cw)];
            }
            sIn[ly][2 * j] = (int16_t)a;
            if (2 * j + 1 < IC) sIn[ly][2 * j + 1] = (int16_t)b;
        }
    }
    __syncthreads();
    // stage B: horizontal predict, d[n] for n in [tx0-1, tx0+TW)
    for (int i = tid; i < IR * (DWT_TW + 1); i += DWT_THREADS) {
        const int ly = i / (DWT_TW + 1), j = i % (DWT_TW + 1);  // j = n - (tx0-1); local col of x[2n] = 2j
        const int d = (int)sIn[ly][2 * j + 1] - (((int)sIn[ly][2 * j] + (int)sIn[ly][2 * j + 2]) >> 1);
        sHd[ly][j] = (int16_t)d;
    }
    __syncthreads();
    // horizontal update, s[n] for n in [tx0, tx0+TW)
    for (int i = tid; i < IR * DWT_TW; i += DWT_THREADS) {
        const int ly = i / DWT_TW, j = i % DWT_TW;  // n = tx0 + j; x[2n] at local col 2j+2; d[n-1] = sHd[j], d[n] = sHd[j+1]
        const int s = (int)sIn[ly][2 * j + 2] + (((int)sHd[ly][j] + (int)sHd[ly][j + 1] + 2) >> 2);
        sHs[ly][j] = (int16_t)s;
    }
    __syncthreads();
    // stage C: vertical predict on both halves, d[m] for m in [ty0-1, ty0+TH); column q < TW: low half, else high half
    for (int i = tid; i < (DWT_TH + 1) * 2 * DWT_TW; i += DWT_THREADS) {
        const int r = i / (2 * DWT_TW), q = i % (2 * DWT_TW);  // r = m - (ty0-1); local row of x[2m] = 2r
        int a, b, e;
        if (q < DWT_TW) { a = sHs[2 * r][q]; b = sHs[2 * r + 1][q]; e = sHs[2 * r + 2][q]; }
        else { a = sHd[2 * r][q - DWT_TW + 1]; b = sHd[2 * r + 1][q - DWT_TW + 1]; e = sHd[2 * r + 2][q - DWT_TW + 1]; }
        sVd[r][q] = (int16_t)(b - ((a + e) >> 1));
    }
    __syncthreads();
    // vertical update + stores: LL/HL get s, LH/HH get d. One item = 4 adjacent columns of one row of one half.
    int16_t *llb = p.ll_band + (size_t)n * p.ll_band_image_stride + (size_t)c * p.ll_band_chan_stride;
    int16_t *pb = p.pub + (size_t)n * p.pub_image_stride + (size_t)c * p.pub_chan_stride + p.level_off;
    const size_t band = (size_t)bw * bh;
    const bool vec_ok = (bw & 3) == 0 && aligned8(llb) && aligned8(pb) && aligned8(pb + band) && aligned8(pb + 2 * band);
    for (int i = tid; i < DWT_TH * 2 * (DWT_TW / 4); i += DWT_THREADS) {
        const int r = i / (2 * (DWT_TW / 4)), rem = i % (2 * (DWT_TW / 4));
        const bool high = rem >= DWT_TW / 4;
        const int j0 = 4 * (high ? rem - DWT_TW / 4 : rem);
        const int m = ty0 + r, nn0 = tx0 + j0;
        if (m >= bh || nn0 >= bw) continue;
        int sv[4], dv[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            const int j = j0 + t, q = high ? DWT_TW + j : j;
            const int x2m = high ? (int)sHd[2 * r + 2][j + 1] : (int)sHs[2 * r + 2][j];
            const int dprev = sVd[r][q], dcur = sVd[r + 1][q];
            sv[t] = x2m + ((dprev + dcur + 2) >> 2);
            dv[t] = dcur;
        }
        const size_t o = (size_t)m * bw + nn0;
        int16_t *ps = high ? pb + 0 * band + o : llb + o;         // HL or LL
        int16_t *pd = high ? pb + 2 * band + o : pb + 1 * band + o;  // HH or LH
        if (vec_ok && nn0 + 3 < bw) {
            *reinterpret_cast<uint2 *>(ps) = make_uint2(pack16(sv[0], sv[1]), pack16(sv[2], sv[3]));
            *reinterpret_cast<uint2 *>(pd) = make_uint2(pack16(dv[0], dv[1]), pack16(dv[2], dv[3]));
        } else {
#pragma unroll
            for (int t = 0; t < 4; ++t)
                if (nn0 + t < bw) { ps[t] = (int16_t)sv[t]; pd[t] = (int16_t)dv[t]; }
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// inverse level: (LL, HL, LH, HH) of size bh x bw -> plane of size 2bh x 2bw; LAST adds 128, clamps, stores uint8
// ------------------------------------------------------------------------------------------------------------
template <bool LAST>
__global__ void __launch_bounds__(DWT_THREADS) dwt_inv_level_kernel(const __grid_constant__ DwtLevelParams p) {
    constexpr int SR = DWT_TH + 2, SC = DWT_TW + 2;  // subband rows m in [ty0-1, ty0+TH], cols n in [tx0-1, tx0+TW]
    __shared__ int16_t sB[4][SR][SC + 2];            // 0 LL, 1 HL, 2 LH, 3 HH
    __shared__ int16_t sL[2 * DWT_TH + 1][SC + 2];   // after vertical synthesis: low-horizontal half, rows 2ty0 .. 2ty0+2TH
    __shared__ int16_t sH[2 * DWT_TH + 1][SC + 2];   // high-horizontal half
    __shared__ int16_t sE[2 * DWT_TH][DWT_TW + 2];   // even output columns x[2n], n in [tx0, tx0+TW]

    const int plane = blockIdx.z;
    const int n = plane / p.C, c = plane % p.C;
    const int tx0 = blockIdx.x * DWT_TW, ty0 = blockIdx.y * DWT_TH;
    const int bw = p.cw >> 1, bh = p.ch >> 1;
    const int tid = threadIdx.x;
    const int16_t *llb = p.ll_band + (size_t)n * p.ll_band_image_stride + (size_t)c * p.ll_band_chan_stride;
    const int16_t *pb = p.pub + (size_t)n * p.pub_image_stride + (size_t)c * p.pub_chan_stride + p.level_off;
    const size_t band = (size_t)bw * bh;

    // load the four bands with their halo; aligned pairs cover columns nn in [tx0-2, tx0+TW+2); lc = nn - (tx0-1)
    {
        constexpr int NP = (SC + 2) / 2;
        const bool pair_ok = (bw & 1) == 0 && (reinterpret_cast<uintptr_t>(llb) & 3u) == 0 && (reinterpret_cast<uintptr_t>(pb) & 3u) == 0 &&
                             (band & 1) == 0;
        for (int i = tid; i < 4 * SR * NP; i += DWT_THREADS) {
            const int b = i / (SR * NP), rem = i % (SR * NP), lr = rem / NP, j = rem % NP;
            const int m = min(max(ty0 - 1 + lr, 0), bh - 1);  // d[-1] = d[0]; rows beyond the end are never used
            const int16_t *src = (b == 0) ? llb : (b == 1) ? pb : (b == 2) ? pb + band : pb + 2 * band;
            src += (size_t)m * bw;
            const int nn = tx0 - 2 + 2 * j;
            int a, e;
            if (pair_ok && nn >= 0 && nn + 1 < bw) {
                const uint32_t q = __ldg(reinterpret_cast<const uint32_t *>(src + nn));
                a = (int16_t)(q & 0xffffu); e = (int16_t)(q >> 16);
            } else {
                a = src[min(max(nn, 0), bw - 1)]; e = src[min(max(nn + 1, 0), bw - 1)];
            }
            const int lc = 2 * j - 1;
            if (lc >= 0) sB[b][lr][lc] = (int16_t)a;
            if (lc + 1 < SC) sB[b][lr][lc + 1] = (int16_t)e;
        }
    }
    __syncthreads();
    // vertical synthesis, even rows x[2m], m in [ty0, ty0+TH] (local r = 0..TH), all SC columns, both halves
    for (int i = tid; i < (DWT_TH + 1) * SC * 2; i += DWT_THREADS) {
        const int half = i / ((DWT_TH + 1) * SC), rem = i % ((DWT_TH + 1) * SC), r = rem / SC, lc = rem % SC;
        const int sb = half ? 1 : 0, db = half ? 3 : 2;  // low-horizontal: (LL, LH); high-horizontal: (HL, HH)
        const int s = sB[sb][r + 1][lc], dprev = sB[db][r][lc], dcur = sB[db][r + 1][lc];
        const int16_t x = (int16_t)(s - ((dprev + dcur + 2) >> 2));
        if (half) sH[2 * r][lc] = x; else sL[2 * r][lc] = x;
    }
    __syncthreads();
    // odd rows x[2m+1], m in [ty0, ty0+TH): uses x[2m], x[2m+2] (x[2bh] = x[2bh-2])
    for (int i = tid; i < DWT_TH * SC * 2; i += DWT_THREADS) {
        const int half = i / (DWT_TH * SC), rem = i % (DWT_TH * SC), r = rem / SC, lc = rem % SC;
        const int db = half ? 3 : 2;
        const int m = ty0 + r;
        const int16_t(*S)[SC + 2] = half ? sH : sL;
        const int a = S[2 * r][lc];
        const int e = (m + 1 < bh) ? (int)S[2 * r + 2][lc] : a;
        const int16_t x = (int16_t)((int)sB[db][r + 1][lc] + ((a + e) >> 1));
        if (half) sH[2 * r + 1][lc] = x; else sL[2 * r + 1][lc] = x;
    }
    __syncthreads();
    // horizontal synthesis, even columns x[2n], n in [tx0, tx0+TW] (local j = 0..TW): s = sL[.][j+1], d = sH[.][j], sH[.][j+1]
    for (int i = tid; i < 2 * DWT_TH * (DWT_TW + 1); i += DWT_THREADS) {
        const int ry = i / (DWT_TW + 1), j = i % (DWT_TW + 1);
        sE[ry][j] = (int16_t)((int)sL[ry][j + 1] - (((int)sH[ry][j] + (int)sH[ry][j + 1] + 2) >> 2));
    }
    __syncthreads();
    // outputs: one item = 16 adjacent output columns (8 even + 8 odd) of one row
    const bool vec_ok = LAST ? (p.C == 1 && (p.img_w & 15) == 0 && (reinterpret_cast<uintptr_t>(p.img_out) & 15u) == 0 && (p.image_stride & 15u) == 0)
                             : ((p.cw & 7) == 0 && (reinterpret_cast<uintptr_t>(p.ll_out_plane) & 15u) == 0 && (p.ll_out_plane_stride & 7u) == 0);
    for (int i = tid; i < 2 * DWT_TH * (2 * DWT_TW / 16); i += DWT_THREADS) {
        const int ry = i / (2 * DWT_TW / 16), cx0 = 16 * (i % (2 * DWT_TW / 16));
        const int y = 2 * ty0 + ry, x0 = 2 * tx0 + cx0;
        if (y >= p.ch || x0 >= p.cw) continue;
        int v[16];
#pragma unroll
        for (int t = 0; t < 8; ++t) {
            const int j = (cx0 >> 1) + t;
            const int a = sE[ry][j];
            const int e = (tx0 + j + 1 < bw) ? (int)sE[ry][j + 1] : a;
            v[2 * t] = a;
            v[2 * t + 1] = (int)sH[ry][j + 1] + ((a + e) >> 1);
        }
        if (LAST) {
#pragma unroll
            for (int t = 0; t < 16; ++t) v[t] = min(max(v[t] + 128, 0), 255);
            uint8_t *dst = p.img_out + (size_t)n * p.image_stride + ((size_t)y * p.img_w + x0) * p.C + c;
            if (vec_ok && x0 + 15 < p.cw) {
                uint4 q;
                q.x = (uint32_t)v[0] | ((uint32_t)v[1] << 8) | ((uint32_t)v[2] << 16) | ((uint32_t)v[3] << 24);
                q.y = (uint32_t)v[4] | ((uint32_t)v[5] << 8) | ((uint32_t)v[6] << 16) | ((uint32_t)v[7] << 24);
                q.z = (uint32_t)v[8] | ((uint32_t)v[9] << 8) | ((uint32_t)v[10] << 16) | ((uint32_t)v[11] << 24);
                q.w = (uint32_t)v[12] | ((uint32_t)v[13] << 8) | ((uint32_t)v[14] << 16) | ((uint32_t)v[15] << 24);
                *reinterpret_cast<uint4 *>(dst) = q;
            } else {
#pragma unroll
                for (int t = 0; t < 16; ++t)
                    if (x0 + t < p.cw) dst[(size_t)t * p.C] = (uint8_t)v[t];
            }
        } else {
            int16_t *dst = p.ll_out_plane + (size_t)plane * p.ll_out_plane_stride + (size_t)y * p.cw + x0;
            if (vec_ok && x0 + 15 < p.cw) {
                uint4 *d4 = reinterpret_cast<uint4 *>(dst);
                d4[0] = make_uint4(pack16(v[0], v[1]), pack16(v[2], v[3]), pack16(v[4], v[5]), pack16(v[6], v[7]));
                d4[1] = make_uint4(pack16(v[8], v[9]), pack16(v[10], v[11]), pack16(v[12], v[13]), pack16(v[14], v[15]));
            } else {
#pragma unroll
                for (int t = 0; t < 16; ++t)
                    if (x0 + t < p.cw) dst[t] = (int16_t)v[t];
            }
        }
    }
}

}  // namespace feds
