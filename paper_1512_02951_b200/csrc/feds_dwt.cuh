// feds_dwt.cuh — Le Gall 5/3 integer lifting, one dyadic level per launch.
//   forward : d[n] = x[2n+1] - floor((x[2n] + x[2n+2]) / 2);  s[n] = x[2n] + floor((d[n-1] + d[n] + 2) / 4)
//   inverse : x[2n] = s[n] - floor((d[n-1] + d[n] + 2) / 4);  x[2n+1] = d[n] + floor((x[2n] + x[2n+2]) / 2)
// with x[N] = x[N-2], d[-1] = d[0] (P:755-762 in the DESIGN.md A12/A14 reading); rows then columns forward
// (P:812), columns then rows inverse. A CTA transforms one tile with its halo staged in shared memory; integer
// arithmetic makes the result independent of the tiling. Arithmetic shifts are floors (toward -inf).
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
};

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

    // stage A: input tile with halo (mirrored at the borders)
    for (int i = tid; i < IR * IC; i += DWT_THREADS) {
        const int ly = i / IC, lx = i % IC;
        const int y = mirror_idx(2 * ty0 - 2 + ly, p.ch), x = mirror_idx(2 * tx0 - 2 + lx, p.cw);
        int v;
        if (FIRST) v = (int)p.img_in[(size_t)n * p.image_stride + ((size_t)y * p.img_w + x) * p.C + c] - 128;
        else v = p.ll_in[(size_t)plane * p.ll_in_plane_stride + (size_t)y * p.cw + x];
        sIn[ly][lx] = (int16_t)v;
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
    // vertical update + stores: LL/HL get s, LH/HH get d
    int16_t *llb = p.ll_band + (size_t)n * p.ll_band_image_stride + (size_t)c * p.ll_band_chan_stride;
    int16_t *pb = p.pub + (size_t)n * p.pub_image_stride + (size_t)c * p.pub_chan_stride + p.level_off;
    const size_t band = (size_t)bw * bh;
    for (int i = tid; i < DWT_TH * 2 * DWT_TW; i += DWT_THREADS) {
        const int r = i / (2 * DWT_TW), q = i % (2 * DWT_TW);  // m = ty0 + r
        const int m = ty0 + r;
        const bool high = q >= DWT_TW;
        const int j = high ? q - DWT_TW : q;
        const int nn = tx0 + j;
        if (m >= bh || nn >= bw) continue;
        const int x2m = high ? (int)sHd[2 * r + 2][j + 1] : (int)sHs[2 * r + 2][j];
        const int dprev = sVd[r][q], dcur = sVd[r + 1][q];
        const int s = x2m + ((dprev + dcur + 2) >> 2);
        const size_t o = (size_t)m * bw + nn;
        if (!high) { llb[o] = (int16_t)s; pb[1 * band + o] = (int16_t)dcur; }       // LL, LH
        else { pb[0 * band + o] = (int16_t)s; pb[2 * band + o] = (int16_t)dcur; }   // HL, HH
    }
}

// ------------------------------------------------------------------------------------------------------------
// inverse level: (LL, HL, LH, HH) of size bh x bw -> plane of size 2bh x 2bw; LAST adds 128, clamps, stores uint8
// ------------------------------------------------------------------------------------------------------------
template <bool LAST>
__global__ void __launch_bounds__(DWT_THREADS) dwt_inv_level_kernel(const __grid_constant__ DwtLevelParams p) {
    constexpr int SR = DWT_TH + 2, SC = DWT_TW + 2;  // subband rows m in [ty0-1, ty0+TH], cols n in [tx0-1, tx0+TW]
    __shared__ int16_t sB[4][SR][SC + 1];            // 0 LL, 1 HL, 2 LH, 3 HH
    __shared__ int16_t sL[2 * DWT_TH + 1][SC + 1];   // after vertical synthesis: low-horizontal half, rows 2ty0 .. 2ty0+2TH
    __shared__ int16_t sH[2 * DWT_TH + 1][SC + 1];   // high-horizontal half
    __shared__ int16_t sE[2 * DWT_TH][DWT_TW + 1];   // even output columns x[2n], n in [tx0, tx0+TW]

    const int plane = blockIdx.z;
    const int n = plane / p.C, c = plane % p.C;
    const int tx0 = blockIdx.x * DWT_TW, ty0 = blockIdx.y * DWT_TH;
    const int bw = p.cw >> 1, bh = p.ch >> 1;
    const int tid = threadIdx.x;
    const int16_t *llb = p.ll_band + (size_t)n * p.ll_band_image_stride + (size_t)c * p.ll_band_chan_stride;
    const int16_t *pb = p.pub + (size_t)n * p.pub_image_stride + (size_t)c * p.pub_chan_stride + p.level_off;
    const size_t band = (size_t)bw * bh;

    for (int i = tid; i < 4 * SR * SC; i += DWT_THREADS) {
        const int b = i / (SR * SC), rem = i % (SR * SC), lr = rem / SC, lc = rem % SC;
        // d[-1] = d[0] (mirror at the low end); beyond the high end values are never used: clamp
        int m = ty0 - 1 + lr, nn = tx0 - 1 + lc;
        m = min(max(m, 0), bh - 1);
        nn = min(max(nn, 0), bw - 1);
        const size_t o = (size_t)m * bw + nn;
        int16_t v;
        if (b == 0) v = llb[o];
        else if (b == 1) v = pb[0 * band + o];
        else if (b == 2) v = pb[1 * band + o];
        else v = pb[2 * band + o];
        sB[b][lr][lc] = v;
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
        const int16_t(*S)[SC + 1] = half ? sH : sL;
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
    // outputs: even and odd columns
    for (int i = tid; i < 2 * DWT_TH * 2 * DWT_TW; i += DWT_THREADS) {
        const int ry = i / (2 * DWT_TW), cx = i % (2 * DWT_TW);
        const int y = 2 * ty0 + ry, x = 2 * tx0 + cx;
        if (y >= p.ch || x >= p.cw) continue;
        const int j = cx >> 1;
        int v;
        if ((cx & 1) == 0) v = sE[ry][j];
        else {
            const int a = sE[ry][j];
            const int e = (tx0 + j + 1 < bw) ? (int)sE[ry][j + 1] : a;
            v = (int)sH[ry][j + 1] + ((a + e) >> 1);
        }
        if (LAST) {
            v = min(max(v + 128, 0), 255);
            p.img_out[(size_t)n * p.image_stride + ((size_t)y * p.img_w + x) * p.C + c] = (uint8_t)v;
        } else {
            p.ll_out_plane[(size_t)plane * p.ll_out_plane_stride + (size_t)y * p.cw + x] = (int16_t)v;
        }
    }
}

}  // namespace feds
