// feds_k_dwt.cu — launchers of the 5/3 level kernels: register-streaming (feds_dwt_fast.cuh) where the level's geometry
// allows, tiled shared-memory (feds_dwt.cuh) otherwise or when the caller asks for them (FEDS_FLAG_DWT_TILED).
#include "feds_dwt.cuh"
#include "feds_dwt_fast.cuh"
#include "feds_host.h"

namespace feds {

namespace {
// Which level kernel: the register-streaming ones need whole per-thread runs and aligned vector accesses; returns the
// pixels per thread (16: planar int16 or gray uint8; 8: interleaved RGB uint8) or 0 = tiled kernel.
int dwt_fast_px(const DwtLevelParams &p, bool u8, int c_img, int n_images) {
    const int px = u8 ? (c_img == 1 ? 16 : c_img == 3 ? 8 : 0) : 16;
    if (px == 0 || p.cw % px != 0 || (p.ch & 1)) return 0;
    const size_t a = (size_t)px / 2;  // subband elements per thread and row: every offset must be a multiple of it
    if (p.level_off % a || (c_img > 1 && (p.pub_chan_stride % a || p.ll_band_chan_stride % a))) return 0;
    if (n_images > 1 && (p.pub_image_stride % a || p.ll_band_image_stride % a || (u8 && (p.image_stride & 15u)))) return 0;
    if ((reinterpret_cast<uintptr_t>(p.ll_band) | reinterpret_cast<uintptr_t>(p.pub)) & 15u) return 0;
    if (u8) { if (p.img_w % (c_img == 1 ? 16 : 8)) return 0; }
    return px;
}
// picks the rows per warp tile (p.rows) so that the launch has at least ~12 warps per SM, and returns the grid
dim3 dwt_fast_grid(DwtLevelParams &p, int px, int planes) {
    const int runs = p.cw / px, bh = p.ch >> 1;
    const unsigned strips = (unsigned)((runs + DWTF_LANES_OUT - 1) / DWTF_LANES_OUT);
    const unsigned long long want = 12ull * (unsigned)sm_count();
    int rows = DWTF_ROWS;
    while (rows > 4 && (unsigned long long)strips * planes * ((bh + rows - 1) / rows) < want) rows /= 2;
    p.rows = rows;
    return dim3(strips, (unsigned)((bh + DWTF_WARPS * rows - 1) / (DWTF_WARPS * rows)), planes);
}
}  // namespace

feds_status launch_dwt_fwd_level(DwtLevelParams &p, bool first, int c, int n_images, bool tiled, cudaStream_t stream) {
    const int bw = p.cw >> 1, bh = p.ch >> 1;
    const int px = tiled ? 0 : dwt_fast_px(p, first, c, n_images);
    const dim3 fgrid = px ? dwt_fast_grid(p, px, first ? n_images : n_images * c) : dim3();   // also sets p.rows
    if (px && first && c == 1) dwt_fwd_fast_kernel<1, 16, true><<<fgrid, DWTF_WARPS * 32, 0, stream>>>(p);
    else if (px && first) dwt_fwd_fast_kernel<3, 8, true><<<fgrid, DWTF_WARPS * 32, 0, stream>>>(p);
    else if (px) dwt_fwd_fast_kernel<1, 16, false><<<fgrid, DWTF_WARPS * 32, 0, stream>>>(p);
    else {
        const dim3 grid((bw + DWT_TW - 1) / DWT_TW, (bh + DWT_TH - 1) / DWT_TH, n_images * c);
        if (first) dwt_fwd_level_kernel<true><<<grid, DWT_THREADS, 0, stream>>>(p);
        else dwt_fwd_level_kernel<false><<<grid, DWT_THREADS, 0, stream>>>(p);
    }
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

feds_status launch_dwt_inv_level(DwtLevelParams &p, bool last, int c, int n_images, bool tiled, cudaStream_t stream) {
    const int bw = p.cw >> 1, bh = p.ch >> 1;
    const int px = tiled ? 0 : dwt_fast_px(p, last, c, n_images);
    const dim3 fgrid = px ? dwt_fast_grid(p, px, last ? n_images : n_images * c) : dim3();
    if (px && last && c == 1) dwt_inv_fast_kernel<1, 16, true><<<fgrid, DWTF_WARPS * 32, 0, stream>>>(p);
    else if (px && last) dwt_inv_fast_kernel<3, 8, true><<<fgrid, DWTF_WARPS * 32, 0, stream>>>(p);
    else if (px) dwt_inv_fast_kernel<1, 16, false><<<fgrid, DWTF_WARPS * 32, 0, stream>>>(p);
    else {
        const dim3 grid((bw + DWT_TW - 1) / DWT_TW, (bh + DWT_TH - 1) / DWT_TH, n_images * c);
        if (last) dwt_inv_level_kernel<true><<<grid, DWT_THREADS, 0, stream>>>(p);
        else dwt_inv_level_kernel<false><<<grid, DWT_THREADS, 0, stream>>>(p);
    }
    FEDS_LAUNCH_CHECK();
    return FEDS_OK;
}

}  // namespace feds
