// Shared host/device declarations for the WBMM kernels (not part of the C ABI).
#pragma once

#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "wbmm.h"

namespace wbmm {

// Geometry derived once on the host from wbmm_desc_t (Eq. 4-5: bottom/right zero padding).
struct Geom {
    int B, C, H, W, w;
    int sh, sw;          // cyclic shift (reading A6), 0 = none
    int layout;          // WBMM_LAYOUT_*
    int Hp, Wp;          // padded extents H', W'
    int nwh, nww;        // windows per column / row
    int N;               // positions per window
    int tw, nb;          // table side 2w-1 and bins (2w-1)^2
    long long nwin;      // windows per channel L = B*nwh*nww
};

inline Geom make_geom(const wbmm_desc_t& d)
{
    Geom g;
    g.B = d.B; g.C = d.C; g.H = d.H; g.W = d.W; g.w = d.w;
    g.sh = d.shift_h; g.sw = d.shift_w; g.layout = d.layout;
    g.Hp = (d.H + d.w - 1) / d.w * d.w;
    g.Wp = (d.W + d.w - 1) / d.w * d.w;
    g.nwh = g.Hp / d.w; g.nww = g.Wp / d.w;
    g.N = d.w * d.w;
    g.tw = 2 * d.w - 1; g.nb = g.tw * g.tw;
    g.nwin = (long long)d.B * g.nwh * g.nww;
    return g;
}

__device__ __forceinline__ float to_f32(float v) { return v; }
__device__ __forceinline__ float to_f32(__nv_bfloat16 v) { return __bfloat162float(v); }
__device__ __forceinline__ float to_f32(__half v) { return __half2float(v); }

template <typename E> __device__ __forceinline__ E from_f32(float v);
template <> __device__ __forceinline__ float from_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }
template <> __device__ __forceinline__ __half from_f32<__half>(float v) { return __float2half_rn(v); }

// Element offset of logical (b,c,h,v) in the activation tensor.
__device__ __forceinline__ long long act_offset(const Geom& g, int b, int c, int h, int v)
{
    if (g.layout == WBMM_LAYOUT_NCHW)
        return (((long long)b * g.C + c) * g.H + h) * g.W + v;
    return (((long long)b * g.H + h) * g.W + v) * g.C + c;
}

// Launchers (defined in the .cu files).  All are asynchronous on `stream` and return the
// cudaGetLastError() of their launches.  `reverse` selects the transposed operator W_c^T
// (table index k -> nb-1-k), which is dX.
cudaError_t simt_forward(const Geom& g, int dtype, const void* x, const void* T, void* y,
                         bool reverse, cudaStream_t stream, int* launches);
cudaError_t simt_grad_table(const Geom& g, int dtype, const void* x, const void* dy, float* dT,
                            cudaStream_t stream, int* launches);
cudaError_t simt_materialize(int C, int w, int dtype, const void* T, void* Wout,
                             cudaStream_t stream, int* launches);
// p[0..n) = 0 (stream-ordered; programmatic dependent launch on both sides).
cudaError_t simt_zero_f32(float* p, long long n, cudaStream_t stream, int* launches);
// Tout = T + scale_c * (the table of a zero-padded kk x kk depthwise conv); Tout may be T.
cudaError_t simt_fold_dwconv(int C, int w, int kk, int dtype, const void* T, const void* K, const float* scale,
                             void* Tout, cudaStream_t stream, int* launches);
// Batched transposition of 16-bit elements in[b][R][Cc] -> out[b][Cc][R] (wbmm_transpose.cu).
bool transpose16_supported(long long R, long long Cc, const void* in, const void* out);
cudaError_t transpose16(const void* in, void* out, int batch, int R, int Cc, cudaStream_t stream, int* launches);
// ... and of 32-bit elements (R and Cc multiples of 4).
bool transpose32_supported(long long R, long long Cc, const void* in, const void* out);
cudaError_t transpose32(const void* in, void* out, int batch, int R, int Cc, cudaStream_t stream, int* launches);
// ... and of 8-bit elements (R and Cc multiples of 16).
bool transpose8_supported(long long R, long long Cc, const void* in, const void* out);
cudaError_t transpose8(const void* in, void* out, int batch, int R, int Cc, cudaStream_t stream, int* launches);
// Largest window the SIMT kernels can stage in shared memory for this layout.
bool simt_supported(const Geom& g);
// Rectangular windows w_h x w_w (wbmm_rect.cu): d.w is w_h, `ww` is w_w; shifts in [0, w_h) x [0, w_w).
bool rect_supported(const wbmm_desc_t& d, int ww);
cudaError_t rect_forward(const wbmm_desc_t& d, int ww, const void* x, const void* T, void* y, bool reverse, cudaStream_t stream, int* launches);
cudaError_t rect_grad_table(const wbmm_desc_t& d, int ww, const void* x, const void* dy, float* dT, cudaStream_t stream, int* launches);
// 3-D windows w_d x w_h x w_w on volumes of depth D (wbmm_rect.cu with a depth axis): d.w is w_h, shift (sd, d.shift_h, d.shift_w).
bool win3d_supported(const wbmm_desc_t& d, int D, int wd, int ww);
cudaError_t win3d_forward(const wbmm_desc_t& d, int D, int wd, int ww, int sd, const void* x, const void* T, void* y, bool reverse,
                          cudaStream_t stream, int* launches);
cudaError_t win3d_grad_table(const wbmm_desc_t& d, int D, int wd, int ww, int sd, const void* x, const void* dy, float* dT,
                             cudaStream_t stream, int* launches);
// Hierarchical operator on FFMA kernels (wbmm_rect.cu): any dtype / layout / shift / ragged size, w even.
cudaError_t fused_simt_forward(const wbmm_desc_t& d, const void* x, const void* T, const void* bias, float ident, void* y, bool transpose,
                               cudaStream_t stream, int* launches);
cudaError_t matrix_simt_forward(const wbmm_desc_t& d, const void* x, const void* M, const void* bias, void* y, bool transpose,
                                cudaStream_t stream, int* launches);
bool hier_simt_supported(const wbmm_desc_t& d);
cudaError_t hier_simt_forward(const wbmm_desc_t& d, const void* x, const void* Tg, const void* Tl, void* y, bool transpose,
                              cudaStream_t stream, int* launches);
cudaError_t hier_simt_grad_tables(const wbmm_desc_t& d, const void* x, const void* dy, float* dTg, float* dTl, cudaStream_t stream,
                                  int* launches);

}  // namespace wbmm
