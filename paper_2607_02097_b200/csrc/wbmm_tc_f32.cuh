// Device helpers shared by the fp32 tensor-core kernels (wbmm_tc_f32.cu: forward / dX, wbmm_tc_f32_dt.cu: table
// gradient): exact splitting of fp32 values into bf16 terms, and per-thread window addressing of fp32 frames.
#pragma once

#include "wbmm_tc_dev.cuh"

namespace wbmm {
namespace {

// (a, b) -> the three bf16 pairs (a in the low half): a = a1 + a2 + a3 up to 2^-24 |a|
__device__ __forceinline__ void split3(float a, float b, uint32_t& p0, uint32_t& p1, uint32_t& p2)
{
    __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
    p0 = *reinterpret_cast<uint32_t*>(&h);
    a -= __uint_as_float(p0 << 16);
    b -= __uint_as_float(p0 & 0xffff0000u);
    h = __floats2bfloat162_rn(a, b);
    p1 = *reinterpret_cast<uint32_t*>(&h);
    a -= __uint_as_float(p1 << 16);
    b -= __uint_as_float(p1 & 0xffff0000u);
    h = __floats2bfloat162_rn(a, b);
    p2 = *reinterpret_cast<uint32_t*>(&h);
}

__device__ __forceinline__ void split3_one(float a, uint16_t* s)
{
    uint32_t p0, p1, p2;
    split3(a, 0.f, p0, p1, p2);
    s[0] = (uint16_t)p0;
    s[1] = (uint16_t)p1;
    s[2] = (uint16_t)p2;
}

// Per-thread window addressing for the general form (shift / ragged): byte offsets of the window's rows and
// columns inside the natural-layout frame image, plus validity masks (bit set = inside H x W).  Offsets of
// padding rows / columns are 0 so that every address is legal.
template <int WS>
struct GenAddrF {
    int rowoff[WS], coloff[WS];
    uint32_t rowmask, colmask;
};

template <int WS>
__device__ __forceinline__ void gen_addr_f32(GenAddrF<WS>& a, const Geom& g, int wyl, int wx)
{
    a.rowmask = a.colmask = 0;
#pragma unroll
    for (int r = 0; r < WS; ++r) {
        int h = wyl * WS + r + g.sh;
        if (h >= g.Hp) h -= g.Hp;
        a.rowoff[r] = h < g.H ? h * g.W * 4 : 0;
        a.rowmask |= (h < g.H ? 1u : 0u) << r;
        int v = wx * WS + r + g.sw;
        if (v >= g.Wp) v -= g.Wp;
        a.coloff[r] = v < g.W ? v * 4 : 0;
        a.colmask |= (v < g.W ? 1u : 0u) << r;
    }
}

}  // namespace
}  // namespace wbmm
