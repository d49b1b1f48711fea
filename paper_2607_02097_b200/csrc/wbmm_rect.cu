// WBMM with RECTANGULAR windows w_h x w_w (section 3.1: "window size w_h x w_w", d = w_h * w_w positions,
// table R in R^{C x (2w_h-1)(2w_w-1)}; Eq. 4-5 pad H by w_h and W by w_w; Eq. 6-7:
//     I[i,j] = (dh + w_h - 1)(2w_w - 1) + (dw + w_w - 1),   dh = h_i - h_j, dw = w_i - w_j).
// w_h = 1 (or w_w = 1) is the 1-D case the paper names as an extension.  SURVEY.md 8(f) NEXT-4.
//
// FFMA kernels (fp32 accumulate), any layout / shift / ragged size / dtype: the general statement of the operator.
// The square sizes 7 and 14 have the tensor-core kernels; nothing here is on their path.
//   forward / dX   a block = one channel x G windows: the table row and the windows staged in shared memory as fp32,
//                  a thread per (output position, four windows) walks the w_h x w_w inputs of its windows
//   dT             a block = one channel x a run of window groups: a thread per bin (dr, dc) sums dy[p] * x[p - (dr, dc)]
//                  over the staged windows, one atomicAdd per bin and block at the end
#include "wbmm_common.cuh"

namespace wbmm {

namespace {

constexpr int kThreadsR = 256;

// A depth axis makes the same kernels serve 3-D windows w_d x w_h x w_w on volumes [B][C][D][H][W] / [B][D][H][W][C]
// (reading A23): in-window position p = (pz * w_h + pr) * w_w + pc, table index
// ((dz + w_d - 1)(2w_h - 1) + (dh + w_h - 1))(2w_w - 1) + (dw + w_w - 1).  2-D problems have D = w_d = 1.
struct RectGeom {
    int B, C, H, W, wh, ww, sh, sw, layout;
    int Hp, Wp, nwh, nww, N, tw, nb;
    int D, wd, sd, Dp, nwd, th;
    long long nwin;
};

__device__ __forceinline__ long long rect_offset(const RectGeom& g, int b, int c, int z, int h, int v)
{
    if (g.layout == WBMM_LAYOUT_NCHW) return ((((long long)b * g.C + c) * g.D + z) * g.H + h) * g.W + v;
    return ((((long long)b * g.D + z) * g.H + h) * g.W + v) * g.C + c;
}

// element of the zero-extended, cyclically shifted frame that window `win` holds at in-window position p; -1 = padding
// (VOL = false: the 2-D problems, D = w_d = 1 -- the depth arithmetic compiles away)
template <bool VOL>
__device__ __forceinline__ long long rect_window_elem(const RectGeom& g, long long win, int p, int c)
{
    if constexpr (!VOL) {
        const int wpi = g.nwh * g.nww;
        const int b = (int)(win / wpi), wl = (int)(win - (long long)b * wpi);
        const int wy = wl / g.nww, wx = wl - wy * g.nww;
        int h = wy * g.wh + p / g.ww + g.sh, v = wx * g.ww + p % g.ww + g.sw;
        if (h >= g.Hp) h -= g.Hp;
        if (v >= g.Wp) v -= g.Wp;
        if (h >= g.H || v >= g.W) return -1;
        if (g.layout == WBMM_LAYOUT_NCHW) return (((long long)b * g.C + c) * g.H + h) * g.W + v;
        return (((long long)b * g.H + h) * g.W + v) * g.C + c;
    }
    const int wps = g.nwh * g.nww, wpi = VOL ? g.nwd * wps : wps;
    const int b = (int)(win / wpi), wv = (int)(win - (long long)b * wpi);
    const int wz = VOL ? wv / wps : 0, wl = wv - wz * wps;
    const int wy = wl / g.nww, wx = wl - wy * g.nww;
    const int area = g.wh * g.ww, pz = VOL ? p / area : 0, p2 = p - pz * area;
    int z = VOL ? wz * g.wd + pz + g.sd : 0, h = wy * g.wh + p2 / g.ww + g.sh, v = wx * g.ww + p2 % g.ww + g.sw;
    if (z >= g.Dp) z -= g.Dp;
    if (h >= g.Hp) h -= g.Hp;
    if (v >= g.Wp) v -= g.Wp;
    if (z >= g.D || h >= g.H || v >= g.W) return -1;
    return rect_offset(g, b, c, z, h, v);
}

// HIER (square windows, w even): the hierarchical operator of PAPER.md:216-227 (Eq. 9) / Algorithm 2 in one pass,
//     y_win = (M_g + diag_blocks(M_l) + 2 I) x_win,
// M_l from the second table Tl [C][(w-1)^2] applied inside each of the 2 x 2 sub-windows of side w/2, 2 I = the two identity
// shortcuts.  The FFMA fallback of wbmm_hier_forward for what the tensor-core kernel does not take (fp32, ...).
// MODE 0: the operator from the table.  1 (HIER): see above.  2 (fused, square windows): y = W_c x + ident * x + bias_c --
// wbmm_forward_fused where the pipelined kernel does not apply; `Tl` carries the bias [C] (nullable).  3 (cached-M,
// PAPER.md:208-210): the GIVEN matrices M [C][N][N] in `T` (reverse = apply M_c^T), bias in `Tl` -- wbmm_forward_matrix
// for float32 and for window sizes without a tensor-core kernel.
enum { kModeTable = 0, kModeHier = 1, kModeFused = 2, kModeMatrix = 3 };

template <typename E, int MODE, bool VOL>
__global__ void __launch_bounds__(kThreadsR)
rect_forward_kernel(RectGeom g, const E* __restrict__ x, const E* __restrict__ T, const E* __restrict__ Tl, E* __restrict__ y, int G, int reverse,
                    float ident)
{
    constexpr bool HIER = MODE == kModeHier;
    // G is a multiple of 4; windows are staged position-major, xs[q][G], so that a thread -- one output position of
    // FOUR windows -- reads the four inputs it needs with one 16-byte load (the same address for every thread of its
    // window quad: a broadcast) and one table entry per input position: 2 shared-memory loads per 4 FFMA.
    extern __shared__ __align__(16) float smem[];
    float* xs = smem;                    // [N][G]
    float* Ts = smem + g.N * G;          // [nb]
    const int c = blockIdx.y;
    const long long win0 = (long long)blockIdx.x * G;
    if constexpr (MODE != kModeMatrix) {
        for (int k = threadIdx.x; k < g.nb; k += kThreadsR)
            Ts[k] = to_f32(T[(long long)c * g.nb + (reverse ? g.nb - 1 - k : k)]);
    }
    const int wl = g.wh / 2, twl = 2 * wl - 1, nbl = twl * twl;      // HIER: the local table
    float* Tls = Ts + g.nb;
    if constexpr (HIER) {
        for (int k = threadIdx.x; k < nbl; k += kThreadsR)
            Tls[k] = to_f32(Tl[(long long)c * nbl + (reverse ? nbl - 1 - k : k)]);
    }
    for (int idx = threadIdx.x; idx < G * g.N; idx += kThreadsR) {
        const int gw = idx / g.N, p = idx - gw * g.N;
        float val = 0.f;
        if (win0 + gw < g.nwin) {
            const long long off = rect_window_elem<VOL>(g, win0 + gw, p, c);
            if (off >= 0) val = to_f32(x[off]);
        }
        xs[p * G + gw] = val;
    }
    __syncthreads();
    const int nq = G / 4;
    for (int idx = threadIdx.x; idx < nq * g.N; idx += kThreadsR) {
        const int gq = idx / g.N, p = idx - gq * g.N;
        const int area = g.wh * g.ww, pz = VOL ? p / area : 0, p2 = p - pz * area;
        const int r = p2 / g.ww, cc = p2 - r * g.ww;
        const int wdn = VOL ? g.wd : 1;
        // Eq. 7 with i = p (output), j = q (input): k = ((pz - zq + w_d - 1)(2w_h - 1) + (r - rq + w_h - 1))(2w_w - 1) + (cc - cq + w_w - 1)
        const float* Tr = VOL ? Ts + ((pz + g.wd - 1) * g.th + r + g.wh - 1) * g.tw + cc + g.ww - 1
                              : Ts + (r + g.wh - 1) * g.tw + cc + g.ww - 1;
        const float4* xq = reinterpret_cast<const float4*>(xs) + gq;
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
        const E* Mc = T + (long long)c * g.N * g.N;                 // MODE 3: this channel's matrix
        for (int zq = 0; zq < wdn; ++zq)
        for (int rq = 0; rq < g.wh; ++rq) {
            const float* Trr = Tr - (zq * g.th + rq) * g.tw;
            const float4* xr = xq + (long long)(zq * g.wh + rq) * g.ww * nq;
            for (int cq = 0; cq < g.ww; ++cq) {
                float t;
                if constexpr (MODE == kModeMatrix) {
                    const int q = (zq * g.wh + rq) * g.ww + cq;
                    t = to_f32(reverse ? Mc[(long long)q * g.N + p] : Mc[(long long)p * g.N + q]);
                } else {
                    t = Trr[-cq];
                }
                if constexpr (MODE == kModeFused) {
                    if (zq == pz && rq == r && cq == cc) t += ident;
                }
                if constexpr (HIER) {
                    if (rq / wl == r / wl && cq / wl == cc / wl) t += Tls[(r - rq + wl - 1) * twl + (cc - cq + wl - 1)];
                    if (zq == pz && rq == r && cq == cc) t += 2.f;
                }
                const float4 v = xr[cq * nq];
                a0 = fmaf(t, v.x, a0); a1 = fmaf(t, v.y, a1); a2 = fmaf(t, v.z, a2); a3 = fmaf(t, v.w, a3);
            }
        }
        float bc = 0.f;
        if constexpr (MODE == kModeFused || MODE == kModeMatrix) {
            if (Tl) bc = to_f32(Tl[c]);
        }
        const float acc[4] = {a0 + bc, a1 + bc, a2 + bc, a3 + bc};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const long long win = win0 + gq * 4 + u;
            if (win >= g.nwin) break;
            const long long off = rect_window_elem<VOL>(g, win, p, c);
            if (off >= 0) y[off] = from_f32<E>(acc[u]);          // padding is cropped (Eq. 4-5)
        }
    }
}

template <typename E, bool VOL>
__global__ void __launch_bounds__(kThreadsR)
rect_grad_table_kernel(RectGeom g, const E* __restrict__ x, const E* __restrict__ dy, float* __restrict__ dT, int G, int groups_per_block)
{
    extern __shared__ __align__(16) float smem[];
    float* xs = smem;                    // [N][G]
    float* gs = smem + G * g.N;          // [N][G]
    const int c = blockIdx.y;
    const long long ngroups = (g.nwin + G - 1) / G;
    const long long grp0 = (long long)blockIdx.x * groups_per_block;
    // bins owned by this thread: k = threadIdx.x + i * kThreadsR, at most kMaxOwn of them
    constexpr int kMaxOwn = 16;          // nb <= 4096
    float acc[kMaxOwn];
#pragma unroll
    for (int i = 0; i < kMaxOwn; ++i) acc[i] = 0.f;
    for (long long grp = grp0; grp < grp0 + groups_per_block && grp < ngroups; ++grp) {
        __syncthreads();
        for (int idx = threadIdx.x; idx < G * g.N; idx += kThreadsR) {
            const int gw = idx / g.N, p = idx - gw * g.N;
            float xv = 0.f, gv = 0.f;
            if (grp * G + gw < g.nwin) {
                const long long off = rect_window_elem<VOL>(g, grp * G + gw, p, c);
                if (off >= 0) { xv = to_f32(x[off]); gv = to_f32(dy[off]); }      // dy is zero outside H x W (A11)
            }
            xs[p * G + gw] = xv;          // position-major: four windows per 16-byte load (G is a multiple of 4)
            gs[p * G + gw] = gv;
        }
        __syncthreads();
        const int nq = G / 4;
        const float4* x4 = reinterpret_cast<const float4*>(xs);
        const float4* g4 = reinterpret_cast<const float4*>(gs);
#pragma unroll
        for (int i = 0; i < kMaxOwn; ++i) {
            const int k = threadIdx.x + i * kThreadsR;
            if (k >= g.nb) break;
            // bin k = ((dz + w_d - 1)(2w_h - 1) + (dr + w_h - 1))(2w_w - 1) + (dc + w_w - 1): pairs p = (zp, rp, cp),
            // q = (zp - dz, rp - dr, cp - dc) inside the window
            const int kz = VOL ? k / (g.th * g.tw) : 0, k2 = k - kz * (g.th * g.tw);
            const int dz = VOL ? kz - (g.wd - 1) : 0, dr = k2 / g.tw - (g.wh - 1), dc = k2 % g.tw - (g.ww - 1);
            const int z0 = VOL ? max(0, dz) : 0, z1 = VOL ? min(g.wd, g.wd + dz) : 1;
            const int r0 = max(0, dr), r1 = min(g.wh, g.wh + dr), c0 = max(0, dc), c1 = min(g.ww, g.ww + dc);
            float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
            for (int zp = z0; zp < z1; ++zp)
            for (int rp = r0; rp < r1; ++rp)
                for (int cp = c0; cp < c1; ++cp) {
                    const float4* gp = g4 + ((zp * g.wh + rp) * g.ww + cp) * nq;
                    const float4* xp = x4 + (((zp - dz) * g.wh + rp - dr) * g.ww + cp - dc) * nq;
                    for (int q = 0; q < nq; ++q) {
                        const float4 gv = gp[q], xv = xp[q];
                        a0 = fmaf(gv.x, xv.x, a0); a1 = fmaf(gv.y, xv.y, a1); a2 = fmaf(gv.z, xv.z, a2); a3 = fmaf(gv.w, xv.w, a3);
                    }
                }
            acc[i] += (a0 + a1) + (a2 + a3);
        }
    }
#pragma unroll
    for (int i = 0; i < kMaxOwn; ++i) {
        const int k = threadIdx.x + i * kThreadsR;
        if (k < g.nb) atomicAdd(dT + (long long)c * g.nb + k, acc[i]);
    }
}

// pad_h, pad_w: the padded extents are multiples of these (default: of the window -- Eq. 4-5; the local sub-windows of the
// hierarchical operator live on the extent padded for the GLOBAL window)
RectGeom make_rect(const wbmm_desc_t& d, int ww, int wh = 0, int pad_h = 0, int pad_w = 0)
{
    RectGeom g;
    g.B = d.B; g.C = d.C; g.H = d.H; g.W = d.W; g.wh = wh ? wh : d.w; g.ww = ww;
    g.sh = d.shift_h; g.sw = d.shift_w; g.layout = d.layout;
    if (pad_h == 0) pad_h = g.wh;
    if (pad_w == 0) pad_w = g.ww;
    g.Hp = (d.H + pad_h - 1) / pad_h * pad_h;
    g.Wp = (d.W + pad_w - 1) / pad_w * pad_w;
    g.nwh = g.Hp / g.wh; g.nww = g.Wp / g.ww;
    g.N = g.wh * g.ww;
    g.tw = 2 * g.ww - 1; g.nb = (2 * g.wh - 1) * g.tw;
    g.nwin = (long long)d.B * g.nwh * g.nww;
    g.D = 1; g.wd = 1; g.sd = 0; g.Dp = 1; g.nwd = 1; g.th = 2 * g.wh - 1;
    return g;
}

// 3-D windows w_d x (d.w = w_h) x w_w on volumes of depth D, shift (sd, d.shift_h, d.shift_w)
RectGeom make_win3d(const wbmm_desc_t& d, int D, int wd, int ww, int sd)
{
    RectGeom g = make_rect(d, ww);
    g.D = D; g.wd = wd; g.sd = sd;
    g.Dp = (D + wd - 1) / wd * wd;
    g.nwd = g.Dp / wd;
    g.N = wd * g.wh * g.ww;
    g.nb = (2 * wd - 1) * g.th * g.tw;
    g.nwin = (long long)d.B * g.nwd * g.nwh * g.nww;
    return g;
}

int rect_group(const RectGeom& g, int budget = 2048) { int G = (budget / g.N) & ~3; return G < 4 ? 4 : (G > 32 ? 32 : G); }      // a multiple of 4

template <typename E, int MODE>
cudaError_t rect_forward_t(const RectGeom& g, const E* x, const E* T, const E* Tl, E* y, bool reverse, cudaStream_t s, float ident = 0.f)
{
    const int G = rect_group(g);
    const int nbl = (g.wh - 1) * (g.wh - 1);
    const size_t smem = sizeof(float) * ((size_t)g.nb + (MODE == kModeHier ? nbl : 0) + (size_t)G * g.N);
    auto k = rect_forward_kernel<E, MODE, false>;
    if constexpr (MODE == kModeTable) { if (g.D > 1 || g.wd > 1) k = rect_forward_kernel<E, MODE, true>; }      // volumes: the table operator only
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)((g.nwin + G - 1) / G), (unsigned)g.C);
    k<<<grid, kThreadsR, smem, s>>>(g, x, T, Tl, y, G, reverse ? 1 : 0, ident);
    return cudaGetLastError();
}

template <typename E>
cudaError_t rect_grad_table_t(const RectGeom& g, const E* x, const E* dy, float* dT, cudaStream_t s)
{
    const int G = rect_group(g, g.nb >= kThreadsR ? 2048 : 1024);      // few bins (1-D windows): smaller groups, more blocks
    const size_t smem = sizeof(float) * 2 * (size_t)G * g.N;
    auto k = (g.D > 1 || g.wd > 1) ? rect_grad_table_kernel<E, true> : rect_grad_table_kernel<E, false>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long ngroups = (g.nwin + G - 1) / G;
    long long want = (8ll * 148 + g.C - 1) / g.C;          // about 8 waves of blocks
    if (want < 1) want = 1;
    long long nsplit = ngroups < want ? ngroups : want;
    const int gpb = (int)((ngroups + nsplit - 1) / nsplit);
    nsplit = (ngroups + gpb - 1) / gpb;
    dim3 grid((unsigned)nsplit, (unsigned)g.C);
    k<<<grid, kThreadsR, smem, s>>>(g, x, dy, dT, G, gpb);
    return cudaGetLastError();
}

}  // namespace

// window area and table size the kernels stage in shared memory / registers
bool rect_supported(const wbmm_desc_t& d, int ww)
{
    if (ww < 1 || d.w < 1 || d.w > 1024 || ww > 1024) return false;
    const long long N = (long long)d.w * ww, nb = (2ll * d.w - 1) * (2ll * ww - 1);
    if (N > 1024 || nb > 4096 || d.C > 65535) return false;
    const RectGeom g = make_rect(d, ww);
    return (g.nwin + rect_group(g) - 1) / rect_group(g) <= 0x7fffffffll;
}

cudaError_t rect_forward(const wbmm_desc_t& d, int ww, const void* x, const void* T, void* y, bool reverse, cudaStream_t s, int* launches)
{
    const RectGeom g = make_rect(d, ww);
    if (g.nwin == 0 || g.C == 0) return cudaSuccess;
    *launches += 1;
    switch (d.dtype) {
    case WBMM_DTYPE_F32: return rect_forward_t<float, kModeTable>(g, (const float*)x, (const float*)T, nullptr, (float*)y, reverse, s);
    case WBMM_DTYPE_BF16: return rect_forward_t<__nv_bfloat16, kModeTable>(g, (const __nv_bfloat16*)x, (const __nv_bfloat16*)T, nullptr, (__nv_bfloat16*)y, reverse, s);
    default: return rect_forward_t<__half, kModeTable>(g, (const __half*)x, (const __half*)T, nullptr, (__half*)y, reverse, s);
    }
}

// adds into dT (the caller clears it)
cudaError_t rect_grad_table(const wbmm_desc_t& d, int ww, const void* x, const void* dy, float* dT, cudaStream_t s, int* launches)
{
    const RectGeom g = make_rect(d, ww);
    if (g.nwin == 0 || g.C == 0) return cudaSuccess;
    *launches += 1;
    switch (d.dtype) {
    case WBMM_DTYPE_F32: return rect_grad_table_t<float>(g, (const float*)x, (const float*)dy, dT, s);
    case WBMM_DTYPE_BF16: return rect_grad_table_t<__nv_bfloat16>(g, (const __nv_bfloat16*)x, (const __nv_bfloat16*)dy, dT, s);
    default: return rect_grad_table_t<__half>(g, (const __half*)x, (const __half*)dy, dT, s);
    }
}

// ---- 3-D windows (wbmm_forward_win3d / wbmm_backward_win3d)
bool win3d_supported(const wbmm_desc_t& d, int D, int wd, int ww)
{
    if (D < 1 || wd < 1 || ww < 1 || d.w < 1 || wd > 1024 || d.w > 1024 || ww > 1024) return false;
    const long long N = (long long)wd * d.w * ww, nb = (2ll * wd - 1) * (2ll * d.w - 1) * (2ll * ww - 1);
    if (N > 1024 || nb > 4096 || d.C > 65535) return false;
    if ((long long)d.B * d.C > (1ll << 40) / ((long long)D * d.H * d.W)) return false;
    const RectGeom g = make_win3d(d, D, wd, ww, 0);
    return (g.nwin + rect_group(g) - 1) / rect_group(g) <= 0x7fffffffll;
}

cudaError_t win3d_forward(const wbmm_desc_t& d, int D, int wd, int ww, int sd, const void* x, const void* T, void* y, bool reverse,
                          cudaStream_t s, int* launches)
{
    const RectGeom g = make_win3d(d, D, wd, ww, sd);
    if (g.nwin == 0 || g.C == 0) return cudaSuccess;
    *launches += 1;
    switch (d.dtype) {
    case WBMM_DTYPE_F32: return rect_forward_t<float, kModeTable>(g, (const float*)x, (const float*)T, nullptr, (float*)y, reverse, s);
    case WBMM_DTYPE_BF16: return rect_forward_t<__nv_bfloat16, kModeTable>(g, (const __nv_bfloat16*)x, (const __nv_bfloat16*)T, nullptr, (__nv_bfloat16*)y, reverse, s);
    default: return rect_forward_t<__half, kModeTable>(g, (const __half*)x, (const __half*)T, nullptr, (__half*)y, reverse, s);
    }
}

// adds into dT (the caller clears it)
cudaError_t win3d_grad_table(const wbmm_desc_t& d, int D, int wd, int ww, int sd, const void* x, const void* dy, float* dT,
                             cudaStream_t s, int* launches)
{
    const RectGeom g = make_win3d(d, D, wd, ww, sd);
    if (g.nwin == 0 || g.C == 0) return cudaSuccess;
    *launches += 1;
    switch (d.dtype) {
    case WBMM_DTYPE_F32: return rect_grad_table_t<float>(g, (const float*)x, (const float*)dy, dT, s);
    case WBMM_DTYPE_BF16: return rect_grad_table_t<__nv_bfloat16>(g, (const __nv_bfloat16*)x, (const __nv_bfloat16*)dy, dT, s);
    default: return rect_grad_table_t<__half>(g, (const __half*)x, (const __half*)dy, dT, s);
    }
}

// ---- hierarchical operator, FFMA fallback (wbmm_hier_forward / wbmm_hier_backward on what the tensor-core kernels do not take)
bool hier_simt_supported(const wbmm_desc_t& d)
{
    return d.w >= 2 && d.w % 2 == 0 && rect_supported(d, d.w);
}

cudaError_t hier_simt_forward(const wbmm_desc_t& d, const void* x, const void* Tg, const void* Tl, void* y, bool transpose,
                              cudaStream_t s, int* launches)
{
    const RectGeom g = make_rect(d, d.w);
    if (g.nwin == 0 || g.C == 0) return cudaSuccess;
    *launches += 1;
    switch (d.dtype) {
    case WBMM_DTYPE_F32: return rect_forward_t<float, kModeHier>(g, (const float*)x, (const float*)Tg, (const float*)Tl, (float*)y, transpose, s);
    case WBMM_DTYPE_BF16: return rect_forward_t<__nv_bfloat16, kModeHier>(g, (const __nv_bfloat16*)x, (const __nv_bfloat16*)Tg, (const __nv_bfloat16*)Tl, (__nv_bfloat16*)y, transpose, s);
    default: return rect_forward_t<__half, kModeHier>(g, (const __half*)x, (const __half*)Tg, (const __half*)Tl, (__half*)y, transpose, s);
    }
}

// adds into dTg and dTl (the caller clears them).  dTl: the table gradient of the (w/2 x w/2)-window operator on the extent
// padded for the GLOBAL window, with the same shift -- its windows are exactly the local sub-windows.
cudaError_t hier_simt_grad_tables(const wbmm_desc_t& d, const void* x, const void* dy, float* dTg, float* dTl, cudaStream_t s, int* launches)
{
    cudaError_t e = rect_grad_table(d, d.w, x, dy, dTg, s, launches);
    if (e != cudaSuccess) return e;
    const RectGeom g = make_rect(d, d.w / 2, d.w / 2, d.w, d.w);
    if (g.nwin == 0 || g.C == 0) return cudaSuccess;
    *launches += 1;
    switch (d.dtype) {
    case WBMM_DTYPE_F32: return rect_grad_table_t<float>(g, (const float*)x, (const float*)dy, dTl, s);
    case WBMM_DTYPE_BF16: return rect_grad_table_t<__nv_bfloat16>(g, (const __nv_bfloat16*)x, (const __nv_bfloat16*)dy, dTl, s);
    default: return rect_grad_table_t<__half>(g, (const __half*)x, (const __half*)dy, dTl, s);
    }
}

// ---- wbmm_forward_fused / wbmm_forward_matrix on FFMA kernels (square windows; what the tensor-core kernels do not take)
template <int MODE>
static cudaError_t square_mode_forward(const wbmm_desc_t& d, const void* x, const void* T, const void* bias, void* y, bool transpose,
                                       float ident, cudaStream_t s, int* launches)
{
    const RectGeom g = make_rect(d, d.w);
    if (g.nwin == 0 || g.C == 0) return cudaSuccess;
    *launches += 1;
    switch (d.dtype) {
    case WBMM_DTYPE_F32: return rect_forward_t<float, MODE>(g, (const float*)x, (const float*)T, (const float*)bias, (float*)y, transpose, s, ident);
    case WBMM_DTYPE_BF16: return rect_forward_t<__nv_bfloat16, MODE>(g, (const __nv_bfloat16*)x, (const __nv_bfloat16*)T, (const __nv_bfloat16*)bias, (__nv_bfloat16*)y, transpose, s, ident);
    default: return rect_forward_t<__half, MODE>(g, (const __half*)x, (const __half*)T, (const __half*)bias, (__half*)y, transpose, s, ident);
    }
}

cudaError_t fused_simt_forward(const wbmm_desc_t& d, const void* x, const void* T, const void* bias, float ident, void* y, bool transpose,
                               cudaStream_t s, int* launches)
{
    return square_mode_forward<kModeFused>(d, x, T, bias, y, transpose, ident, s, launches);
}

cudaError_t matrix_simt_forward(const wbmm_desc_t& d, const void* x, const void* M, const void* bias, void* y, bool transpose,
                                cudaStream_t s, int* launches)
{
    return square_mode_forward<kModeMatrix>(d, x, M, bias, y, transpose, 0.f, s, launches);
}

}  // namespace wbmm
