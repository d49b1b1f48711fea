// General WBMM kernels on the fp32 ALUs (FFMA): any window side, dtype, layout, shift and ragged
// size.  They are the fp32 path (BASELINE.json config 1), the route for shapes the tensor-core
// kernels do not cover, and the on-GPU cross-check for them.  Window partition, zero padding,
// cyclic shift and un-partition are index arithmetic in the loads and stores (Alg. 1 l.1-4, l.17;
// PAPER.md:157-173); W_c is never formed: each thread walks the (2w-1)^2 table staged in shared
// memory with the Eq. 7 index.
#include "wbmm_common.cuh"

namespace wbmm {

namespace {

constexpr int kThreads = 256;

// One block works on CB channels x G windows.  Shared memory (floats):
//   Ts[CB][nbp]      table rows (reversed for the transposed operator), nbp = nb rounded up to 4
//   xs[CB][N][G]     input windows, window index fastest (float4 broadcast loads)
//   ys[CB][N][G]     output windows (forward) / dY windows (table gradient)
struct TileIndex {
    int cb, g, q;
};

// Flat staging index -> (cb, g, q).  NCHW: q fastest (runs of w contiguous elements);
// NHWC: cb fastest (contiguous channels).
template <int G>
__device__ __forceinline__ TileIndex decode(const Geom& g, int idx, int CB)
{
    TileIndex t;
    if (g.layout == WBMM_LAYOUT_NCHW) {
        t.q = idx % g.N;
        int r = idx / g.N;
        t.g = r % G;
        t.cb = r / G;
    } else {
        t.cb = idx % CB;
        int r = idx / CB;
        t.q = r % g.N;
        t.g = r / g.N;
    }
    return t;
}

// Source/destination element of window `win`, in-window position q, after zero padding and the
// cyclic shift: returns -1 when the position lies in the padding.
__device__ __forceinline__ long long window_elem(const Geom& g, long long win, int q, int c)
{
    int per_img = g.nwh * g.nww;
    int b = (int)(win / per_img);
    int r = (int)(win % per_img);
    int wy = r / g.nww, wx = r % g.nww;
    int h = wy * g.w + q / g.w + g.sh;
    int v = wx * g.w + q % g.w + g.sw;
    if (h >= g.Hp) h -= g.Hp;
    if (v >= g.Wp) v -= g.Wp;
    if (h >= g.H || v >= g.W) return -1;
    return act_offset(g, b, c, h, v);
}

template <typename E, int G>
__device__ __forceinline__ void stage_windows(const Geom& g, const E* __restrict__ src, float* dst,
                                              long long win0, int c0, int CB)
{
    const int total = CB * G * g.N;
    for (int idx = threadIdx.x; idx < total; idx += kThreads) {
        TileIndex t = decode<G>(g, idx, CB);
        long long win = win0 + t.g;
        int c = c0 + t.cb;
        float val = 0.f;
        if (win < g.nwin && c < g.C) {
            long long off = window_elem(g, win, t.q, c);
            if (off >= 0) val = to_f32(src[off]);
        }
        dst[(t.cb * g.N + t.q) * G + t.g] = val;
    }
}

// Forward / dX staging without per-element 64-bit divisions: the G windows of a block are located once
// (image, first row and column in the padded + shifted frame), an element then costs one division by the window side.
struct WinBase {
    int b, h0, v0;      // b = -1: beyond the last window
};

template <int G>
__device__ __forceinline__ void window_bases(const Geom& g, long long win0, WinBase* wb)
{
    if (threadIdx.x < G) {
        const long long win = win0 + threadIdx.x;
        WinBase r;
        r.b = -1;
        r.h0 = r.v0 = 0;
        if (win < g.nwin) {
            const int per_img = g.nwh * g.nww;
            r.b = (int)(win / per_img);
            const int rr = (int)(win - (long long)r.b * per_img);
            const int wy = rr / g.nww;
            r.h0 = wy * g.w + g.sh;
            r.v0 = (rr - wy * g.nww) * g.w + g.sw;
        }
        wb[threadIdx.x] = r;
    }
}

// The element of window `b`, in-window position q (same result as window_elem).
template <int WS>
__device__ __forceinline__ long long window_elem_at(const Geom& g, const WinBase& b, int q, int c)
{
    const int w = WS ? WS : g.w;
    const int qr = q / w;
    int h = b.h0 + qr, v = b.v0 + (q - qr * w);
    if (h >= g.Hp) h -= g.Hp;
    if (v >= g.Wp) v -= g.Wp;
    if (h >= g.H || v >= g.W) return -1;
    return act_offset(g, b.b, c, h, v);
}

template <int G, int WS>
__device__ __forceinline__ TileIndex decode_ws(const Geom& g, int idx, int CB)
{
    const int N = WS ? WS * WS : g.N;
    TileIndex t;
    if (g.layout == WBMM_LAYOUT_NCHW) {
        const int r = idx / N;
        t.q = idx - r * N;
        t.cb = r / G;
        t.g = r - t.cb * G;
    } else {
        const int r = idx / CB;
        t.cb = idx - r * CB;
        t.g = r / N;
        t.q = r - t.g * N;
    }
    return t;
}

// WS: the window side when it is known at compile time (7, 14: the inner loop over a window row is unrolled, its
// shared-memory loads issued ahead of the FFMAs), 0 = any side (read from g.w).
template <typename E, int G, int WS>
__global__ void __launch_bounds__(kThreads)
simt_forward_kernel(Geom g, const E* __restrict__ x, const E* __restrict__ T, E* __restrict__ y,
                    int CB, int reverse)
{
    extern __shared__ __align__(16) float smem[];
    const int nbp = (g.nb + 3) & ~3;
    float* Ts = smem;
    float* xs = Ts + CB * nbp;
    float* ys = xs + CB * g.N * G;
    const int c0 = blockIdx.y * CB;
    const long long win0 = (long long)blockIdx.x * G;

    for (int idx = threadIdx.x; idx < CB * g.nb; idx += kThreads) {
        int cb = idx / g.nb, k = idx % g.nb;
        int c = c0 + cb;
        int ks = reverse ? g.nb - 1 - k : k;
        Ts[cb * nbp + k] = c < g.C ? to_f32(T[(long long)c * g.nb + ks]) : 0.f;
    }
    __shared__ WinBase wbase[G];
    window_bases<G>(g, win0, wbase);
    __syncthreads();
    const int total = CB * G * g.N;
    for (int idx = threadIdx.x; idx < total; idx += kThreads) {
        const TileIndex t = decode_ws<G, WS>(g, idx, CB);
        const int c = c0 + t.cb;
        float val = 0.f;
        if (wbase[t.g].b >= 0 && c < g.C) {
            const long long off = window_elem_at<WS>(g, wbase[t.g], t.q, c);
            if (off >= 0) val = to_f32(x[off]);
        }
        xs[(t.cb * g.N + t.q) * G + t.g] = val;
    }
    __syncthreads();

    // One unit = (channel of the block, two outputs side by side in a window row: p0 = (rp, cp0), p1 = (rp, cp0 + 1)).
    // The two outputs share every broadcast load of the input windows, and the table entry p1 needs at input column
    // cq is the one p0 used at cq - 1 (Eq. 7 depends on cp - cq only), so a row of the window costs w + 1 table loads
    // for both outputs: (w + 1) + w * G/4 shared-memory loads per 2 * w * G FFMA.  The units of all CB channels are
    // spread over the threads, so that a 7 x 7 window (28 units) does not leave most of the block idle.
    const int w = WS ? WS : g.w, tw = 2 * w - 1;
    const int WH = (w + 1) / 2, NU = w * WH;
    for (int u = threadIdx.x; u < CB * NU; u += kThreads) {
        const int cb = u / NU, pp = u - cb * NU;
        const int rp = pp / WH, cp0 = 2 * (pp - rp * WH);
        const bool has1 = cp0 + 1 < w;                 // odd w: the last unit of a row has one output
        const int p0 = rp * w + cp0;
        const float* xc = xs + cb * g.N * G;
        // Eq. 7 with i = p (output), j = q (input): idx = (rp-rq+w-1)*tw + (cp-cq+w-1)
        const float* Tc0 = Ts + cb * nbp + (rp + w - 1) * tw + cp0 + w - 1;
        float acc0[G], acc1[G];
#pragma unroll
        for (int k = 0; k < G; ++k) acc0[k] = acc1[k] = 0.f;
        for (int rq = 0; rq < w; ++rq) {
            const float* Tr0 = Tc0 - rq * tw;
            const float4* xr = reinterpret_cast<const float4*>(xc + rq * w * G);
            float t1 = has1 ? Tr0[1] : 0.f;            // p1 at cq = 0
#pragma unroll (WS ? WS : 1)
            for (int cq = 0; cq < w; ++cq) {
                const float t0 = Tr0[-cq];
#pragma unroll
                for (int k4 = 0; k4 < G / 4; ++k4) {
                    float4 xv = xr[cq * (G / 4) + k4];
                    acc0[4 * k4 + 0] = fmaf(t0, xv.x, acc0[4 * k4 + 0]);
                    acc0[4 * k4 + 1] = fmaf(t0, xv.y, acc0[4 * k4 + 1]);
                    acc0[4 * k4 + 2] = fmaf(t0, xv.z, acc0[4 * k4 + 2]);
                    acc0[4 * k4 + 3] = fmaf(t0, xv.w, acc0[4 * k4 + 3]);
                    acc1[4 * k4 + 0] = fmaf(t1, xv.x, acc1[4 * k4 + 0]);
                    acc1[4 * k4 + 1] = fmaf(t1, xv.y, acc1[4 * k4 + 1]);
                    acc1[4 * k4 + 2] = fmaf(t1, xv.z, acc1[4 * k4 + 2]);
                    acc1[4 * k4 + 3] = fmaf(t1, xv.w, acc1[4 * k4 + 3]);
                }
                t1 = t0;                               // p1 at cq + 1 reads what p0 read at cq
            }
        }
        float4* yo0 = reinterpret_cast<float4*>(ys + (cb * g.N + p0) * G);
#pragma unroll
        for (int k4 = 0; k4 < G / 4; ++k4)
            yo0[k4] = make_float4(acc0[4 * k4], acc0[4 * k4 + 1], acc0[4 * k4 + 2], acc0[4 * k4 + 3]);
        if (has1) {
            float4* yo1 = yo0 + G / 4;
#pragma unroll
            for (int k4 = 0; k4 < G / 4; ++k4)
                yo1[k4] = make_float4(acc1[4 * k4], acc1[4 * k4 + 1], acc1[4 * k4 + 2], acc1[4 * k4 + 3]);
        }
    }
    __syncthreads();

    // Un-partition: an output of the shifted frame returns to the element its input came from.
    for (int idx = threadIdx.x; idx < total; idx += kThreads) {
        const TileIndex t = decode_ws<G, WS>(g, idx, CB);
        const int c = c0 + t.cb;
        if (wbase[t.g].b >= 0 && c < g.C) {
            const long long off = window_elem_at<WS>(g, wbase[t.g], t.q, c);
            if (off >= 0) y[off] = from_f32<E>(ys[(t.cb * g.N + t.q) * G + t.g]);
        }
    }
}

// dT[c,k] = sum over windows and pairs (p,q) with rel(p,q)=k of dY[p]*X[q].  One thread per bin:
// for bin (dr,dc) the pairs are p=(rp,cp), q=(rp-dr,cp-dc) with both inside the window.
template <typename E, int G>
__global__ void __launch_bounds__(kThreads)
simt_grad_table_kernel(Geom g, const E* __restrict__ x, const E* __restrict__ dy, float* __restrict__ dT,
                       int CB, int groups_per_block)
{
    extern __shared__ __align__(16) float smem[];
    const int nbp = (g.nb + 3) & ~3;
    float* Ds = smem;                    // per-block partial table gradient
    float* xs = Ds + CB * nbp;
    float* gs = xs + CB * g.N * G;
    const int c0 = blockIdx.y * CB;
    const long long ngroups = (g.nwin + G - 1) / G;
    const long long grp0 = (long long)blockIdx.x * groups_per_block;

    for (int idx = threadIdx.x; idx < CB * nbp; idx += kThreads) Ds[idx] = 0.f;

    const int w = g.w, tw = g.tw;
    for (long long grp = grp0; grp < grp0 + groups_per_block && grp < ngroups; ++grp) {
        __syncthreads();
        stage_windows<E, G>(g, x, xs, grp * G, c0, CB);
        stage_windows<E, G>(g, dy, gs, grp * G, c0, CB);
        __syncthreads();
        for (int cb = 0; cb < CB; ++cb) {
            const float* xc = xs + cb * g.N * G;
            const float* gc = gs + cb * g.N * G;
            for (int k = threadIdx.x; k < g.nb; k += kThreads) {
                const int dr = k / tw - (w - 1), dc = k % tw - (w - 1);
                const int r0 = max(0, dr), r1 = min(w, w + dr);
                const int q0 = max(0, dc), q1 = min(w, w + dc);
                float acc = 0.f;
                for (int rp = r0; rp < r1; ++rp)
                    for (int cp = q0; cp < q1; ++cp) {
                        const float4* gv = reinterpret_cast<const float4*>(gc + (rp * w + cp) * G);
                        const float4* xv = reinterpret_cast<const float4*>(xc + ((rp - dr) * w + cp - dc) * G);
#pragma unroll
                        for (int k4 = 0; k4 < G / 4; ++k4) {
                            float4 a = gv[k4], b = xv[k4];
                            acc = fmaf(a.x, b.x, acc);
                            acc = fmaf(a.y, b.y, acc);
                            acc = fmaf(a.z, b.z, acc);
                            acc = fmaf(a.w, b.w, acc);
                        }
                    }
                Ds[cb * nbp + k] += acc;      // each (cb,k) is owned by one thread
            }
        }
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < CB * g.nb; idx += kThreads) {
        int cb = idx / g.nb, k = idx % g.nb;
        if (c0 + cb < g.C) atomicAdd(&dT[(long long)(c0 + cb) * g.nb + k], Ds[cb * nbp + k]);
    }
}

template <typename E>
__global__ void materialize_kernel(int C, int w, const E* __restrict__ T, E* __restrict__ Wout)
{
    const int N = w * w, tw = 2 * w - 1, nb = tw * tw;
    const long long total = (long long)C * N * N;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        int j = (int)(idx % N);
        long long r = idx / N;
        int i = (int)(r % N);
        int c = (int)(r / N);
        int rel = (i / w - j / w + w - 1) * tw + (i % w - j % w + w - 1);   // Eq. 6-7
        Wout[idx] = T[(long long)c * nb + rel];                              // Eq. 8: a copy
    }
}

// Section 3.7: a zero-padded depthwise conv on a one-window map is the operator whose table
// holds the conv kernel around the centre: Tout[c, (w-1-i)(2w-1) + (w-1-j)] = T[...] + scale_c * K[c, i+k, j+k]
// (Eq. 1 read through Eq. 6-7: output p = (h, v) reads input q = (h+i, v+j)).  fp32 arithmetic, one RNE rounding.
template <typename E>
__global__ void fold_dwconv_kernel(int C, int w, int kk, const E* __restrict__ T, const E* __restrict__ K,
                                   const float* __restrict__ scale, E* __restrict__ Tout)
{
    const int tw = 2 * w - 1, nb = tw * tw, k = kk / 2;
    const long long total = (long long)C * nb;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int c = (int)(idx / nb), b = (int)(idx % nb);
        const int i = (w - 1) - b / tw, j = (w - 1) - b % tw;      // the conv tap this bin is
        float v = to_f32(T[idx]);
        if (i >= -k && i <= k && j >= -k && j <= k)
            v = fmaf(scale ? scale[c] : 1.f, to_f32(K[((long long)c * kk + (i + k)) * kk + (j + k)]), v);
        Tout[idx] = from_f32<E>(v);
    }
}

struct TileCfg {
    int CB, G;
    size_t smem_fwd, smem_dt;
};

TileCfg tile_cfg(const Geom& g)
{
    TileCfg t;
    const size_t nbp = (g.nb + 3) & ~3;
    if (g.layout == WBMM_LAYOUT_NCHW) { t.CB = 1; t.G = 8; }
    else { t.CB = 8; t.G = 4; }
    t.smem_fwd = sizeof(float) * t.CB * (nbp + 2ull * g.N * t.G);
    t.smem_dt = t.smem_fwd;
    return t;
}

// Forward / dX: channels per block chosen so that the (channel, output pair) units fill the 256 threads
// (w = 7: 28 units per channel, 9 channels = 252 units), within 48 KB of shared memory so that four or more blocks
// stay resident (w = 14: 98 pairs, 2 channels = 196 units).  The table-gradient kernel keeps tile_cfg.
TileCfg tile_cfg_fwd(const Geom& g)
{
    TileCfg t = tile_cfg(g);
    if (g.layout != WBMM_LAYOUT_NCHW) return t;
    const size_t per_c = t.smem_fwd / t.CB;
    const int NH = g.w * ((g.w + 1) / 2);      // units per channel: pairs of neighbouring outputs, row by row
    int best = 1;
    double best_eff = 0.0;
    for (int cb = 1; cb <= 16 && cb <= g.C; ++cb) {
        if (cb > 1 && cb * per_c > 48 * 1024) break;
        const int units = cb * NH;
        const double eff = (double)units / (double)((units + kThreads - 1) / kThreads * kThreads);
        if (eff > best_eff + 1e-9) { best_eff = eff; best = cb; }
    }
    t.CB = best;
    t.smem_fwd = per_c * best;
    return t;
}

constexpr size_t kMaxSmem = 227 * 1024;

template <typename E>
cudaError_t forward_t(const Geom& g, const E* x, const E* T, E* y, bool reverse, cudaStream_t s)
{
    TileCfg t = tile_cfg_fwd(g);
    dim3 grid((unsigned)((g.nwin + t.G - 1) / t.G), (unsigned)((g.C + t.CB - 1) / t.CB));
    auto launch = [&](auto k) -> cudaError_t {
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t.smem_fwd);
        if (e != cudaSuccess) return e;
        k<<<grid, kThreads, t.smem_fwd, s>>>(g, x, T, y, t.CB, reverse ? 1 : 0);
        return cudaGetLastError();
    };
    if (t.G == 8) {
        if (g.w == 14) return launch(simt_forward_kernel<E, 8, 14>);
        if (g.w == 7) return launch(simt_forward_kernel<E, 8, 7>);
        return launch(simt_forward_kernel<E, 8, 0>);
    }
    if (g.w == 14) return launch(simt_forward_kernel<E, 4, 14>);
    if (g.w == 7) return launch(simt_forward_kernel<E, 4, 7>);
    return launch(simt_forward_kernel<E, 4, 0>);
}

template <typename E>
cudaError_t grad_table_t(const Geom& g, const E* x, const E* dy, float* dT, cudaStream_t s)
{
    TileCfg t = tile_cfg(g);
    const long long ngroups = (g.nwin + t.G - 1) / t.G;
    const int cblocks = (g.C + t.CB - 1) / t.CB;
    // about 8 waves of blocks; each block folds its windows into one set of atomics
    long long want = (8ll * 148 + cblocks - 1) / cblocks;
    if (want < 1) want = 1;
    long long nsplit = ngroups < want ? ngroups : want;
    int gpb = (int)((ngroups + nsplit - 1) / nsplit);
    nsplit = (ngroups + gpb - 1) / gpb;
    dim3 grid((unsigned)nsplit, (unsigned)cblocks);
    cudaError_t e;
    if (t.G == 8) {
        auto k = simt_grad_table_kernel<E, 8>;
        e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t.smem_dt);
        if (e != cudaSuccess) return e;
        k<<<grid, kThreads, t.smem_dt, s>>>(g, x, dy, dT, t.CB, gpb);
    } else {
        auto k = simt_grad_table_kernel<E, 4>;
        e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t.smem_dt);
        if (e != cudaSuccess) return e;
        k<<<grid, kThreads, t.smem_dt, s>>>(g, x, dy, dT, t.CB, gpb);
    }
    return cudaGetLastError();
}

}  // namespace

bool simt_supported(const Geom& g)
{
    TileCfg t = tile_cfg(g);       // tile_cfg_fwd falls back to this size when more channels do not fit
    return t.smem_fwd <= kMaxSmem && g.C <= 65535ll * t.CB && (g.nwin + t.G - 1) / t.G <= 0x7fffffffll;
}

cudaError_t simt_forward(const Geom& g, int dtype, const void* x, const void* T, void* y,
                         bool reverse, cudaStream_t s, int* launches)
{
    if (g.nwin == 0 || g.C == 0) return cudaSuccess;
    *launches += 1;
    switch (dtype) {
    case WBMM_DTYPE_F32: return forward_t<float>(g, (const float*)x, (const float*)T, (float*)y, reverse, s);
    case WBMM_DTYPE_BF16: return forward_t<__nv_bfloat16>(g, (const __nv_bfloat16*)x, (const __nv_bfloat16*)T, (__nv_bfloat16*)y, reverse, s);
    default: return forward_t<__half>(g, (const __half*)x, (const __half*)T, (__half*)y, reverse, s);
    }
}

cudaError_t simt_grad_table(const Geom& g, int dtype, const void* x, const void* dy, float* dT,
                            cudaStream_t s, int* launches)
{
    if (g.nwin == 0 || g.C == 0) return cudaSuccess;
    *launches += 1;
    switch (dtype) {
    case WBMM_DTYPE_F32: return grad_table_t<float>(g, (const float*)x, (const float*)dy, dT, s);
    case WBMM_DTYPE_BF16: return grad_table_t<__nv_bfloat16>(g, (const __nv_bfloat16*)x, (const __nv_bfloat16*)dy, dT, s);
    default: return grad_table_t<__half>(g, (const __half*)x, (const __half*)dy, dT, s);
    }
}

cudaError_t simt_materialize(int C, int w, int dtype, const void* T, void* Wout, cudaStream_t s, int* launches)
{
    const long long total = (long long)C * w * w * w * w;
    if (total == 0) return cudaSuccess;
    int blocks = (int)((total + 255) / 256 < 148 * 16 ? (total + 255) / 256 : 148 * 16);
    *launches += 1;
    if (dtype == WBMM_DTYPE_F32)
        materialize_kernel<uint32_t><<<blocks, 256, 0, s>>>(C, w, (const uint32_t*)T, (uint32_t*)Wout);
    else
        materialize_kernel<uint16_t><<<blocks, 256, 0, s>>>(C, w, (const uint16_t*)T, (uint16_t*)Wout);
    return cudaGetLastError();
}

// dT is accumulated with atomics by several CTAs per channel, so it is zeroed first.  A kernel instead of a memset
// node: with programmatic dependent launch the table-gradient kernel's prologue overlaps it (a memset node in
// front of that kernel measured 3.5 us per call on config 5, this ~1 us).
__global__ void zero_f32_kernel(float* __restrict__ p, long long n)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");              // earlier readers of p have finished
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const long long i4 = (long long)blockIdx.x * blockDim.x + threadIdx.x, stride = (long long)gridDim.x * blockDim.x;
    if ((reinterpret_cast<uintptr_t>(p) & 15) == 0) {
        for (long long i = i4; i < n / 4; i += stride) reinterpret_cast<float4*>(p)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        for (long long i = (n / 4) * 4 + i4; i < n; i += stride) p[i] = 0.f;
    } else {
        for (long long i = i4; i < n; i += stride) p[i] = 0.f;
    }
}

cudaError_t simt_zero_f32(float* p, long long n, cudaStream_t s, int* launches)
{
    if (n <= 0) return cudaSuccess;
    long long blocks = (n / 4 + 255) / 256;
    if (blocks < 1) blocks = 1;
    if (blocks > 148) blocks = 148;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)blocks);
    cfg.blockDim = dim3(256);
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    *launches += 1;
    return cudaLaunchKernelEx(&cfg, zero_f32_kernel, p, n);
}

cudaError_t simt_fold_dwconv(int C, int w, int kk, int dtype, const void* T, const void* K, const float* scale,
                             void* Tout, cudaStream_t s, int* launches)
{
    const long long total = (long long)C * (2 * w - 1) * (2 * w - 1);
    if (total == 0) return cudaSuccess;
    const int blocks = (int)((total + 255) / 256 < 148 * 4 ? (total + 255) / 256 : 148 * 4);
    *launches += 1;
    switch (dtype) {
    case WBMM_DTYPE_F32: fold_dwconv_kernel<float><<<blocks, 256, 0, s>>>(C, w, kk, (const float*)T, (const float*)K, scale, (float*)Tout); break;
    case WBMM_DTYPE_BF16: fold_dwconv_kernel<__nv_bfloat16><<<blocks, 256, 0, s>>>(C, w, kk, (const __nv_bfloat16*)T, (const __nv_bfloat16*)K, scale, (__nv_bfloat16*)Tout); break;
    default: fold_dwconv_kernel<__half><<<blocks, 256, 0, s>>>(C, w, kk, (const __half*)T, (const __half*)K, scale, (__half*)Tout); break;
    }
    return cudaGetLastError();
}

}  // namespace wbmm
