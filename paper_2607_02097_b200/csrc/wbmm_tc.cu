// WBMM forward / dX on the 5th-generation tensor cores (tcgen05.mma, accumulator in TMEM),
// bf16 / fp16 inputs, fp32 accumulation.
//
// Per channel c the operator is the GEMM  D[m, i] = sum_j X[m, j] * W_c[i, j]  with m = window,
// i = output position, j = input position (Alg. 1 l.15; orientation per DESIGN.md A1).
//   * A = X  comes from TMEM (tcgen05.mma "TS" form): lane m holds window m's N values, two 16-bit
//     values per 32-bit column, in natural row-major in-window order -- no K padding per window row.
//   * B = W_c is built in shared memory from the (2w-1)^2 table (Eq. 6-8) in the
//     K-major no-swizzle core-matrix layout, once per (CTA, channel); it never exists in HBM.
//   * D (128 lanes x N_PAD fp32 columns) is read back with tcgen05.ld, rounded (RNE) and written
//     through a shared-memory frame in image layout, so partition and un-partition (Alg. 1 l.3-4,
//     l.17) are pure address arithmetic.
#include "wbmm_tc.cuh"

#include "wbmm_ptx.cuh"

namespace wbmm {

namespace {

constexpr int kThreadsG = 256;   // generic kernel: 8 warps; warps 0-3 own the 128 TMEM lanes

template <int WS>
struct WinCfg {
    static constexpr int N = WS * WS;                    // positions per window
    static constexpr int K_PAD = (N + 15) / 16 * 16;     // MMA K (16 per instruction)
    static constexpr int N_PAD = (N + 15) / 16 * 16;     // MMA N (multiple of 16 for M = 128)
    static constexpr int KSTEPS = K_PAD / 16;
    static constexpr int NW = (N + 1) / 2;               // 32-bit words per window (A columns used)
    static constexpr int A_COLS = K_PAD / 2;
    static constexpr int TW = 2 * WS - 1;
    static constexpr int NB = TW * TW;
    static constexpr int LBO = N_PAD * 16;               // bytes between K chunks (8 values) of W_c
    static constexpr int WC_BYTES = (K_PAD / 8) * LBO;
    static constexpr int D_COL = (A_COLS + 31) / 32 * 32;
    static constexpr int TMEM_COLS = (D_COL + N_PAD) <= 128 ? 128 : ((D_COL + N_PAD) <= 256 ? 256 : 512);
    static constexpr int TS_BYTES = (NB * 2 + 15) / 16 * 16;
};

// Stage one channel's table row in shared memory (reversed for the transposed operator) and build
// W_c[i][j] = T[c, rel(i,j)] in the K-major core-matrix layout: value (i, j) lives at byte
// (j/8)*LBO + i*16 + (j%8)*2.  Rows i >= N and columns j >= N are zero.
template <int WS>
__device__ __forceinline__ void build_weight(const uint16_t* __restrict__ Tc, bool reverse, uint16_t* Ts,
                                             uint8_t* Wc, int tid, int nthreads)
{
    using Cf = WinCfg<WS>;
    for (int k = tid; k < Cf::NB; k += nthreads) Ts[k] = Tc[reverse ? Cf::NB - 1 - k : k];
    __syncthreads();
    constexpr int NCHUNK = (Cf::K_PAD / 8) * Cf::N_PAD;
    for (int id = tid; id < NCHUNK; id += nthreads) {
        const int kc = id / Cf::N_PAD, i = id % Cf::N_PAD;
        uint32_t pk[4] = {0u, 0u, 0u, 0u};
        if (i < Cf::N) {
            const int ri = i / WS, ci = i % WS;
            int j = kc * 8;
            int rj = j / WS, cj = j % WS;
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                uint32_t v = 0;
                if (j < Cf::N) v = Ts[(ri - rj + WS - 1) * Cf::TW + (ci - cj + WS - 1)];   // Eq. 7
                pk[e >> 1] |= v << ((e & 1) * 16);
                ++j;
                if (++cj == WS) { cj = 0; ++rj; }
            }
        }
        *reinterpret_cast<uint4*>(Wc + kc * Cf::LBO + i * 16) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
    }
}

// Word wi (values 2wi, 2wi+1 in row-major in-window order) of the window whose top-left frame
// element is at `win` (bytes), frame row pitch rowB bytes.
template <int WS>
__device__ __forceinline__ uint32_t load_word(const uint8_t* win, int rowB, int wi)
{
    if constexpr (WS % 2 == 0) {
        const int r = (2 * wi) / WS, cc = (2 * wi) % WS;
        return *reinterpret_cast<const uint32_t*>(win + r * rowB + cc * 2);
    } else {
        const int e0 = 2 * wi, e1 = 2 * wi + 1;
        uint32_t lo = *reinterpret_cast<const uint16_t*>(win + (e0 / WS) * rowB + (e0 % WS) * 2);
        uint32_t hi = 0;
        if (e1 < WS * WS) hi = *reinterpret_cast<const uint16_t*>(win + (e1 / WS) * rowB + (e1 % WS) * 2);
        return lo | (hi << 16);
    }
}

template <int WS>
__device__ __forceinline__ void store_word(uint8_t* win, int rowB, int wi, uint32_t v)
{
    if constexpr (WS % 2 == 0) {
        const int r = (2 * wi) / WS, cc = (2 * wi) % WS;
        *reinterpret_cast<uint32_t*>(win + r * rowB + cc * 2) = v;
    } else {
        const int e0 = 2 * wi, e1 = 2 * wi + 1;
        *reinterpret_cast<uint16_t*>(win + (e0 / WS) * rowB + (e0 % WS) * 2) = (uint16_t)(v & 0xffffu);
        if (e1 < WS * WS) *reinterpret_cast<uint16_t*>(win + (e1 / WS) * rowB + (e1 % WS) * 2) = (uint16_t)(v >> 16);
    }
}

template <bool BF16>
__device__ __forceinline__ uint32_t pack2(uint32_t a, uint32_t b)
{
    const float fa = __uint_as_float(a), fb = __uint_as_float(b);
    if constexpr (BF16) {
        __nv_bfloat162 h = __floats2bfloat162_rn(fa, fb);
        return *reinterpret_cast<uint32_t*>(&h);
    } else {
        __half2 h = __floats2half2_rn(fa, fb);
        return *reinterpret_cast<uint32_t*>(&h);
    }
}

// Window -> TMEM A: all 32 lanes of the warp take part (tcgen05.st is warp-collective); lanes
// without a window write zeros.
template <int WS>
__device__ __forceinline__ void window_to_tmem(const uint8_t* win, bool valid, int rowB, uint32_t taddr)
{
    using Cf = WinCfg<WS>;
#pragma unroll
    for (int ch = 0; ch < Cf::A_COLS / 16; ++ch) {
        uint32_t v[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const int wi = ch * 16 + e;
            v[e] = (wi < Cf::NW && valid) ? load_word<WS>(win, rowB, wi) : 0u;
        }
        ptx::tmem_st16(taddr + ch * 16, v);
    }
    if constexpr (Cf::A_COLS % 16 != 0) {
        static_assert(Cf::A_COLS % 16 == 8, "A columns come in 8s");
        constexpr int ch = Cf::A_COLS / 16;
        uint32_t v[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const int wi = ch * 16 + e;
            v[e] = (wi < Cf::NW && valid) ? load_word<WS>(win, rowB, wi) : 0u;
        }
        ptx::tmem_st8(taddr + ch * 16, v);
    }
    ptx::tmem_wait_st();
}

// TMEM D -> rounded 16-bit values in the window's frame position.
template <int WS, bool BF16>
__device__ __forceinline__ void tmem_to_window(uint8_t* win, bool valid, int rowB, uint32_t taddr)
{
    using Cf = WinCfg<WS>;
#pragma unroll
    for (int ch = 0; ch < Cf::N_PAD / 16; ++ch) {
        if (ch * 8 < Cf::NW) {
            uint32_t v[16];
            ptx::tmem_ld16(taddr + ch * 16, v);
            ptx::tmem_wait_ld();
            if (valid) {
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int wi = ch * 8 + e;
                    if (wi < Cf::NW) store_word<WS>(win, rowB, wi, pack2<BF16>(v[2 * e], v[2 * e + 1]));
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Generic kernel ("tcgen05+gather"): any shift, ragged size, W and layout.  The frame is filled
// and drained by plain predicated loads/stores (index arithmetic does padding, shift and layout),
// one tile at a time, all phases separated by block barriers.
template <int WS, bool BF16>
__global__ void __launch_bounds__(kThreadsG, 1)
tc_generic_kernel(Geom g, TcTiles tl, const uint16_t* __restrict__ x, const uint16_t* __restrict__ T,
                  uint16_t* __restrict__ y, int reverse)
{
    using Cf = WinCfg<WS>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* Wc = smem;
    uint16_t* Ts = reinterpret_cast<uint16_t*>(smem + Cf::WC_BYTES);
    uint8_t* frame = smem + Cf::WC_BYTES + Cf::TS_BYTES;
    __shared__ __align__(8) uint64_t mma_bar;
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t bar = ptx::smem_u32(&mma_bar);
    if (warp == 0) ptx::tmem_alloc(ptx::smem_u32(&tmem_base_s), Cf::TMEM_COLS);
    if (tid == 32) {
        ptx::mbar_init(bar, 1);
        ptx::fence_mbar_init();
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::tc_fence_after_sync();
    const uint32_t tmem = tmem_base_s;
    const uint32_t tmem_a = tmem, tmem_d = tmem + Cf::D_COL;
    constexpr uint32_t idesc = ptx::idesc_f16(BF16 ? 1 : 0, 128, Cf::N_PAD);

    const long long t0 = tl.ntiles * blockIdx.x / gridDim.x, t1 = tl.ntiles * (blockIdx.x + 1) / gridDim.x;
    const int rowB = g.Wp * 2;
    const int frame_elems = tl.frame_rows * g.Wp;
    int cur_c = -1;
    uint32_t phase = 0;

    // this thread's window (warps 0-3 only)
    const int m = tid & 127;
    const int wl = m / tl.NP, pl = m % tl.NP;
    const int wyl = wl / g.nww, wx = wl % g.nww;
    uint8_t* win = frame + pl * tl.S + ((wyl * WS) * g.Wp + wx * WS) * 2;

    for (long long t = t0; t < t1; ++t) {
        const int c = (int)(t / tl.tiles_per_c);
        const int rem = (int)(t % tl.tiles_per_c);
        const int gb = rem / tl.nstrips, strip = rem % tl.nstrips;
        const int b0 = gb * tl.NP, wy0 = strip * tl.NSY;
        const int np_eff = min(tl.NP, g.B - b0);

        if (c != cur_c) {   // (the previous tile's MMAs have completed: every thread waited on mma_bar)
            build_weight<WS>(T + (long long)c * Cf::NB, reverse != 0, Ts, Wc, tid, kThreadsG);
            cur_c = c;
        }
        // frame <- x (padded + shifted coordinates)
        for (int idx = tid; idx < np_eff * frame_elems; idx += kThreadsG) {
            const int p = idx / frame_elems, r2 = idx % frame_elems;
            const int hh = r2 / g.Wp, vv = r2 % g.Wp;
            const int hp = wy0 * WS + hh;
            uint16_t val = 0;
            if (hp < g.Hp) {
                int h = hp + g.sh, v = vv + g.sw;
                if (h >= g.Hp) h -= g.Hp;
                if (v >= g.Wp) v -= g.Wp;
                if (h < g.H && v < g.W) val = x[act_offset(g, b0 + p, c, h, v)];
            }
            *reinterpret_cast<uint16_t*>(frame + p * tl.S + r2 * 2) = val;
        }
        ptx::fence_proxy_async_smem();   // W_c (generic-proxy stores) -> tcgen05.mma operand reads
        __syncthreads();

        const bool valid = wl < tl.NSY * g.nww && pl < np_eff && wy0 + wyl < g.nwh;
        if (warp < 4) {
            window_to_tmem<WS>(win, valid, rowB, tmem_a + ((uint32_t)(warp * 32) << 16));
            ptx::tc_fence_before_sync();
        }
        __syncthreads();
        if (warp == 4 && lane == 0) {
            ptx::tc_fence_after_sync();
            const uint32_t wc_addr = ptx::smem_u32(Wc);
#pragma unroll
            for (int ks = 0; ks < Cf::KSTEPS; ++ks) {
                const uint64_t bdesc = ptx::smem_desc_kmajor_noswz(wc_addr + ks * 2 * Cf::LBO, Cf::LBO, 128);
                ptx::mma_ts(tmem_d, tmem_a + ks * 8, bdesc, idesc, ks > 0 ? 1u : 0u);
            }
            ptx::mma_commit(bar);
        }
        ptx::mbar_wait(bar, phase);
        phase ^= 1;
        ptx::tc_fence_after_sync();
        if (warp < 4) {
            tmem_to_window<WS, BF16>(win, valid, rowB, tmem_d + ((uint32_t)(warp * 32) << 16));
            ptx::tc_fence_before_sync();
        }
        __syncthreads();
        // y <- frame (un-shift, crop)
        for (int idx = tid; idx < np_eff * frame_elems; idx += kThreadsG) {
            const int p = idx / frame_elems, r2 = idx % frame_elems;
            const int hh = r2 / g.Wp, vv = r2 % g.Wp;
            const int hp = wy0 * WS + hh;
            if (hp < g.Hp) {
                int h = hp + g.sh, v = vv + g.sw;
                if (h >= g.Hp) h -= g.Hp;
                if (v >= g.Wp) v -= g.Wp;
                if (h < g.H && v < g.W)
                    y[act_offset(g, b0 + p, c, h, v)] = *reinterpret_cast<const uint16_t*>(frame + p * tl.S + r2 * 2);
            }
        }
        __syncthreads();
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 0) ptx::tmem_dealloc(tmem, Cf::TMEM_COLS);
}

template <int WS>
size_t generic_smem(const TcTiles& tl)
{
    return (size_t)WinCfg<WS>::WC_BYTES + WinCfg<WS>::TS_BYTES + (size_t)tl.NP * tl.S;
}

int num_sms()
{
    static int n = 0;
    if (n == 0) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
        if (n <= 0) n = 148;
    }
    return n;
}

template <int WS, bool BF16>
cudaError_t launch_generic(const Geom& g, const TcTiles& tl, const void* x, const void* T, void* y, bool reverse,
                           cudaStream_t s)
{
    auto k = tc_generic_kernel<WS, BF16>;
    const size_t smem = generic_smem<WS>(tl);
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int grid = (int)(tl.ntiles < num_sms() ? tl.ntiles : num_sms());
    k<<<grid, kThreadsG, smem, s>>>(g, tl, (const uint16_t*)x, (const uint16_t*)T, (uint16_t*)y, reverse ? 1 : 0);
    return cudaGetLastError();
}

}  // namespace

bool tc_tiles(const Geom& g, TcTiles* t)
{
    const int wpp = g.nwh * g.nww;
    if (g.nww > 128) return false;
    if (wpp <= 128) {
        t->NSY = g.nwh;
        t->NP = 128 / wpp;
        if (t->NP > g.B) t->NP = g.B;
    } else {
        t->NP = 1;
        t->NSY = 128 / g.nww;
    }
    t->nstrips = (g.nwh + t->NSY - 1) / t->NSY;
    t->ngb = (g.B + t->NP - 1) / t->NP;
    t->tiles_per_c = t->ngb * t->nstrips;
    t->frame_rows = t->NSY * g.w;
    int s16 = (t->frame_rows * g.Wp * 2 + 15) / 16;
    if (s16 % 2 == 0) ++s16;
    t->S = s16 * 16;
    t->ntiles = (long long)g.C * t->tiles_per_c;
    return true;
}

bool tc_forward_supported(const Geom& g, int dtype, const void*, const void*)
{
    if (dtype != WBMM_DTYPE_BF16 && dtype != WBMM_DTYPE_F16) return false;
    if (g.w != 7 && g.w != 14) return false;
    TcTiles tl;
    if (!tc_tiles(g, &tl)) return false;
    const size_t smem = g.w == 7 ? generic_smem<7>(tl) : generic_smem<14>(tl);
    return smem <= 227 * 1024 - 64;
}

cudaError_t tc_forward(const Geom& g, int dtype, const void* x, const void* T, void* y, bool reverse,
                       cudaStream_t stream, int* launches, int* path)
{
    TcTiles tl;
    if (!tc_tiles(g, &tl)) return cudaErrorNotSupported;
    if (tl.ntiles == 0) return cudaSuccess;
    *launches += 1;
    *path = WBMM_PATH_TC_GATHER;
    const bool bf = dtype == WBMM_DTYPE_BF16;
    if (g.w == 7)
        return bf ? launch_generic<7, true>(g, tl, x, T, y, reverse, stream)
                  : launch_generic<7, false>(g, tl, x, T, y, reverse, stream);
    return bf ? launch_generic<14, true>(g, tl, x, T, y, reverse, stream)
              : launch_generic<14, false>(g, tl, x, T, y, reverse, stream);
}

bool tc_grad_table_supported(const Geom&, int, const void*, const void*) { return false; }
cudaError_t tc_grad_table(const Geom&, int, const void*, const void*, float*, cudaStream_t, int*, int*)
{
    return cudaErrorNotSupported;
}
void tc_release() {}

}  // namespace wbmm
