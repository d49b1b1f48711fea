// WBMM forward / dX for NHWC activations on the tensor cores WITHOUT scratch ("tcgen05+gather" path).
// The default NHWC route is two transposition passes around the NCHW kernels (wbmm_api.cu,
// wbmm_transpose.cu: 2.5x faster forward, 20x faster dT); these kernels serve WBMM_FLAG_NO_SCRATCH, shapes
// whose C or H*W is not a multiple of 8 where they still apply, and allocation failures.
//
// In NHWC the channel -- the BATCH index of the per-channel GEMM (Alg. 1 l.15) -- is
// the contiguous axis, so no tcgen05 operand layout can read a window of one channel from global
// memory.  This kernel works on a group of 8 channels (one 16-byte vector per pixel) at a time:
//
//   1. gather   every pixel of the tile's frame (padded + shifted coordinates, as in the generic
//               kernel) with ONE 16-byte load: 8 channels of a pixel (padding pixels read as zero), and
//               transpose on the fly into 8 channel-planar frames in shared memory (8 conflict-free
//               2-byte stores per pixel: consecutive lanes hold consecutive pixels)
//   2. for each of the 8 channels: build its weights in shared memory (Eq. 6-8: the 13.5 KB
//               block-Toeplitz library for w = 14, the full W_c for w = 7), copy the channel's windows
//               from its planar frame into TMEM (the same word-wide loaders as the NCHW kernels),
//               KSTEPS tcgen05.mma, and write the rounded results back into the planar frame IN PLACE
//   3. scatter  the frames back to y: 8 two-byte loads per pixel, one 16-byte store, un-shifted and cropped
//
// Global traffic is one 16-byte access per pixel and channel group each way: every byte of x is read
// once and every byte of y written once, in half-sector (16 of 32 bytes) pieces.  A tile holds at most
// 64-128 windows of the 8 channels (the frames are 8 x larger than in NCHW) and the phases are
// separated by block barriers: this is the slow corner of the operator, not a
// pipelined kernel.  Without scratch, dT for NHWC is served by the SIMT kernel.
#include "wbmm_tc.cuh"

#include <cuda.h>

#include <mutex>
#include <type_traits>

#include "wbmm_tc_dev.cuh"

namespace wbmm {

using namespace tcdev;

namespace {

constexpr int kThreadsN = 256;
constexpr int kCG = 8;            // channels per group = one 16-byte vector of 16-bit values

// Unsigned division by a run-time constant without a divide (Granlund-Montgomery, round-up form):
// n / d = (t + ((n - t) >> s1)) >> s2,  t = umulhi(m, n);  valid for all 32-bit n, d >= 1.
struct FastDiv {
    uint32_t m, s1, s2;
};
inline FastDiv make_fastdiv(uint32_t d)
{
    FastDiv f;
    uint32_t l = 0;
    while ((1ull << l) < d) ++l;
    f.m = (uint32_t)(((1ull << 32) * ((1ull << l) - d)) / d + 1);
    f.s1 = l < 1 ? l : 1;
    f.s2 = l < 1 ? 0 : l - 1;
    return f;
}
__device__ __forceinline__ uint32_t fdiv(uint32_t n, const FastDiv& f)
{
    const uint32_t t = __umulhi(f.m, n);
    return (t + ((n - t) >> f.s1)) >> f.s2;
}

// Frames of the NHWC kernel: NP images x NSY window-rows x all nww windows across, pixel = 16 bytes.
struct NhwcTiles {
    int NP, NSY, nstrips, ngb, tiles_per_cg, frame_rows, frame_px;   // frame_px: pixels of one frame image
    long long ntiles;
    FastDiv div_px, div_wp;   // by frame_px and by W'
};

template <int WS>
struct NhwcSmem {
    using Bc = BulkCfg<WS>;
    using Cf = WinCfg<WS>;
    static constexpr int TAB_ONE = ((Cf::NB + 2) * 2 + 15) / 16 * 16;
    static constexpr int TAB_BYTES = 2 * TAB_ONE;
    static constexpr int FIXED = Bc::WC_BYTES + TAB_BYTES;
    static constexpr long long ROOM = 227ll * 1024 - 1024 - FIXED;
};

template <int WS>
bool nhwc_tiles(const Geom& g, NhwcTiles* t)
{
    const long long max_px = NhwcSmem<WS>::ROOM / 16;
    const int wpp = g.nwh * g.nww;
    const long long img_px = (long long)g.Hp * g.Wp;
    if (g.nww > 128) return false;
    if (wpp <= 128 && img_px <= max_px) {
        t->NSY = g.nwh;
        long long np = 128 / wpp;
        if (np > max_px / img_px) np = max_px / img_px;
        if (np > g.B) np = g.B;
        t->NP = (int)np;
    } else {
        t->NP = 1;
        long long nsy = 128 / g.nww;
        const long long fit = max_px / ((long long)WS * g.Wp);
        if (nsy > fit) nsy = fit;
        if (nsy > g.nwh) nsy = g.nwh;
        if (nsy < 1) return false;
        t->NSY = (int)nsy;
    }
    t->nstrips = (g.nwh + t->NSY - 1) / t->NSY;
    t->ngb = (g.B + t->NP - 1) / t->NP;
    t->tiles_per_cg = t->ngb * t->nstrips;
    t->frame_rows = t->NSY * g.w;
    t->frame_px = t->frame_rows * g.Wp;
    t->ntiles = (long long)(g.C / kCG) * t->tiles_per_cg;
    t->div_px = make_fastdiv((uint32_t)t->frame_px);
    t->div_wp = make_fastdiv((uint32_t)g.Wp);
    return t->ntiles <= 0x3fffffffll;
}

template <int WS, bool BF16>
__global__ void __launch_bounds__(kThreadsN, 1)
tc_nhwc_kernel(Geom g, NhwcTiles nt, const uint16_t* __restrict__ x, const uint16_t* __restrict__ T,
               uint16_t* __restrict__ y, int reverse)
{
    using Cf = WinCfg<WS>;
    using Bc = BulkCfg<WS>;
    using Sm = NhwcSmem<WS>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* Wc = smem;
    uint16_t* tab = reinterpret_cast<uint16_t*>(smem + Bc::WC_BYTES);
    uint8_t* frame = smem + Sm::FIXED;
    __shared__ __align__(8) uint64_t mma_bar;
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t bar = ptx::smem_u32(&mma_bar);
    if (warp == 0) ptx::tmem_alloc(ptx::smem_u32(&tmem_base_s), 512);
    if (tid == 32) {
        ptx::mbar_init(bar, 1);
        ptx::fence_mbar_init();
    }
    if constexpr (Bc::TOEP) {   // build_lib14 never writes the padding rows of the blocks
        for (int i = tid; i < Bc::WC_BYTES / 16; i += kThreadsN) reinterpret_cast<uint4*>(Wc)[i] = make_uint4(0, 0, 0, 0);
    }
    for (int i = tid; i < Sm::TAB_BYTES / 4; i += kThreadsN) reinterpret_cast<uint32_t*>(tab)[i] = 0u;
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::tc_fence_after_sync();
    const uint32_t tmem = tmem_base_s;
    constexpr uint32_t A_STRIDE = (Bc::A_COLS + 31) / 32 * 32;
    const uint32_t tmem_a = tmem, tmem_d = tmem + A_STRIDE;
    static_assert(((Bc::A_COLS + 31) / 32 * 32) + Bc::D_COLS <= 512, "TMEM budget");

    const long long t0 = nt.ntiles * blockIdx.x / gridDim.x, t1 = nt.ntiles * (blockIdx.x + 1) / gridDim.x;
    const int wpf = nt.NSY * g.nww;                 // windows per frame image
    const long long pix_stride = (long long)g.C;    // elements between pixels in x / y

    // this thread's window (warps 0-3): MMA row m = pl*wpf + wl
    const int m = tid & 127;
    const int pl = m / wpf, wl = m % wpf;
    const int wyl = wl / g.nww, wx = wl % g.nww;
    const int rowB = g.Wp * 2;
    const uint32_t plane_bytes = (uint32_t)nt.NP * nt.frame_px * 2;      // one channel's planar frame
    const uint32_t img_off = (uint32_t)pl * nt.frame_px * 2;
    const uint32_t win_off = img_off + (uint32_t)((wyl * WS) * g.Wp + wx * WS) * 2;
    constexpr bool WG = WS % 2 == 1;                                     // odd w: word-granular window addressing
    GenAddr<WG ? WS : 1> ga;
    if constexpr (WG) gen_addr_init_plain<WS>(ga, g.Wp, wyl, wx);
    uint32_t phase = 0;
    constexpr int PB = 8;                                                // pixels in flight per thread

    auto pixel_src = [&](int idx, int b0, int wy0, long long& off) {
        const int p = (int)fdiv((uint32_t)idx, nt.div_px), r2 = idx - p * nt.frame_px;
        const int hh = (int)fdiv((uint32_t)r2, nt.div_wp), vv = r2 - hh * g.Wp;
        const int hp = wy0 * WS + hh;
        int h = hp + g.sh, v = vv + g.sw;
        if (h >= g.Hp) h -= g.Hp;
        if (v >= g.Wp) v -= g.Wp;
        const bool ok = hp < g.Hp && h < g.H && v < g.W;
        off = ok ? (((long long)(b0 + p) * g.H + h) * g.W + v) * pix_stride : 0;
        return ok;
    };

    for (long long t = t0; t < t1; ++t) {
        const int cg = (int)(t / nt.tiles_per_cg);
        const int rem = (int)(t % nt.tiles_per_cg);
        const int gb = rem / nt.nstrips, strip = rem % nt.nstrips;
        const int b0 = gb * nt.NP, wy0 = strip * nt.NSY;
        const int np_eff = min(nt.NP, g.B - b0);
        const int npx = np_eff * nt.frame_px;
        const uint16_t* xg = x + cg * kCG;
        uint16_t* yg = y + cg * kCG;

        // ---- 1. gather + transpose: planar frame kc, pixel idx <- x[b0+p, h, v, cg*8 + kc]
        for (int i0 = tid; i0 < npx; i0 += kThreadsN * PB) {
            uint4 px[PB];
#pragma unroll
            for (int u = 0; u < PB; ++u) {
                const int idx = i0 + u * kThreadsN;
                px[u] = make_uint4(0, 0, 0, 0);
                if (idx < npx) {
                    long long off;
                    if (pixel_src(idx, b0, wy0, off)) px[u] = __ldg(reinterpret_cast<const uint4*>(xg + off));
                }
            }
#pragma unroll
            for (int u = 0; u < PB; ++u) {
                const int idx = i0 + u * kThreadsN;
                if (idx < npx) {
                    uint8_t* q = frame + (size_t)idx * 2;
                    const uint32_t w4[4] = {px[u].x, px[u].y, px[u].z, px[u].w};
#pragma unroll
                    for (int kc = 0; kc < kCG; ++kc)
                        *reinterpret_cast<uint16_t*>(q + (size_t)kc * plane_bytes) = (uint16_t)(w4[kc >> 1] >> ((kc & 1) * 16));
                }
            }
        }
        __syncthreads();

        const bool valid = pl < np_eff && wy0 + wyl < g.nwh;
        for (int kc = 0; kc < kCG; ++kc) {
            const int c = cg * kCG + kc;
            uint8_t* plane = frame + (size_t)kc * plane_bytes;
            // ---- 2a. weights of channel c (every MMA of the previous channel has completed)
            const uint16_t* Tc = T + (long long)c * Cf::NB;
            if constexpr (Bc::TOEP) {
                if (tid >= 128) {
                    uint16_t tabv[kTabRegs];
                    table_to_regs14(Tc, reverse != 0, tid - 128, tabv);
                    build_lib14(tabv, tab, tab + Sm::TAB_ONE / 2, Wc, tid - 128);
                    ptx::fence_proxy_async_smem();
                }
            } else {
                build_weight<WS>(Tc, reverse != 0, tab, Wc, tid, kThreadsN);
                ptx::fence_proxy_async_smem();
            }
            // ---- 2b. the channel's windows -> TMEM A (w = 14: while warps 4-7 build the library)
            if (warp < 4) {
                const uint32_t taddr = tmem_a + ((uint32_t)(warp * 32) << 16);
                if constexpr (WG) window_to_tmem_gen<WS>(plane + (pl < nt.NP ? img_off : 0u), ga, valid, false, taddr);
                else window_to_tmem_bulk<WS>(plane + (pl < nt.NP ? win_off : 0u), valid, rowB, taddr);
                ptx::tc_fence_before_sync();
            }
            __syncthreads();
            // ---- 2c. contraction
            if (warp == 4 && lane == 0) {
                ptx::tc_fence_after_sync();
                const uint32_t wc_addr = ptx::smem_u32(Wc);
#pragma unroll
                for (int h = 0; h < Bc::NH; ++h) {
                    const uint32_t idesc = ptx::idesc_f16(BF16 ? 1 : 0, 128, Bc::ncols(h));
#pragma unroll
                    for (int ks = 0; ks < Bc::KSTEPS; ++ks) {
                        const uint64_t bdesc = ptx::smem_desc_kmajor_noswz(wc_addr + Bc::b_off(ks, h), Bc::LBO, 128);
                        ptx::mma_ts(tmem_d + Bc::col0(h), tmem_a + ks * 8, bdesc, idesc, ks > 0 ? 1u : 0u);
                    }
                }
                ptx::mma_commit(bar);
            }
            ptx::mbar_wait(bar, phase);
            phase ^= 1;
            ptx::tc_fence_after_sync();
            // ---- 2d. rounded results back into the channel's planar frame, in place
            if (warp < 4) {
                auto drain_half = [&](auto hc) {
                    constexpr int h = decltype(hc)::value;
                    uint32_t pk[Bc::TOEP ? 49 : Bc::ncols(h) / 2];
                    accum_half_to_packed<WS, BF16, h>(tmem_d + Bc::col0(h) + ((uint32_t)(warp * 32) << 16), pk);
                    if (valid) {
                        if constexpr (WG) packed_to_window_gen<WS, Bc::word0(h), Bc::word1(h), false>(plane + img_off, ga, pk);
                        else packed_to_window<WS, Bc::word0(h), Bc::word1(h)>(plane + win_off, rowB, pk);
                    }
                };
                drain_half(std::integral_constant<int, 0>{});
                if constexpr (Bc::NH > 1) drain_half(std::integral_constant<int, 1>{});
                ptx::tc_fence_before_sync();
            }
            __syncthreads();
        }

        // ---- 3. transpose back + scatter: y[b0+p, h, v, cg*8 ..] <- the 8 planar frames (un-shift, crop)
        for (int idx = tid; idx < npx; idx += kThreadsN) {
            long long off;
            if (pixel_src(idx, b0, wy0, off)) {
                const uint8_t* q = frame + (size_t)idx * 2;
                uint32_t w4[4];
#pragma unroll
                for (int kk = 0; kk < 4; ++kk) {
                    const uint32_t lo = *reinterpret_cast<const uint16_t*>(q + (size_t)(2 * kk) * plane_bytes);
                    const uint32_t hi = *reinterpret_cast<const uint16_t*>(q + (size_t)(2 * kk + 1) * plane_bytes);
                    w4[kk] = lo | (hi << 16);
                }
                *reinterpret_cast<uint4*>(yg + off) = make_uint4(w4[0], w4[1], w4[2], w4[3]);
            }
        }
        __syncthreads();
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 0) ptx::tmem_dealloc(tmem, 512);
}

// ------------------------------------------------------------------------------------------------
// Tensor-map variant (no shift): the 8-channel slab of every frame image is ONE 4-D TMA box
// {8 channels, W', rows, 1 image} of a tensor map over x viewed as (C, W, H, B) -- out-of-bounds
// rows / columns (the zero padding of Eq. 4-5) are zero-filled by the copy engine on the way in and
// clipped on the way out.  The frame keeps the memory order [row][col][8 channels]; the channels are
// separated by the repack itself, two at a time: one 32-bit load per pixel gives the values of a
// channel pair, which go to the two A buffers in TMEM; the two channels' results are interleaved
// again in registers and stored 32 bits per pixel.  No LSU gather, no transposition pass.
template <int WS>
struct NhwcTmaSmem {
    using Bc = BulkCfg<WS>;
    static constexpr int FIXED = (NhwcSmem<WS>::FIXED + 127) / 128 * 128;     // the TMA destination is 128-byte aligned
};

template <int WS>
__device__ __forceinline__ void packed_half_to_tmem(const uint32_t* v, int h, uint32_t taddr)
{
    using Bc = BulkCfg<WS>;
    if constexpr (Bc::TOEP) {
        // 7 window rows of 7 words -> 7 padded rows of 8 columns starting at column 56 h
        uint32_t u[56];
#pragma unroll
        for (int r = 0; r < 7; ++r) {
#pragma unroll
            for (int k = 0; k < 8; ++k) u[r * 8 + k] = k < 7 ? v[r * 7 + k] : 0u;
        }
        ptx::tmem_st16(taddr + 56 * h, u);
        ptx::tmem_st16(taddr + 56 * h + 16, u + 16);
        ptx::tmem_st16(taddr + 56 * h + 32, u + 32);
        ptx::tmem_st8(taddr + 56 * h + 48, u + 48);
        ptx::tmem_wait_st();
    } else {
        packed_window_to_tmem<WS>(v, taddr);
    }
}

template <int WS, bool BF16>
__global__ void __launch_bounds__(kThreadsN, 1)
tc_nhwc_tma_kernel(Geom g, NhwcTiles nt, const __grid_constant__ CUtensorMap mx, const __grid_constant__ CUtensorMap my,
                   const uint16_t* __restrict__ T, int reverse)
{
    using Cf = WinCfg<WS>;
    using Bc = BulkCfg<WS>;
    using Sm = NhwcSmem<WS>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* Wc = smem;
    uint16_t* tab = reinterpret_cast<uint16_t*>(smem + Bc::WC_BYTES);
    uint8_t* frame = smem + NhwcTmaSmem<WS>::FIXED;
    __shared__ __align__(8) uint64_t bars[2];
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t mma_bar = ptx::smem_u32(&bars[0]), load_bar = ptx::smem_u32(&bars[1]);
    if (warp == 0) ptx::tmem_alloc(ptx::smem_u32(&tmem_base_s), 512);
    if (tid == 32) {
        ptx::mbar_init(mma_bar, 1);
        ptx::mbar_init(load_bar, 1);
        ptx::fence_mbar_init();
        ptx::tma_prefetch_desc(&mx);
        ptx::tma_prefetch_desc(&my);
    }
    if constexpr (Bc::TOEP) {
        for (int i = tid; i < Bc::WC_BYTES / 16; i += kThreadsN) reinterpret_cast<uint4*>(Wc)[i] = make_uint4(0, 0, 0, 0);
    }
    for (int i = tid; i < Sm::TAB_BYTES / 4; i += kThreadsN) reinterpret_cast<uint32_t*>(tab)[i] = 0u;
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::tc_fence_after_sync();
    const uint32_t tmem = tmem_base_s;
    constexpr uint32_t A_STRIDE = (Bc::A_COLS + 31) / 32 * 32;
    const uint32_t tmem_d = tmem + 2 * A_STRIDE;
    static_assert(2 * ((Bc::A_COLS + 31) / 32 * 32) + Bc::D_COLS <= 512, "TMEM budget");

    const long long t0 = nt.ntiles * blockIdx.x / gridDim.x, t1 = nt.ntiles * (blockIdx.x + 1) / gridDim.x;
    const int wpf = nt.NSY * g.nww;
    const int m = tid & 127;
    const int pl = m / wpf, wl = m % wpf;
    const int wyl = wl / g.nww, wx = wl % g.nww;
    const uint32_t img_bytes = (uint32_t)nt.frame_px * 16;                     // one TMA box
    const uint32_t img_stride = (img_bytes + 127u) & ~127u;                     // boxes land 128-byte aligned
    const uint32_t win_byte = (uint32_t)pl * img_stride + (uint32_t)((wyl * WS) * g.Wp + wx * WS) * 16;
    const uint32_t row_bytes = (uint32_t)g.Wp * 16;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    uint32_t mma_phase = 0, load_phase = 0;
    constexpr int NWH = Bc::TOEP ? 49 : Cf::NW;        // packed words of one half (w = 14) / of the window (w = 7)

    for (long long t = t0; t < t1; ++t) {
        const int cg = (int)(t / nt.tiles_per_cg);
        const int rem = (int)(t % nt.tiles_per_cg);
        const int gb = rem / nt.nstrips, strip = rem % nt.nstrips;
        const int b0 = gb * nt.NP, wy0 = strip * nt.NSY;
        const int np_eff = min(nt.NP, g.B - b0);

        // ---- 1. the frame: one tensor-map box per image
        if (tid == 0) {
            ptx::mbar_arrive_expect_tx(load_bar, (uint32_t)np_eff * img_bytes);
            for (int p = 0; p < np_eff; ++p)
                ptx::tma_load_4d(ptx::smem_u32(frame + (size_t)p * img_stride), &mx, cg * kCG, 0, wy0 * WS, b0 + p, load_bar);
        }
        ptx::mbar_wait(load_bar, load_phase);
        load_phase ^= 1;

        const bool valid = pl < np_eff && pl < nt.NP && wy0 + wyl < g.nwh;
        const uint8_t* wsrc = frame + (valid ? win_byte : 0u);
        for (int kp = 0; kp < kCG / 2; ++kp) {
            // ---- 2a. the windows of channels 2kp, 2kp+1 -> TMEM A0, A1 (one 32-bit load per pixel)
            if (warp < 4) {
#pragma unroll
                for (int h = 0; h < Bc::NH; ++h) {
                    uint32_t vA[NWH], vB[NWH];
#pragma unroll
                    for (int wi = 0; wi < NWH; ++wi) {
                        const int i0 = 2 * (Bc::word0(h) + wi), i1 = i0 + 1;
                        const uint32_t e0 = *reinterpret_cast<const uint32_t*>(wsrc + (i0 / WS) * row_bytes + (i0 % WS) * 16 + 4 * kp);
                        const uint32_t e1 = i1 < Cf::N ? *reinterpret_cast<const uint32_t*>(wsrc + (i1 / WS) * row_bytes + (i1 % WS) * 16 + 4 * kp) : 0u;
                        vA[wi] = __byte_perm(e0, e1, 0x5410);
                        vB[wi] = __byte_perm(e0, e1, 0x7632);
                    }
                    packed_half_to_tmem<WS>(vA, h, tmem + lane_off);
                    packed_half_to_tmem<WS>(vB, h, tmem + A_STRIDE + lane_off);
                }
                ptx::tc_fence_before_sync();
            }
            uint32_t keep[Bc::NH * NWH];                 // channel 2kp's rounded results, until 2kp+1's are there
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const int c = cg * kCG + 2 * kp + q;
                // ---- 2b. weights of channel c
                const uint16_t* Tc = T + (long long)c * Cf::NB;
                if constexpr (Bc::TOEP) {
                    if (tid >= 128) {
                        uint16_t tabv[kTabRegs];
                        table_to_regs14(Tc, reverse != 0, tid - 128, tabv);
                        build_lib14(tabv, tab, tab + Sm::TAB_ONE / 2, Wc, tid - 128);
                        ptx::fence_proxy_async_smem();
                    }
                } else {
                    build_weight<WS>(Tc, reverse != 0, tab, Wc, tid, kThreadsN);
                    ptx::fence_proxy_async_smem();
                }
                __syncthreads();
                // ---- 2c. contraction
                if (warp == 4 && lane == 0) {
                    ptx::tc_fence_after_sync();
                    const uint32_t wc_addr = ptx::smem_u32(Wc);
#pragma unroll
                    for (int h = 0; h < Bc::NH; ++h) {
                        const uint32_t idesc = ptx::idesc_f16(BF16 ? 1 : 0, 128, Bc::ncols(h));
#pragma unroll
                        for (int ks = 0; ks < Bc::KSTEPS; ++ks) {
                            const uint64_t bdesc = ptx::smem_desc_kmajor_noswz(wc_addr + Bc::b_off(ks, h), Bc::LBO, 128);
                            ptx::mma_ts(tmem_d + Bc::col0(h), tmem + q * A_STRIDE + ks * 8, bdesc, idesc, ks > 0 ? 1u : 0u);
                        }
                    }
                    ptx::mma_commit(mma_bar);
                }
                ptx::mbar_wait(mma_bar, mma_phase);
                mma_phase ^= 1;
                ptx::tc_fence_after_sync();
                // ---- 2d. results: keep channel 2kp in registers, interleave with 2kp+1 and store 32 bits per pixel
                if (warp < 4) {
                    auto drain_half = [&](auto hc) {
                        constexpr int h = decltype(hc)::value;
                        uint32_t pk[Bc::TOEP ? 49 : Bc::ncols(h) / 2];
                        accum_half_to_packed<WS, BF16, h>(tmem_d + Bc::col0(h) + lane_off, pk);
                        if (q == 0) {
#pragma unroll
                            for (int wi = 0; wi < NWH; ++wi) keep[h * NWH + wi] = pk[wi];
                        } else if (valid) {
                            uint8_t* wdst = frame + win_byte;
#pragma unroll
                            for (int wi = 0; wi < NWH; ++wi) {
                                const int i0 = 2 * (Bc::word0(h) + wi), i1 = i0 + 1;
                                const uint32_t a = keep[h * NWH + wi], b = pk[wi];
                                *reinterpret_cast<uint32_t*>(wdst + (i0 / WS) * row_bytes + (i0 % WS) * 16 + 4 * kp) = __byte_perm(a, b, 0x5410);
                                if (i1 < Cf::N)
                                    *reinterpret_cast<uint32_t*>(wdst + (i1 / WS) * row_bytes + (i1 % WS) * 16 + 4 * kp) = __byte_perm(a, b, 0x7632);
                            }
                        }
                    };
                    drain_half(std::integral_constant<int, 0>{});
                    if constexpr (Bc::NH > 1) drain_half(std::integral_constant<int, 1>{});
                    ptx::tc_fence_before_sync();
                }
                __syncthreads();
            }
        }

        // ---- 3. the frame back to y: one tensor-map box per image (padding clipped by the copy engine)
        ptx::fence_proxy_async_smem();
        __syncthreads();
        if (tid == 0) {
            for (int p = 0; p < np_eff; ++p)
                ptx::tma_store_4d(&my, cg * kCG, 0, wy0 * WS, b0 + p, ptx::smem_u32(frame + (size_t)p * img_stride));
            ptx::bulk_commit();
            ptx::bulk_wait_read<0>();
        }
        __syncthreads();
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 0) ptx::tmem_dealloc(tmem, 512);
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (libcuda is not linked).
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
        else
            cudaGetLastError();
    });
    return fn;
}

// x or y viewed as (C, W, H, B), box {8, W', frame rows, 1}
bool make_nhwc_map(const Geom& g, const NhwcTiles& nt, int dtype, const void* base, CUtensorMap* map)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)g.C, (cuuint64_t)g.W, (cuuint64_t)g.H, (cuuint64_t)g.B};
    const cuuint64_t strides[3] = {(cuuint64_t)g.C * 2, (cuuint64_t)g.C * 2 * g.W, (cuuint64_t)g.C * 2 * g.W * g.H};
    const cuuint32_t box[4] = {kCG, (cuuint32_t)g.Wp, (cuuint32_t)nt.frame_rows, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUresult r = fn(map, dtype == WBMM_DTYPE_BF16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 4,
                          const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

template <int WS>
bool nhwc_tma_tiles(const Geom& g, NhwcTiles* t)
{
    // same frames as the gather kernel, with the frame start 128-byte aligned
    if (g.sh != 0 || g.sw != 0 || g.Wp > 256) return false;
    if (!nhwc_tiles<WS>(g, t)) return false;
    if (t->frame_rows > 256) return false;
    const long long room = 227ll * 1024 - 1024 - NhwcTmaSmem<WS>::FIXED;
    return (long long)t->NP * (((long long)t->frame_px * 16 + 127) / 128 * 128) <= room;
}

template <int WS, bool BF16>
cudaError_t launch_nhwc_tma(const Geom& g, const NhwcTiles& nt, const CUtensorMap& mx, const CUtensorMap& my, const void* T,
                            bool reverse, cudaStream_t s)
{
    auto k = tc_nhwc_tma_kernel<WS, BF16>;
    const size_t smem = (size_t)NhwcTmaSmem<WS>::FIXED + (size_t)nt.NP * (((size_t)nt.frame_px * 16 + 127) / 128 * 128);
    static SmemOptIn smem_state;
    cudaError_t e = ensure_dynamic_smem(reinterpret_cast<const void*>(k), smem, &smem_state);
    if (e != cudaSuccess) return e;
    const int grid = (int)(nt.ntiles < num_sms() ? nt.ntiles : num_sms());
    k<<<grid, kThreadsN, smem, s>>>(g, nt, mx, my, (const uint16_t*)T, reverse ? 1 : 0);
    return cudaGetLastError();
}

template <int WS, bool BF16>
cudaError_t launch_nhwc(const Geom& g, const NhwcTiles& nt, const void* x, const void* T, void* y, bool reverse,
                        cudaStream_t s)
{
    auto k = tc_nhwc_kernel<WS, BF16>;
    const size_t smem = (size_t)NhwcSmem<WS>::FIXED + (size_t)nt.NP * nt.frame_px * 16;
    static SmemOptIn smem_state;
    cudaError_t e = ensure_dynamic_smem(reinterpret_cast<const void*>(k), smem, &smem_state);
    if (e != cudaSuccess) return e;
    const int grid = (int)(nt.ntiles < num_sms() ? nt.ntiles : num_sms());
    k<<<grid, kThreadsN, smem, s>>>(g, nt, (const uint16_t*)x, (const uint16_t*)T, (uint16_t*)y, reverse ? 1 : 0);
    return cudaGetLastError();
}

}  // namespace


bool tc_nhwc_supported(const Geom& g, int dtype, const void* x, const void* y)
{
    if (g.layout != WBMM_LAYOUT_NHWC) return false;
    if (dtype != WBMM_DTYPE_BF16 && dtype != WBMM_DTYPE_F16) return false;
    if (g.w != 7 && g.w != 14) return false;
    if (g.C % kCG != 0) return false;
    if (g.w % 2 == 1 && g.Wp % 2 == 1) return false;   // odd w: frame rows must be word-aligned
    if (reinterpret_cast<uintptr_t>(x) % 16 != 0 || reinterpret_cast<uintptr_t>(y) % 16 != 0) return false;
    NhwcTiles nt;
    return g.w == 7 ? nhwc_tiles<7>(g, &nt) : nhwc_tiles<14>(g, &nt);
}

cudaError_t tc_nhwc_forward(const Geom& g, int dtype, const void* x, const void* T, void* y, bool reverse,
                            cudaStream_t stream, int* launches)
{
    NhwcTiles nt;
    const bool bf = dtype == WBMM_DTYPE_BF16;
    // tensor-map variant first (no shift, W' and the frame rows within a TMA box)
    if (g.w == 7 ? nhwc_tma_tiles<7>(g, &nt) : nhwc_tma_tiles<14>(g, &nt)) {
        CUtensorMap mx, my;
        if (nt.ntiles == 0) return cudaSuccess;
        if (make_nhwc_map(g, nt, dtype, x, &mx) && make_nhwc_map(g, nt, dtype, y, &my)) {
            *launches += 1;
            if (g.w == 7)
                return bf ? launch_nhwc_tma<7, true>(g, nt, mx, my, T, reverse, stream) : launch_nhwc_tma<7, false>(g, nt, mx, my, T, reverse, stream);
            return bf ? launch_nhwc_tma<14, true>(g, nt, mx, my, T, reverse, stream) : launch_nhwc_tma<14, false>(g, nt, mx, my, T, reverse, stream);
        }
    }
    const bool ok = g.w == 7 ? nhwc_tiles<7>(g, &nt) : nhwc_tiles<14>(g, &nt);
    if (!ok) return cudaErrorNotSupported;
    if (nt.ntiles == 0) return cudaSuccess;
    *launches += 1;
    if (g.w == 7)
        return bf ? launch_nhwc<7, true>(g, nt, x, T, y, reverse, stream) : launch_nhwc<7, false>(g, nt, x, T, y, reverse, stream);
    return bf ? launch_nhwc<14, true>(g, nt, x, T, y, reverse, stream) : launch_nhwc<14, false>(g, nt, x, T, y, reverse, stream);
}

}  // namespace wbmm
