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

#include <cuda.h>

#include <cstring>

#include <cstdlib>
#include <mutex>
#include <type_traits>

#include "wbmm_tc_dev.cuh"

namespace wbmm {

using namespace tcdev;

namespace {

constexpr int kThreadsG = 256;   // generic kernel: 8 warps; warps 0-3 own the 128 TMEM lanes

// ------------------------------------------------------------------------------------------------
// Generic kernel ("tcgen05+gather"): any shift, ragged size, W and layout.  The frame is filled
// and drained by plain predicated loads/stores (index arithmetic does padding, shift and layout),
// one tile at a time, all phases separated by block barriers.
template <int WS, bool BF16>
__global__ void __launch_bounds__(kThreadsG, 1)
tc_generic_kernel(Geom g, TcTiles tl, const uint16_t* __restrict__ x, const uint16_t* __restrict__ T,
                  uint16_t* __restrict__ y, int reverse, const uint16_t* __restrict__ Mfull, const uint16_t* __restrict__ bias)
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

    for (int t = t0; t < t1; ++t) {
        const int c = (int)(t / tl.tiles_per_c);
        const int rem = (int)(t % tl.tiles_per_c);
        const int gb = rem / tl.nstrips, strip = rem % tl.nstrips;
        const int b0 = gb * tl.NP, wy0 = strip * tl.NSY;
        const int np_eff = min(tl.NP, g.B - b0);

        if (c != cur_c) {   // (the previous tile's MMAs have completed: every thread waited on mma_bar)
            // cached-M mode: the channel's matrix is given (reverse = apply its transpose); else Eq. 6-8 from the table
            if (Mfull) load_weight<WS>(Mfull + (long long)c * Cf::N * Cf::N, reverse != 0, Wc, tid, kThreadsG);
            else build_weight<WS>(T + (long long)c * Cf::NB, reverse != 0, Ts, Wc, tid, kThreadsG);
            cur_c = c;
        }
        // frame <- x (padded + shifted coordinates); eight loads in flight per thread
        auto src_offset = [&](int idx) -> long long {
            const int p = idx / frame_elems, r2 = idx - p * frame_elems;
            const int hh = r2 / g.Wp, vv = r2 - hh * g.Wp;
            const int hp = wy0 * WS + hh;
            if (hp >= g.Hp) return -1;
            int h = hp + g.sh, v = vv + g.sw;
            if (h >= g.Hp) h -= g.Hp;
            if (v >= g.Wp) v -= g.Wp;
            return h < g.H && v < g.W ? act_offset(g, b0 + p, c, h, v) : -1;
        };
        auto frame_at = [&](int idx) -> uint16_t* {
            const int p = idx / frame_elems, r2 = idx - p * frame_elems;
            return reinterpret_cast<uint16_t*>(frame + p * tl.S + r2 * 2);
        };
        const int nfe = np_eff * frame_elems;
        for (int base = tid; base < nfe; base += 8 * kThreadsG) {
            uint16_t val[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int idx = base + u * kThreadsG;
                const long long off = idx < nfe ? src_offset(idx) : -1;
                val[u] = off >= 0 ? x[off] : (uint16_t)0;
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int idx = base + u * kThreadsG;
                if (idx < nfe) *frame_at(idx) = val[u];
            }
        }
        ptx::fence_proxy_async_smem();   // W_c (generic-proxy stores) -> tcgen05.mma operand reads
        __syncthreads();

        const bool valid = wl < tl.NSY * g.nww && pl < np_eff && wy0 + wyl < g.nwh;
        if (warp < 4) {
            window_to_tmem<WS>(valid ? win : frame, valid, rowB, tmem_a + ((uint32_t)(warp * 32) << 16));
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
            float bc = 0.f;
            if (bias) bc = BF16 ? __uint_as_float((uint32_t)bias[c] << 16) : __half2float(__ushort_as_half(bias[c]));
            tmem_to_window<WS, BF16>(win, valid, rowB, tmem_d + ((uint32_t)(warp * 32) << 16), bc);
            ptx::tc_fence_before_sync();
        }
        __syncthreads();
        // y <- frame (un-shift, crop)
        for (int idx = tid; idx < nfe; idx += kThreadsG) {
            const long long off = src_offset(idx);
            if (off >= 0) y[off] = *frame_at(idx);
        }
        __syncthreads();
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 0) ptx::tmem_dealloc(tmem, Cf::TMEM_COLS);
}

// ------------------------------------------------------------------------------------------------
// Fast kernel ("tcgen05+tma"): NCHW, no shift, H and W multiples of w.  Every frame image is one
// contiguous run of global memory, so the TMA engine moves it with 1-D bulk copies
// (cp.async.bulk, completion on an mbarrier) and the whole path is a warp-specialised pipeline:
//
//   warp 0      producer   bulk loads  x -> ring of frame-image slots            (full/empty barriers)
//   warp 1      MMA        KSTEPS tcgen05.mma per tile, A from TMEM, B = W_c     (a_full/a_empty, d_full/d_empty)
//   warps 2-5   repack     slot -> registers -> tcgen05.st into A[buf] (2 buffers); build W_c on a channel change
//   warps 6-9   epilogue   tcgen05.ld D -> RNE 16-bit -> back into the window's slot, in place  (out_full)
//   warp 10     store      bulk stores slot -> y, then hands the slot back to the producer      (empty)
//
// Each 32-bit shared-memory access of the repack / epilogue warps is conflict-free for the
// headline geometry: lanes are (4 adjacent windows) x (8 images) and the image stride is 16*odd bytes.

template <int WS>
struct BulkSmem {
    using Cf = WinCfg<WS>;
    static constexpr int TAB_ONE = ((Cf::NB + 2) * 2 + 15) / 16 * 16;
    static constexpr int TAB_BYTES = 2 * TAB_ONE;                              // F0 and F1 (or Ts for the generic builder)
    static constexpr int BAR_BYTES = (2 * kMaxSlots + 8 + 2 * kMaxOutBufs) * 8;
    // layout: barriers | staged table | weights (W_c or the Toeplitz library) | hierarchical libraries | ring ...
    static constexpr int OFF_TAB = (BAR_BYTES + 15) / 16 * 16;
    static constexpr int OFF_WC = (OFF_TAB + TAB_BYTES + 127) / 128 * 128;
    static constexpr int FIXED = (OFF_WC + BulkCfg<WS>::WC_BYTES + BulkCfg<WS>::HIER_BYTES + 127) / 128 * 128;   // tensor-map boxes land 128-byte aligned
    // cached-M mode at w = 14: the 100 KB matrix starts where the library would (which it replaces) and pushes the ring back
    static constexpr int FULL_EXTRA = (OFF_WC + kFullBytes + 1023) / 1024 * 1024 - FIXED;
};

// STRIP (with GEN): general addressing on strips of window rows in rolled row order (maps with more than 128
// windows per image); a template flag so that the whole-image general form pays nothing for it.
// CTAs per SM: two for the aligned w = 7 form (96 registers, 128 TMEM columns, tiles of 12.5 KB: the hand-off
// latencies of one CTA's pipeline are hidden by the other's) and for its strip form (B32 C96 112x112 shift: 40.3 ->
// 34.8 us); one otherwise -- the whole-image general form spills at 80 registers and loses (ragged 60x60: 52 -> 70 us).
template <int WS, bool GEN, bool STRIP = false>
constexpr int bulk_ctas_per_sm() { return (WS == 7 && (!GEN || STRIP)) ? 2 : 1; }
template <int WS>
constexpr int bulk_tmem_cols() { return (2 * ((BulkCfg<WS>::A_COLS + 31) / 32 * 32) + BulkCfg<WS>::D_COLS) <= 128 ? 128 : 512; }

// `np` planes of `chunks` units U each, shared memory (pitch `spitch`) -> global (pitch `dpitch`), by one warp.
template <typename U>
__device__ __forceinline__ void copy_planes_out(const uint8_t* src, uint8_t* dst, int np, int spitch, long long dpitch,
                                                int chunks, int lane)
{
    for (int ch = lane; ch < chunks; ch += 32) {
        const uint8_t* s0 = src + (size_t)ch * sizeof(U);
        uint8_t* d0 = dst + (size_t)ch * sizeof(U);
        int p = 0;
        for (; p + 8 <= np; p += 8) {
            U v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = *reinterpret_cast<const U*>(s0 + (size_t)u * spitch);
#pragma unroll
            for (int u = 0; u < 8; ++u) *reinterpret_cast<U*>(d0 + u * dpitch) = v[u];
            s0 += 8 * (size_t)spitch;
            d0 += 8 * dpitch;
        }
        for (; p < np; ++p) {
            *reinterpret_cast<U*>(d0) = *reinterpret_cast<const U*>(s0);
            s0 += spitch;
            d0 += dpitch;
        }
    }
}

// V: the variant, a template parameter so that the plain table kernel carries none of the other modes' registers and
// branches (as run-time flags they cost the general form 7 % and the aligned w = 7 form 4 %):
//   0  the operator from the table, nothing else
//   1  extras chosen at run time: hierarchical libraries (Tl), identity block, fused bias; w = 7: a given matrix in Tl
//   2  w = 14: cached-M mode (the given matrix Mfull instead of the Toeplitz library); w = 7: the flat form of 7 x 7
//      maps (one window = one plane); bias and, at w = 7, a given matrix in Tl as in 1
template <int WS, bool BF16, bool GEN, bool STRIP, int V>
__global__ void __launch_bounds__(kThreadsB, bulk_ctas_per_sm<WS, GEN, STRIP>())
tc_bulk_kernel(Geom g, TcTiles tl, TilePart part_, int nslot, int nout, const uint16_t* __restrict__ x, const uint16_t* __restrict__ T,
               const uint16_t* __restrict__ Tl, uint16_t* __restrict__ y, int reverse, int box, int sbox,
               const __grid_constant__ CUtensorMap mx, const __grid_constant__ CUtensorMap my,
               const uint16_t* __restrict__ bias, uint32_t ident_bits, const uint16_t* __restrict__ Mfull)
{
    using Cf = WinCfg<WS>;
    using Sm = BulkSmem<WS>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* Wc = smem + Sm::OFF_WC;
    using Bc = BulkCfg<WS>;
    uint8_t* hier = Wc + Bc::WC_BYTES;                      // w = 14: libA | libI | local table (hierarchical operator)
    uint16_t* tab = reinterpret_cast<uint16_t*>(smem + Sm::OFF_TAB);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    const bool is_hier = V == 1 && Bc::TOEP && Tl != nullptr;
    // Epilogue fusions without an epilogue: y = W_c x + ident * x + bias_c.  The identity term is the 16 x 16 block
    // ident * I applied by 14 extra N = 16 MMAs (w = 14; 2 * I for the hierarchical operator); the bias is one more
    // K index: a column of ones in the A operand's padding against a weight row that holds bias_c.
    const bool use_I = V == 1 && Bc::TOEP && (is_hier || ident_bits != 0u);
    const uint16_t* const biasp = V != 0 ? bias : nullptr;
    const uint16_t* const Mw7 = (V != 0 && WS == 7) ? Tl : nullptr;      // w = 7: a given matrix (cached-M mode)
    const uint32_t pad0 = biasp ? (BF16 ? 0x3F80u : 0x3C00u) : 0u;     // 1.0
    // 7 x 7 maps at w = 7: one window = one plane of 49 contiguous elements (plane boxes; see window_to_tmem_flat7)
    constexpr bool flat7 = WS == 7 && !GEN && V == 2;      // (the variant flag of the w = 7 kernel: launched for 7 x 7 maps only)
    // cached-M mode at w = 14: the given matrix of the current channel, 100 KB between the fixed area and the ring
    constexpr bool fullw = WS == 14 && V == 2;      // a template flag: the table kernels pay nothing for this mode
    uint8_t* wfull = Wc;
    uint8_t* ring = smem + Sm::FIXED + (fullw ? Sm::FULL_EXTRA : 0);  // input ring: nslot frame-image slots
    uint8_t* outb = ring + (size_t)nslot * tl.S;            // output ring: nout group buffers of og.images frame images
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t bar0 = ptx::smem_u32(bars);
    auto FULL = [&](int s) { return bar0 + 8u * s; };
    auto EMPTY = [&](int s) { return bar0 + 8u * (kMaxSlots + s); };
    // A_FULL[2] A_EMPTY[2] D_FULL[2] D_EMPTY[2] OUT_FULL[nout] OUT_EMPTY[nout]
    const uint32_t A_FULL = bar0 + 8u * (2 * kMaxSlots), A_EMPTY = A_FULL + 16, D_FULL = A_FULL + 32, D_EMPTY = A_FULL + 48,
                   OUT_FULL = A_FULL + 64, OUT_EMPTY = OUT_FULL + 8 * kMaxOutBufs;
    using Hs = BulkCfg<WS>;
    constexpr bool WG = GEN || (WS % 2 == 1);   // word-granular window addressing (GenAddr)

    const int wpf = tl.NSY * g.nww;   // windows per frame image
    // Output hand-off groups: the smallest runs of whole epilogue warps that cover whole frame images
    // (lanes are image-major), so a group's images can be stored as soon as ITS warps are done.
    const OutGroups og = out_groups(tl, wpf);
    if (warp == 1) ptx::tmem_alloc(ptx::smem_u32(&tmem_base_s), bulk_tmem_cols<WS>());
    if (tid >= 64 && tid < 64 + nslot) {
        ptx::mbar_init(FULL(tid - 64), 1);
        ptx::mbar_init(EMPTY(tid - 64), box ? box * wpf : wpf);   // box mode: one barrier pair per group of `box` images
        ptx::fence_mbar_init();
    }
    if (tid == 0) {
        ptx::mbar_init(A_FULL, 128);
        ptx::mbar_init(A_FULL + 8, 128);
        ptx::mbar_init(A_EMPTY, 1);
        ptx::mbar_init(A_EMPTY + 8, 1);
        for (int h = 0; h < 2; ++h) {
            ptx::mbar_init(D_FULL + 8 * h, 1);
            ptx::mbar_init(D_EMPTY + 8 * h, 128);
        }
        for (int ob = 0; ob < nout; ++ob) {
            ptx::mbar_init(OUT_FULL + 8 * ob, og.lanes);
            ptx::mbar_init(OUT_EMPTY + 8 * ob, 1);
        }
        ptx::fence_mbar_init();
    }
    if constexpr (Bc::TOEP) {
        // build_lib14 never writes the padding rows ci = 14, 15 of the blocks: zero the library once
        for (int i = tid; i < (Bc::WC_BYTES + Bc::HIER_BYTES) / 16; i += kThreadsB) reinterpret_cast<uint4*>(Wc)[i] = make_uint4(0, 0, 0, 0);
    }
    for (int i = tid; i < Sm::TAB_BYTES / 4; i += kThreadsB) reinterpret_cast<uint32_t*>(tab)[i] = 0u;
    ptx::fence_proxy_async_smem();
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::tc_fence_after_sync();
    // Programmatic dependent launch: everything above overlapped the previous kernel's tail; no
    // global memory is touched before this point.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const uint32_t tmem = tmem_base_s;
    constexpr uint32_t A_STRIDE = (Bc::A_COLS + 31) / 32 * 32;
    const uint32_t tmem_d = tmem + 2 * A_STRIDE;
    static_assert(2 * ((Bc::A_COLS + 31) / 32 * 32) + Bc::D_COLS <= 512, "TMEM budget");

    const int t0 = part_.start[blockIdx.x], t1 = part_.start[blockIdx.x + 1];
    const int rowB = g.W * 2;
    const long long plane_elems = (long long)g.H * g.W;
    const bool ragged = g.H != g.Hp || g.W != g.Wp;

    // Every role walks the CTA's tiles in order: (channel, image group, strip) of the current tile, one
    // division at the start and increments afterwards.  tile_decode() returns the current tile and advances.
    int it_c = t0 / tl.tiles_per_c, it_gb, it_strip;
    {
        const int rem = t0 - it_c * tl.tiles_per_c;
        it_gb = rem / tl.nstrips;
        it_strip = rem - it_gb * tl.nstrips;
    }
    auto tile_decode = [&](int, int& c, int& b0, int& wy0, int& np_eff, int& rows_eff) {
        c = it_c;
        b0 = it_gb * tl.NP;
        wy0 = it_strip * tl.NSY;
        np_eff = min(tl.NP, g.B - b0);
        // GEN: whole images (nstrips == 1), or the rolled rows of a strip (gstrip)
        rows_eff = GEN ? (!STRIP ? g.H : min(tl.frame_rows, g.Hp - wy0 * WS)) : min(tl.frame_rows, g.H - wy0 * WS);
        if (++it_strip == tl.nstrips) {
            it_strip = 0;
            if (++it_gb == tl.ngb) {
                it_gb = 0;
                ++it_c;
            }
        }
    };

    if (warp == 0) {
        // ------------------------------------------------------------------ producer
        // lane p issues the copies of frame images p, p+32, ... of every tile
        uint32_t k = 0;
        for (int t = t0; t < t1; ++t) {
            int c, b0, wy0, np_eff, rows_eff;
            tile_decode(t, c, b0, wy0, np_eff, rows_eff);
            // sbox == 2 ("plane boxes"): planes whose byte size is not a multiple of 16 (14 x 14: 392 B) -- the map is over
            // [B][C*H*W], a box is box images x (H*W rounded up to 8) elements from element c*H*W: slot pitch tl.S
            const uint32_t bytes = sbox == 2 ? (uint32_t)tl.S : (uint32_t)rows_eff * rowB;
            if (box) {
                // small images: ONE tensor-map box {a, b, 1 channel, box images} per group instead of `box` copies
                for (int p = lane * box; p < np_eff; p += 32 * box) {
                    const uint32_t kk = k + p;
                    const int slot = kk % nslot;            // first slot of the group (nslot, k, p are multiples of box)
                    ptx::mbar_wait(EMPTY(slot), ((kk / nslot) & 1) ^ 1);
                    ptx::mbar_arrive_expect_tx(FULL(slot), bytes * box);
                    // (the box starts on a 16-byte boundary at or below the plane: the plane sits poff bytes into the slot)
                    const int pe0 = c * (int)plane_elems;
                    ptx::tma_load_4d(ptx::smem_u32(ring + (size_t)slot * tl.S), &mx, sbox == 2 ? (plane_box_2d(plane_elems) ? 0 : pe0 & ~7) : 0,
                                     sbox == 2 && plane_box_2d(plane_elems) ? pe0 >> 3 : 0, sbox == 2 ? 0 : c, b0 + p, FULL(slot));
                }
            } else
            for (int p = lane; p < np_eff; p += 32) {
                const uint32_t kk = k + p;
                const int slot = kk % nslot;
                ptx::mbar_wait(EMPTY(slot), ((kk / nslot) & 1) ^ 1);
                if constexpr (STRIP) {
                    // strip of a shifted / ragged map: the rolled rows are up to two runs of image rows (none at all
                    // when the strip lies in the padding: the barrier then completes on the arrival alone)
                    const StripRuns sr = strip_runs(g, wy0 * WS, rows_eff);
                    const uint16_t* pl0 = x + ((long long)(b0 + p) * g.C + c) * plane_elems;
                    const uint32_t dst0 = ptx::smem_u32(ring + (size_t)slot * tl.S);
                    ptx::mbar_arrive_expect_tx(FULL(slot), (uint32_t)(sr.nA + sr.nB) * rowB);
                    if (sr.nA > 0) ptx::bulk_g2s(dst0, pl0 + (long long)sr.a0 * g.W, (uint32_t)sr.nA * rowB, FULL(slot));
                    if (sr.nB > 0) ptx::bulk_g2s(dst0 + sr.n1 * rowB, pl0, (uint32_t)sr.nB * rowB, FULL(slot));
                    continue;
                }
                ptx::mbar_arrive_expect_tx(FULL(slot), bytes);
                const uint16_t* src = x + ((long long)(b0 + p) * g.C + c) * plane_elems + (long long)wy0 * WS * g.W;
                ptx::bulk_g2s(ptx::smem_u32(ring + (size_t)slot * tl.S), src, bytes, FULL(slot));
            }
            k += np_eff;
            __syncwarp();   // no lane starts the next tile's copies before every copy of this tile is issued (see the repack warps)
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer
        // The whole warp walks the loop and one elected lane issues: the compiler then keeps the operands in uniform
        // registers and emits the tcgen05.mma of a half back to back (issued from inside `if (lane == 0)` every
        // instruction sat in its own elect-and-retry loop behind a rebuilt descriptor, ~75 cycles per issue).  The
        // descriptors differ from a base value by compile-time constants in their 14-bit address field.
        {
            const uint32_t wc_addr = ptx::smem_u32(Wc);
            const uint64_t bd0 = fullw ? ptx::smem_desc_kmajor_noswz(ptx::smem_u32(wfull), kFullLbo, 128)
                                       : ptx::smem_desc_kmajor_noswz(wc_addr, Bc::LBO, 128);
            const uint32_t b_hi = (uint32_t)(bd0 >> 32), b_lo = (uint32_t)bd0;
            uint32_t lt = 0;
            for (int t = t0; t < t1; ++t, ++lt) {
                const uint32_t buf = lt & 1;
                ptx::mbar_wait(A_FULL + 8 * buf, (lt >> 1) & 1);
                const uint32_t tmem_a = tmem + buf * A_STRIDE;
#pragma unroll
                for (int h = 0; h < Hs::NH; ++h) {
                    ptx::mbar_wait(D_EMPTY + 8 * h, (lt & 1) ^ 1);      // the epilogue has drained this half of tile lt-1
                    ptx::tc_fence_after_sync();
                    if (ptx::elect_one()) {
                        const uint32_t idesc = ptx::idesc_f16(BF16 ? 1 : 0, 128, Hs::ncols(h));
#pragma unroll
                        for (int ks = 0; ks < Bc::KSTEPS; ++ks) {
                            const uint32_t boff = (WS == 14 && fullw) ? (uint32_t)((2 * ks * kFullLbo + h * 112 * 16) >> 4)
                                                                      : (uint32_t)(Bc::b_off(ks, h) >> 4);
                            uint64_t bdesc = ((uint64_t)b_hi << 32) | (b_lo + boff);
                            if constexpr (Bc::TOEP) {
                                if (is_hier && ks / 7 == h)     // input and output rows in the same half: global + local blocks
                                    bdesc = ptx::smem_desc_kmajor_noswz(wc_addr + Bc::WC_BYTES + Bc::b_off_a(ks, h), Bc::LBO_A, 128);
                            }
                            ptx::mma_ts(tmem_d + Hs::col0(h), tmem_a + ks * 8, bdesc, idesc, ks > 0 ? 1u : 0u);
                        }
                        if constexpr (Bc::TOEP) {
                            if (use_I) {        // + ident * x: output row ri takes input row ri through the ident*I block
                                const uint32_t idesc_i = ptx::idesc_f16(BF16 ? 1 : 0, 128, 16);
                                const uint64_t idn = ptx::smem_desc_kmajor_noswz(wc_addr + Bc::WC_BYTES + Bc::LIBA_BYTES, Bc::LBO_I, 128);
#pragma unroll
                                for (int ri = 7 * h; ri < 7 * h + 7; ++ri)
                                    ptx::mma_ts(tmem_d + ri * 16, tmem_a + ri * 8, idn, idesc_i, 1u);
                            }
                        }
                        ptx::mma_commit(D_FULL + 8 * h);
                        if (h == Hs::NH - 1) ptx::mma_commit(A_EMPTY + 8 * buf);
                    }
                    __syncwarp();
                }
            }
        }
    } else if (warp < 6) {
        // ------------------------------------------------------------------ repack (+ W_c builder)
        const int q = warp & 3;
        const int m = q * 32 + lane;
        const int rt = (warp - 2) * 32 + lane;   // 0..127 among the repack threads
        const int pl = m / wpf, wl = m % wpf;   // image-major: a warp covers few images, so slots are consumed and released as they land
        const int wyl = wl / g.nww, wx = wl % g.nww;
        const int win_off = wl < wpf ? ((wyl * WS) * g.W + wx * WS) * 2 : 0;   // lanes without a window read a legal address
        GenAddr<WG ? WS : 1> ga;
        if constexpr (STRIP) gen_addr_init_strip<WS>(ga, g, wyl, wx);
        else if constexpr (GEN) gen_addr_init<WS>(ga, g, wyl, wx);
        else if constexpr (WG) gen_addr_init_plain<WS>(ga, g.W, wyl, wx);
        uint32_t k = 0, lt = 0;
        int cur_c = -1;
        uint16_t tabv[kTabRegs];
        bool tabv_ready = false;
        auto rebuild_weight = [&](int c, uint32_t lt) {
            if (c != cur_c) {
                if (lt > 0) ptx::mbar_wait(A_EMPTY + 8 * ((lt - 1) & 1), ((lt - 1) >> 1) & 1);   // MMA(lt-1) done with W_c
                const uint16_t* Tc = T + (long long)c * Cf::NB;
                if (WS == 14 && fullw) {
                    if constexpr (WS == 14)
                        load_weight14_full(Mfull + (long long)c * Cf::N * Cf::N, reverse != 0, wfull, rt, biasp ? (uint32_t)biasp[c] : 0u);
                } else if constexpr (WS == 14) {
                    if (!tabv_ready) table_to_regs14(Tc, reverse != 0, rt, tabv);
                    build_lib14(tabv, tab, tab + Sm::TAB_ONE / 2, Wc, rt, biasp ? (uint32_t)biasp[c] : 0u);
                    tabv_ready = false;
                    // libI = ident * I (hierarchical: the two identity shortcuts, 2.0 = 0x4000 in bf16 and in fp16)
                    if (use_I && rt < 14)
                        *reinterpret_cast<uint16_t*>(hier + Bc::LIBA_BYTES + (rt >> 3) * Bc::LBO_I + rt * 16 + (rt & 7) * 2) =
                            (uint16_t)(is_hier ? 0x4000u : ident_bits);
                    if (is_hier) {
                        uint16_t* FL = reinterpret_cast<uint16_t*>(hier + Bc::LIBA_BYTES + Bc::LIBI_BYTES);
                        const uint16_t* Tlc = Tl + (long long)c * 169;
                        for (int qq = rt; qq < 169; qq += 128) FL[qq] = Tlc[reverse ? qq : 168 - qq];
                        ptx::named_bar_sync(2, 128);          // the global library and FL are complete
                        build_lib14_local<BF16>(Wc, FL, hier, rt);
                    }
                } else if (Mw7) {
                    // cached-M mode (w = 7 only: `Tl` carries the given matrices [C][N][N]) -- the same
                    // operand layout, loaded instead of built; the bias row meets the column of ones at K index N + 1
                    load_weight<WS>(Mw7 + (long long)c * Cf::N * Cf::N, reverse != 0, Wc, rt, 128);
                    if (biasp) {
                        ptx::named_bar_sync(2, 128);
                        for (int i = rt; i < Cf::N; i += 128)
                            *reinterpret_cast<uint16_t*>(Wc + ((Cf::N + 1) / 8) * Cf::LBO + i * 16 + ((Cf::N + 1) % 8) * 2) = biasp[c];
                    }
                } else {
                    static_assert(WS == 14 || Cf::NB <= 2 * 128, "two table entries per repack thread");
                    if (!tabv_ready) table_to_regs7(Tc, reverse != 0, rt, tabv);
#pragma unroll
                    for (int u = 0; u < 2; ++u)
                        if (rt + u * 128 < Cf::NB) tab[rt + u * 128] = tabv[u];
                    tabv_ready = false;
                    ptx::named_bar_sync(2, 128);
                    constexpr int NCHUNK = (Cf::K_PAD / 8) * Cf::N_PAD;
                    for (int id = rt; id < NCHUNK; id += 128) {
                        const int kc = id / Cf::N_PAD, i = id % Cf::N_PAD;
                        uint32_t pk[4] = {0u, 0u, 0u, 0u};
                        if (i < Cf::N) {
                            const int ri = i / WS, ci = i % WS;
                            int j = kc * 8, rj = j / WS, cj = j % WS;
#pragma unroll
                            for (int e = 0; e < 8; ++e) {
                                uint32_t v = 0;
                                if (j < Cf::N) v = tab[(ri - rj + WS - 1) * Cf::TW + (ci - cj + WS - 1)];
                                else if (j == Cf::N + 1 && bias) v = biasp[c];      // K index of the column of ones
                                pk[e >> 1] |= v << ((e & 1) * 16);
                                ++j;
                                if (++cj == WS) { cj = 0; ++rj; }
                            }
                        }
                        *reinterpret_cast<uint4*>(Wc + kc * Cf::LBO + i * 16) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
                    }
                }
                ptx::fence_proxy_async_smem();
                cur_c = c;
            }
        };
        for (int t = t0; t < t1; ++t, ++lt) {
            int c, b0, wy0, np_eff, rows_eff;
            tile_decode(t, c, b0, wy0, np_eff, rows_eff);
            const uint32_t buf = lt & 1;
            // Slot barriers are tested by phase PARITY, and successive fills of one slot are consumed by
            // different threads: a thread may only test fill n once fill n-1 is known to have landed.
            // After this barrier every repack thread has passed its waits of the previous tile, and a
            // slot's previous fill always belongs to an earlier tile (nslot > images per tile).
            // With a ring of at least two tiles the wait below already implies it: MMA(lt-2) committed
            // after every repack thread had finished tile lt-2, and the slot's previous fill is that old.
            if (nslot < 2 * tl.NP) ptx::named_bar_sync(2, 128);
            ptx::mbar_wait(A_EMPTY + 8 * buf, ((lt >> 1) & 1) ^ 1);   // MMA(lt-2) has consumed A[buf]
            const bool part = wl < wpf && pl < np_eff;               // this thread's frame image was loaded
            const bool valid = part && wy0 + wyl < g.nwh;
            if constexpr (STRIP) {
                if (ragged) ga.rowmask = gen_strip_rowmask<WS>(g, wy0 + wyl);
            }
            const uint32_t kk = k + pl;
            const int slot = kk % nslot;
            const int poff = sbox == 2 ? ((c * (int)plane_elems) & 7) * 2 : 0;    // plane boxes: offset of the plane in its slot
            if (lt == 0) rebuild_weight(c, lt);   // first tile: build while its loads are in flight
            const int bslot = box ? slot - slot % box : slot;      // the barrier pair that covers this image
            if (part) ptx::mbar_wait(FULL(bslot), (kk / nslot) & 1);
            if constexpr (flat7) {
                    window_to_tmem_flat7(ring + (size_t)slot * tl.S, poff, valid, tmem + buf * A_STRIDE + ((uint32_t)(q * 32) << 16), pad0);
            } else if constexpr (WG)
            {
                const uint32_t ta = tmem + buf * A_STRIDE + ((uint32_t)(q * 32) << 16);
                if constexpr (GEN && WS % 2 == 0) {      // even w: every window starts on the parity of the column shift
                    if (g.sw & 1) window_to_tmem_gen<WS, 1>(ring + (size_t)slot * tl.S + poff, ga, valid, ragged, ta, pad0);
                    else window_to_tmem_gen<WS, 0>(ring + (size_t)slot * tl.S + poff, ga, valid, ragged, ta, pad0);
                } else {
                    window_to_tmem_gen<WS>(ring + (size_t)slot * tl.S + poff, ga, valid, GEN && ragged, ta, pad0);
                }
            }
            else
                window_to_tmem_bulk<WS>(ring + (size_t)slot * tl.S + poff + win_off, valid, rowB,
                                        tmem + buf * A_STRIDE + ((uint32_t)(q * 32) << 16), pad0);
            if (part) ptx::mbar_arrive(EMPTY(bslot));   // every window of this image is in TMEM
            // W_c of a new channel is rebuilt AFTER this tile's windows are in TMEM, so the copy above
            // overlaps the last MMA of the previous channel.
            if (lt > 0) rebuild_weight(c, lt);
            ptx::tc_fence_before_sync();
            ptx::mbar_arrive(A_FULL + 8 * buf);
            k += np_eff;
            // the next tile starts a new channel: have its table row in flight during the next copy
            if (t + 1 < t1 && (t + 1) - c * tl.tiles_per_c == tl.tiles_per_c) {
                if constexpr (WS == 14) {
                    if (!fullw) {
                        table_to_regs14(T + (long long)(c + 1) * Cf::NB, reverse != 0, rt, tabv);
                        tabv_ready = true;
                    }
                } else if (!Mw7) {
                    table_to_regs7(T + (long long)(c + 1) * Cf::NB, reverse != 0, rt, tabv);
                    tabv_ready = true;
                }
            }
        }
    } else if (warp < 10) {
        // ------------------------------------------------------------------ epilogue
        const int q = warp & 3;
        const int m = q * 32 + lane;
        const int pl = m / wpf, wl = m % wpf;
        const int wyl = wl / g.nww, wx = wl % g.nww;
        const int win_off = ((wyl * WS) * g.W + wx * WS) * 2;
        GenAddr<WG ? WS : 1> ga;
        if constexpr (STRIP) gen_addr_init_strip<WS>(ga, g, wyl, wx);
        else if constexpr (GEN) gen_addr_init<WS>(ga, g, wyl, wx);
        else if constexpr (WG) gen_addr_init_plain<WS>(ga, g.W, wyl, wx);
        const int gq = m / og.lanes;                    // output group of this thread
        const int pg = pl - gq * og.images;             // image inside the group
        const uint32_t out_bytes = (uint32_t)og.images * tl.S;
        uint32_t lt = 0;
        for (int t = t0; t < t1; ++t, ++lt) {
            int c, b0, wy0, np_eff, rows_eff;
            tile_decode(t, c, b0, wy0, np_eff, rows_eff);
            const bool valid = pl < np_eff && wy0 + wyl < g.nwh;
            if constexpr (STRIP) {
                if (ragged) ga.rowmask = gen_strip_rowmask<WS>(g, wy0 + wyl);
            }
            // the output frame is nout / og.n tiles deep: tile lt uses frame lt mod depth, group gq its buffer gq
            const uint32_t otile = lt % (nout / og.n), ob = otile * og.n + gq, use = lt / (nout / og.n);
            uint8_t* img = outb + (size_t)ob * out_bytes + (size_t)pg * tl.S;
            auto drain_half = [&](auto hc) {
                constexpr int h = decltype(hc)::value;
                uint32_t pk[Hs::TOEP ? 49 : Hs::ncols(h) / 2];
                ptx::mbar_wait(D_FULL + 8 * h, lt & 1);
                ptx::tc_fence_after_sync();
                accum_half_to_packed<WS, BF16, h>(tmem_d + Hs::col0(h) + ((uint32_t)(q * 32) << 16), pk);
                ptx::tc_fence_before_sync();
                ptx::mbar_arrive(D_EMPTY + 8 * h);                                 // the MMAs of the next tile may overwrite this half
                if (h == 0 && sbox != 2) ptx::mbar_wait(OUT_EMPTY + 8 * ob, (use & 1) ^ 1);     // the buffer's previous contents have been read out
                if constexpr (flat7) {
                    if (valid) packed_to_flat7(img, pk);
                } else if (valid) {
                    if constexpr (WG) {
                        if constexpr (GEN && WS % 2 == 0) {
                            if (g.sw & 1) {
                                if (ragged) packed_to_window_gen<WS, Hs::word0(h), Hs::word1(h), true, 1>(img, ga, pk);
                                else packed_to_window_gen<WS, Hs::word0(h), Hs::word1(h), false, 1>(img, ga, pk);
                            } else {
                                if (ragged) packed_to_window_gen<WS, Hs::word0(h), Hs::word1(h), true, 0>(img, ga, pk);
                                else packed_to_window_gen<WS, Hs::word0(h), Hs::word1(h), false, 0>(img, ga, pk);
                            }
                        } else if (GEN && ragged) {
                            packed_to_window_gen<WS, Hs::word0(h), Hs::word1(h), true>(img, ga, pk);
                        } else {
                            packed_to_window_gen<WS, Hs::word0(h), Hs::word1(h), false>(img, ga, pk);
                        }
                    } else {
                        packed_to_window<WS, Hs::word0(h), Hs::word1(h)>(img + win_off, rowB, pk);
                    }
                }
            };
            drain_half(std::integral_constant<int, 0>{});
            if constexpr (Hs::NH > 1) drain_half(std::integral_constant<int, 1>{});
            if (sbox == 2) {
                // plane boxes: a plane is not a multiple of 16 bytes, so no bulk store can write it.  A group is this
                // warp's own images (a warp always covers whole images here), so the warp copies them out itself with
                // 8-byte stores (4-byte when H*W is not a multiple of 4), lane = chunk of a plane, eight planes in
                // flight: four warps in parallel instead of the one store warp (which ran at 3 bytes per cycle, bound by
                // its own instruction latencies: 11 us per tile of 128 14 x 14 planes).
                __syncwarp();
                const int p_first = gq * og.images, np = min(og.images, np_eff - p_first);
                if (np > 0) {
                    const uint8_t* src = outb + (size_t)ob * out_bytes;
                    uint8_t* dst = reinterpret_cast<uint8_t*>(y + ((long long)(b0 + p_first) * g.C + c) * plane_elems);
                    if (plane_elems % 4 == 0) copy_planes_out<uint2>(src, dst, np, tl.S, (long long)g.C * plane_elems * 2, (int)(plane_elems / 4), lane);
                    else if (plane_elems % 2 == 0) copy_planes_out<uint32_t>(src, dst, np, tl.S, (long long)g.C * plane_elems * 2, (int)(plane_elems / 2), lane);
                    else copy_planes_out<uint16_t>(src, dst, np, tl.S, (long long)g.C * plane_elems * 2, (int)plane_elems, lane);   // 7 x 7: planes start on odd elements
                }
                __syncwarp();
                continue;
            }
            ptx::fence_proxy_async_smem();      // generic-proxy writes -> the bulk store's async-proxy reads
            ptx::mbar_arrive(OUT_FULL + 8 * ob);
        }
    } else {
        // ------------------------------------------------------------------ store
        if (t1 > t0 && T) {   // pull this CTA's table rows into L2 ahead of the W_c builds
            const int c_first = t0 / tl.tiles_per_c, c_last = (t1 - 1) / tl.tiles_per_c;
            const char* base = reinterpret_cast<const char*>(T + (long long)c_first * Cf::NB);
            const long long nbytes = (long long)(c_last - c_first + 1) * Cf::NB * 2;
            for (long long off = lane * 128ll; off < nbytes; off += 32 * 128)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(base + off));
        }
        if (sbox == 2) {
            // plane boxes: the epilogue warps store their own groups
        } else if (lane < nout) {
            // Lane ob = (frame, gq) owns output buffer ob: group gq of the tiles lt = frame mod depth.  It
            // bulk-stores the group's images and releases the buffer once the copy engine has read it.
            // One lane per buffer, so the ~1.4 us a store needs before its source may be overwritten is
            // waited for in parallel.  (A single thread issuing everything in order and releasing a tile
            // late measured 2 us slower per launch on cfg3; a rotation that put the lanes several tiles
            // apart hung: every lane walks the tile loop in step and skips the tiles that are not its own.)
            const uint32_t depth = nout / og.n, frame = lane / og.n, gq = lane - frame * og.n;
            const uint32_t out_bytes = (uint32_t)og.images * tl.S;
            uint32_t lt = 0;
            for (int t = t0; t < t1; ++t, ++lt) {
                int c, b0, wy0, np_eff, rows_eff;
                tile_decode(t, c, b0, wy0, np_eff, rows_eff);
                if (lt % depth != frame) continue;
                const uint32_t bytes = (uint32_t)rows_eff * rowB;
                ptx::mbar_wait(OUT_FULL + 8 * lane, (lt / depth) & 1);
                const int p_first = gq * og.images, p_end = min(p_first + og.images, np_eff);
                if (sbox) {
                    if (p_first < p_end) ptx::tma_store_4d(&my, 0, 0, c, b0 + p_first, ptx::smem_u32(outb + (size_t)lane * out_bytes));
                } else
                for (int p = p_first; p < p_end; ++p) {
                    const uint32_t src = ptx::smem_u32(outb + (size_t)lane * out_bytes + (size_t)(p - p_first) * tl.S);
                    if constexpr (STRIP) {           // strip in rolled row order: up to two runs of image rows
                        const StripRuns sr = strip_runs(g, wy0 * WS, rows_eff);
                        uint16_t* pl0 = y + ((long long)(b0 + p) * g.C + c) * plane_elems;
                        if (sr.nA > 0) ptx::bulk_s2g(pl0 + (long long)sr.a0 * g.W, src, (uint32_t)sr.nA * rowB);
                        if (sr.nB > 0) ptx::bulk_s2g(pl0, src + sr.n1 * rowB, (uint32_t)sr.nB * rowB);
                        continue;
                    }
                    uint16_t* dst = y + ((long long)(b0 + p) * g.C + c) * plane_elems + (long long)wy0 * WS * g.W;
                    ptx::bulk_s2g(dst, src, bytes);
                }
                ptx::bulk_commit();
                ptx::bulk_wait_read<0>();
                ptx::mbar_arrive(OUT_EMPTY + 8 * lane);
            }
            ptx::bulk_wait_read<0>();   // the sources are in this CTA's shared memory: reads must finish before it exits
        }
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem, bulk_tmem_cols<WS>());
}

// Shared memory left after the weights / tables / barriers is cut into frame-image slots: an output
// frame `depth` tiles deep (one buffer per output group and tile) and an input ring of `nslot` slots.
// Both sides want about 96 KB: a bulk store takes ~1.4 us until its source may be overwritten and a
// load ~1.5-2 us to land, i.e. ~50 KB in flight per SM each way at the ~35 GB/s per SM the copy engine
// sustains, plus the tile being worked on.  More input in flight measured SLOWER (112 x 112 maps:
// 4 slots of 25 KB 114 us, 3 slots 104 us; also for a plain bulk-copy ring,
// DESIGN.md section 7.7); less starves small tiles (w = 7: 12.5 KB per tile).
// Returns false when a tile of output plus a tile + 1 of input does not fit.
template <int WS>
bool bulk_slots(const TcTiles& tl, int wpf, int* nslot, int* nout, int ctas = 1, int extra = 0)
{
    const OutGroups og = out_groups(tl, wpf);
    const long long room = (ctas == 1 ? 227ll * 1024 : 113ll * 1024) - 1024 - BulkSmem<WS>::FIXED - extra;
    const long long total = room / tl.S, out_tile = (long long)og.n * og.images;
    const long long kSide = 96 * 1024 / ctas;
    long long depth = (kSide + out_tile * tl.S / 2) / (out_tile * tl.S);
    if (depth > kMaxOutBufs / og.n) depth = kMaxOutBufs / og.n;
    while (depth > 1 && total - depth * out_tile < tl.NP + 1) --depth;
    if (depth < 1) return false;
    long long ni = total - depth * out_tile;
    long long in_cap = kSide / tl.S;
    if (in_cap < tl.NP + 1) in_cap = tl.NP + 1;
    if (ni > in_cap) ni = in_cap;
    if (ni > kMaxSlots) ni = kMaxSlots;
    if (ni < tl.NP + 1) return false;
    *nslot = (int)ni;
    *nout = (int)(depth * og.n);
    return true;
}

// 0 = not servable by the bulk kernel, 1 = aligned fast form, 2 = general form (shift / ragged).
template <int WS>
int bulk_mode(const Geom& g, const TcTiles& tl, const void* x, const void* y)
{
    if (g.layout != WBMM_LAYOUT_NCHW) return 0;
    const bool pb = ((long long)g.H * g.W * 2) % 16 != 0;       // planes no bulk copy can move: tensor-map "plane boxes"
    if (pb && plane_box_images(g, tl) == 0) return 0;
    if (reinterpret_cast<uintptr_t>(x) % 16 != 0 || reinterpret_cast<uintptr_t>(y) % 16 != 0) return 0;
    if (tl.NP > kMaxSlots || tl.ntiles > 0x3fffffffll) return 0;
    int nslot_, nout_;
    if (!bulk_slots<WS>(tl, tl.NSY * g.nww, &nslot_, &nout_)) return 0;
    const bool plain = g.sh == 0 && g.sw == 0 && g.H == g.Hp && g.W == g.Wp;
    if (plain && (pb || (tl.frame_rows * g.W * 2) % 16 == 0) && (WS % 2 == 0 || g.W % 2 == 0 || (pb && g.H == WS && g.W == WS))) return 1;   // odd w: rows must be word-aligned (7 x 7 maps: the flat form)
    // general form: whole images in natural layout, word-granular window addressing (W, W' even)
    // (an odd W' -- ragged maps at odd w -- is fine without a column shift: nothing wraps)
    // maps cut into strips of window rows (more than 128 windows per image): rolled-order frames, rows of 16-byte multiples
    return ((tl.nstrips == 1 || (g.W * 2) % 16 == 0) && g.W % 2 == 0 && (g.Wp % 2 == 0 || g.sw == 0)) ? 2 : 0;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (libcuda is not linked).
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn bulk_encode_fn()
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

// Small frame images (28 x 28: 1568 bytes) make one bulk copy per image the bottleneck: 64 copy-engine
// operations per tile.  When whole images are tiled (nstrips == 1) the images of one output group are
// moved by ONE tensor-map box instead: the activation is viewed as (a, b, C, B) with a*b = H*W, a a
// multiple of 8 elements and both <= 256, box {a, b, 1, group}.  Returns the group size (0 = not applicable).
}  // namespace

// Tensor map over an NCHW activation viewed as (a, b, C, B), a*b = H*W, with box {a, b, 1, images}: `images`
// whole frame images of one channel per copy.  False when H*W has no legal factorisation or the driver
// entry point is missing.  `map` is a CUtensorMap.
// Plane boxes: when H*W*2 is not a multiple of 16 (14 x 14 maps: 392 B) neither a bulk copy nor a tensor map with a
// channel dimension can address one plane, but a map over [B][C*H*W] can: a box of `images` rows x (H*W + 7 rounded up
// to 8) elements starting at the 16-byte boundary at or below element c*H*W (it also reads a few elements of the
// neighbouring planes; the slot pitch is the padded size and the plane sits (c*H*W mod 8) elements into its slot).  Returns the images per box (8, 4 or 2), 0 when the shape does not allow it.
constexpr long long kPlaneBoxMax = 2048;        // padded plane elements: 256 box rows of 8

int plane_box_images(const Geom& g, const TcTiles& tl)
{
    const long long hw = (long long)g.H * g.W;
    const long long hwp = (hw + 14) / 8 * 8;       // the box starts up to 7 elements before the plane (16-byte boundary)
    const bool flat7 = g.w == 7 && g.H == 7 && g.W == 7 && g.sh == 0 && g.sw == 0;      // the plane is one window (window_to_tmem_flat7)
    if (tl.nstrips != 1 || (hw % 2 != 0 && !flat7) || hwp > kPlaneBoxMax || (g.C * hw * 2) % 16 != 0 || g.C * hw > 0x7fffffffll) return 0;
    for (int cand = 8; cand >= 2; cand >>= 1)
        if (tl.NP % cand == 0 && g.B % cand == 0 && (cand * hwp * 2) % 128 == 0) return cand;
    return 0;
}

bool plane_box_map(const Geom& g, int dtype, const void* base, int images, void* map)
{
    const long long hw = (long long)g.H * g.W, hwp = (hw + 14) / 8 * 8;
    EncodeTiledFn fn = bulk_encode_fn();
    if (!fn || images < 1 || images > 256 || hwp > kPlaneBoxMax) return false;
    const cuuint64_t row = (cuuint64_t)g.C * hw;
    // planes of more than 256 elements (30 x 30: 900): a box dimension holds at most 256 elements, so the row of an image
    // is viewed as (8 elements, C*H*W / 8) and the box is {8, padded plane / 8}: the same dense bytes in shared memory,
    // box start (0, c*H*W / 8) -- see plane_box_2d()
    const bool two_d = hwp > 256;
    const cuuint64_t dims[4] = {two_d ? 8 : row, two_d ? row / 8 : 1, 1, (cuuint64_t)g.B};
    const cuuint64_t strides[3] = {two_d ? 16 : row * 2, row * 2, row * 2};
    const cuuint32_t boxd[4] = {(cuuint32_t)(two_d ? 8 : hwp), (cuuint32_t)(two_d ? hwp / 8 : 1), 1, (cuuint32_t)images};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUtensorMapDataType dt = dtype == WBMM_DTYPE_BF16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16;
    return fn(static_cast<CUtensorMap*>(map), dt, 4, const_cast<void*>(base), dims, strides, boxd, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool image_box_map(const Geom& g, int dtype, const void* base, int images, void* map)
{
    const long long hw = (long long)g.H * g.W, ib = hw * 2;
    int a = 0;
    for (int cand = 256; cand >= 8; cand -= 8)
        if (hw % cand == 0 && hw / cand <= 256) { a = cand; break; }
    EncodeTiledFn fn = bulk_encode_fn();
    if (a == 0 || !fn || images < 1 || images > 256) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)a, (cuuint64_t)(hw / a), (cuuint64_t)g.C, (cuuint64_t)g.B};
    const cuuint64_t strides[3] = {(cuuint64_t)a * 2, (cuuint64_t)ib, (cuuint64_t)ib * g.C};
    const cuuint32_t boxd[4] = {(cuuint32_t)a, (cuuint32_t)(hw / a), 1, (cuuint32_t)images};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUtensorMapDataType dt = dtype == WBMM_DTYPE_BF16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16;
    return fn(static_cast<CUtensorMap*>(map), dt, 4, const_cast<void*>(base), dims, strides, boxd, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

namespace {

int bulk_box_mode(const Geom& g, const TcTiles& tl, int dtype, const void* x, const void* y, int* S, int* sbox,
                  CUtensorMap* mx, CUtensorMap* my)
{
    *sbox = 0;
    if (tl.nstrips != 1) return 0;
    const long long hw = (long long)g.H * g.W, ib = hw * 2;
    if (ib > 4096) return 0;
    // load box: the largest group of images (a divisor of the tile and of the batch, at most 8: the repack
    // warps start on a group as soon as it has landed) whose bytes are a multiple of 128
    int LB = 0;
    for (int cand = 8; cand >= 2; cand >>= 1)
        if (tl.NP % cand == 0 && g.B % cand == 0 && (cand * ib) % 128 == 0) { LB = cand; break; }
    if (LB == 0) return 0;
    // store box: one output group, when that is a legal box too
    const int G = out_groups(tl, tl.NSY * g.nww).images;
    const bool sb = G >= 2 && g.B % G == 0 && tl.NP % G == 0 && (G * ib) % 128 == 0;
    if (!image_box_map(g, dtype, x, LB, mx)) return 0;
    if (sb && !image_box_map(g, dtype, y, G, my)) return 0;
    *S = (int)ib;      // boxes land densely: the slot stride is exactly one image
    *sbox = sb ? 1 : 0;
    return LB;
}

template <int WS, bool BF16, bool GEN, bool STRIP = false, int V = 0>
cudaError_t launch_bulk(const Geom& g, const TcTiles& tl_in, const void* x, const void* T, const void* Tl, void* y,
                        bool reverse, cudaStream_t s, const void* bias, uint32_t ident_bits, const void* Mfull = nullptr)
{
    const int extra = (WS == 14 && V == 2) ? BulkSmem<WS>::FULL_EXTRA : 0;      // cached-M mode at w = 14: the given matrix pushes the ring back
    auto k = tc_bulk_kernel<WS, BF16, GEN, STRIP, V>;
    int nslot = 0, nout = 0;
    TcTiles tl = tl_in;
    CUtensorMap mx, my;
    memset(&mx, 0, sizeof(mx));
    memset(&my, 0, sizeof(my));
    int sbox = 0, box = 0;
    const int wpf = tl.NSY * g.nww;
    // shared-memory plan for `ctas` CTAs per SM; false when nothing fits
    auto configure = [&](int ctas) -> bool {
        tl = tl_in;
        sbox = box = 0;
        if (((long long)g.H * g.W * 2) % 16 != 0) {
            // plane boxes (see plane_box_images): loads by tensor map, stores by the store warp's own 8-byte stores
            box = plane_box_images(g, tl_in);
            if (box == 0 || !plane_box_map(g, BF16 ? WBMM_DTYPE_BF16 : WBMM_DTYPE_F16, x, box, &mx)) return false;
            sbox = 2;
            tl.S = (int)(((long long)g.H * g.W + 14) / 8 * 8 * 2);
            if (!bulk_slots<WS>(tl, wpf, &nslot, &nout, ctas, extra)) return false;
            nslot -= nslot % box;
            return nslot >= tl.NP + box;
        }
        box = bulk_box_mode(g, tl_in, BF16 ? WBMM_DTYPE_BF16 : WBMM_DTYPE_F16, x, y, &tl.S, &sbox, &mx, &my);
        if (box) {
            nslot = 0;
            if (bulk_slots<WS>(tl, wpf, &nslot, &nout, ctas, extra)) nslot -= nslot % box;      // groups never wrap around the ring
            if (nslot >= tl.NP + box) return true;
            box = sbox = 0;                                                             // (does not fit: one copy per image)
            tl = tl_in;
        }
        return bulk_slots<WS>(tl, wpf, &nslot, &nout, ctas, extra);
    };
    int ctas = bulk_ctas_per_sm<WS, GEN, STRIP>();
    if (!configure(ctas)) {
        if (ctas == 1) return cudaErrorInvalidConfiguration;
        ctas = 1;
        if (!configure(ctas)) return cudaErrorInvalidConfiguration;
    }
    const size_t smem = (size_t)BulkSmem<WS>::FIXED + extra + (size_t)(nslot + nout * out_groups(tl, wpf).images) * tl.S;
    static SmemOptIn smem_state;
    cudaError_t e = ensure_dynamic_smem(reinterpret_cast<const void*>(k), smem, &smem_state);
    if (e != cudaSuccess) return e;
    int grid = (int)(tl.ntiles < (long long)num_sms() * ctas ? tl.ntiles : (long long)num_sms() * ctas);
    if (grid > kMaxGrid) grid = kMaxGrid;
    // the schedule depends on (tiles, tiles per channel, grid) only: keep the last one
    static std::mutex mu;
    static TilePart cached;
    static long long key_n = -1;
    static int key_tpc = -1, key_grid = -1, cached_used = 0;
    TilePart part;
    {
        std::lock_guard<std::mutex> lock(mu);
        if (key_n != tl.ntiles || key_tpc != tl.tiles_per_c || key_grid != grid) {
            cached_used = partition_tiles(tl, grid, WS == 14 ? 0.15 : 0.3, &cached);
            key_n = tl.ntiles; key_tpc = tl.tiles_per_c; key_grid = grid;
        }
        part = cached;
        grid = cached_used;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(kThreadsB);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k, g, tl, part, nslot, nout, (const uint16_t*)x, (const uint16_t*)T, (const uint16_t*)Tl,
                              (uint16_t*)y, reverse ? 1 : 0, box, sbox, mx, my, (const uint16_t*)bias, ident_bits, (const uint16_t*)Mfull);
}

// the table kernel (V = 0), or the one with the run-time extras (V = 1)
template <int WS, bool BF16, bool GEN, bool STRIP = false>
cudaError_t launch_bulk_v(bool extras, const Geom& g, const TcTiles& tl, const void* x, const void* T, const void* Tl, void* y,
                          bool reverse, cudaStream_t s, const void* bias, uint32_t ident_bits)
{
    // The general form at w = 14 sits at the register limit (168, with spills), and ptxas spills MORE in its V = 0
    // instantiation than in V = 1 (cfg5 forward 22.5 -> 24.2 us): that one form keeps the run-time flags.
    if constexpr (WS == 14 && GEN) return launch_bulk<WS, BF16, GEN, STRIP, 1>(g, tl, x, T, Tl, y, reverse, s, bias, ident_bits);
    return extras ? launch_bulk<WS, BF16, GEN, STRIP, 1>(g, tl, x, T, Tl, y, reverse, s, bias, ident_bits)
                  : launch_bulk<WS, BF16, GEN, STRIP, 0>(g, tl, x, T, Tl, y, reverse, s, bias, ident_bits);
}

template <int WS>
size_t generic_smem(const TcTiles& tl)
{
    return (size_t)WinCfg<WS>::WC_BYTES + WinCfg<WS>::TS_BYTES + (size_t)tl.NP * tl.S;
}

template <int WS, bool BF16>
cudaError_t launch_generic(const Geom& g, const TcTiles& tl, const void* x, const void* T, void* y, bool reverse,
                           cudaStream_t s, const void* Mfull = nullptr, const void* bias = nullptr)
{
    auto k = tc_generic_kernel<WS, BF16>;
    const size_t smem = generic_smem<WS>(tl);
    static SmemOptIn smem_state;
    cudaError_t e = ensure_dynamic_smem(reinterpret_cast<const void*>(k), smem, &smem_state);
    if (e != cudaSuccess) return e;
    const int grid = (int)(tl.ntiles < num_sms() ? tl.ntiles : num_sms());
    k<<<grid, kThreadsG, smem, s>>>(g, tl, (const uint16_t*)x, (const uint16_t*)T, (uint16_t*)y, reverse ? 1 : 0,
                                    (const uint16_t*)Mfull, (const uint16_t*)bias);
    return cudaGetLastError();
}

}  // namespace

cudaError_t ensure_dynamic_smem(const void* kernel, size_t bytes, SmemOptIn* state)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool cached = dev >= 0 && dev < kMaxDevices;
    if (cached && (size_t)state->bytes[dev].load(std::memory_order_acquire) >= bytes) return cudaSuccess;
    static std::mutex mu;      // the attribute is per (kernel, device): raise it once, monotonically
    std::lock_guard<std::mutex> lock(mu);
    if (cached && (size_t)state->bytes[dev].load(std::memory_order_relaxed) >= bytes) return cudaSuccess;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess && cached) state->bytes[dev].store((int)bytes, std::memory_order_release);
    return e;
}

// Multiprocessors of the CURRENT device (cached per device).
int num_sms()
{
    static std::atomic<int> cache[kMaxDevices];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 148;
    const bool cached = dev >= 0 && dev < kMaxDevices;
    int n = cached ? cache[dev].load(std::memory_order_relaxed) : 0;
    if (n == 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        if (cached) cache[dev].store(n, std::memory_order_relaxed);
    }
    return n;
}

// Greedy contiguous partition of the tile sequence over `grid` CTAs minimising the largest cost,
// cost = tiles + kSwitchCost per channel boundary strictly inside a CTA's range.
int partition_tiles(const TcTiles& tl, int grid, double kSwitchCost, TilePart* part)
{
    const int n = (int)tl.ntiles, tpc = tl.tiles_per_c;
    auto fill = [&](double cap, TilePart* out) {
        int b = 0, t = 0;
        if (out) out->start[0] = 0;
        while (t < n) {
            double cost = 0;
            int first = t;
            while (t < n) {
                const double add = 1.0 + ((t > first && t % tpc == 0) ? kSwitchCost : 0.0);
                if (cost + add > cap + 1e-9 && t > first) break;
                cost += add;
                ++t;
            }
            ++b;
            if (out && b <= kMaxGrid) out->start[b] = t;
            if (b > grid) return b;
        }
        return b;
    };
    double lo = (double)n / grid, hi = (double)n / grid * 2 + 4;
    for (int it = 0; it < 40; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (fill(mid, nullptr) <= grid) hi = mid; else lo = mid;
    }
    // `hi` is the smallest achievable maximum cost; packing every CTA up to it would leave the last CTAs
    // idle (cfg5 dT: 128 of 148), and the kernels are bound by per-SM copy-engine throughput, so spread
    // the tiles over ALL CTAs instead: each CTA takes its share of what is left, never more than `hi`.
    const double cap = hi;
    int t = 0, used = 0;
    part->start[0] = 0;
    for (int b = 0; b < grid && t < n; ++b) {
        // cost of everything that is left if a CTA starts at tile t: tiles + channel boundaries inside (t, n)
        const double rem = (n - t) + kSwitchCost * ((n - 1) / tpc - t / tpc);
        const double target = rem / (grid - b);
        double cost = 0;
        const int first = t;
        while (t < n) {
            const double add = 1.0 + ((t > first && t % tpc == 0) ? kSwitchCost : 0.0);
            if (t > first && (cost + add > cap + 1e-9 || cost + 0.5 * add > target)) break;
            cost += add;
            ++t;
        }
        part->start[b + 1] = t;
        used = b + 1;
    }
    if (t < n) used = fill(hi, part);     // (rounding left tiles over: fall back to the packed schedule)
    for (int b = used; b < kMaxGrid; ++b) part->start[b + 1] = n;
    return used;
}

bool tc_tiles(const Geom& g, TcTiles* t)
{
    const int wpp = g.nwh * g.nww;
    if (g.nww > 128) return false;
    if (wpp <= 128) {
        t->NSY = g.nwh;
        t->NP = 128 / wpp;
        if (t->NP > 64) t->NP = 64;      // one window per image (14 x 14 at w = 14): half-filled tiles, so that the ring's
                                         // slot count (one frame image each) stays within kMaxSlots
        if (t->NP > g.B) t->NP = g.B;
        // planes that only tensor-map "plane boxes" can move (H*W*2 not a multiple of 16): the images of a tile come in
        // boxes of 8, 4 or 2 -- take the largest tile that is whole boxes (30 x 30 at w = 14: 14 -> 12 images)
        const long long hw = (long long)g.H * g.W, hwp = (hw + 14) / 8 * 8;
        if (g.layout == WBMM_LAYOUT_NCHW && (hw * 2) % 16 != 0 && (hw % 2 == 0 || (g.w == 7 && hw == 49)) && hwp <= kPlaneBoxMax && (g.C * hw * 2) % 16 == 0) {
            int best = 0;
            for (int cand = 8; cand >= 2; cand >>= 1)
                if (g.B % cand == 0 && (cand * hwp * 2) % 128 == 0 && t->NP / cand * cand > best) best = t->NP / cand * cand;
            if (best > 0) t->NP = best;
        }
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

bool tc_bulk_supported(const Geom& g, int dtype, const void* x, const void* y)
{
    if (dtype != WBMM_DTYPE_BF16 && dtype != WBMM_DTYPE_F16) return false;
    if (g.w != 7 && g.w != 14) return false;
    TcTiles tl;
    if (!tc_tiles(g, &tl)) return false;
    return (g.w == 7 ? bulk_mode<7>(g, tl, x, y) : bulk_mode<14>(g, tl, x, y)) != 0;
}

bool tc_hier_supported(const Geom& g, int dtype, const void* x, const void* y)
{
    if (dtype != WBMM_DTYPE_BF16 && dtype != WBMM_DTYPE_F16) return false;
    if (g.w != 14) return false;
    TcTiles tl;
    if (!tc_tiles(g, &tl)) return false;
    return bulk_mode<14>(g, tl, x, y) != 0;
}

cudaError_t tc_forward(const Geom& g, int dtype, const void* x, const void* T, const void* Tl, void* y, bool reverse,
                       cudaStream_t stream, int* launches, int* path, const void* bias, uint32_t ident_bits)
{
    TcTiles tl;
    if (!tc_tiles(g, &tl)) return cudaErrorNotSupported;
    if (tl.ntiles == 0) return cudaSuccess;
    *launches += 1;
    const bool bf = dtype == WBMM_DTYPE_BF16;
    const int mode = g.w == 7 ? bulk_mode<7>(g, tl, x, y) : bulk_mode<14>(g, tl, x, y);
    if (mode != 0) {
        *path = WBMM_PATH_TC_TMA;
        const bool extras = Tl || bias || ident_bits;
        if (mode == 2 && tl.nstrips > 1) {      // general addressing on strips of window rows
            if (g.w == 7) return bf ? launch_bulk_v<7, true, true, true>(extras, g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits)
                                    : launch_bulk_v<7, false, true, true>(extras, g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits);
            return bf ? launch_bulk_v<14, true, true, true>(extras, g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits)
                      : launch_bulk_v<14, false, true, true>(extras, g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits);
        }
        if (g.w == 7 && mode == 1 && g.H == 7 && g.W == 7)       // one-window maps: the flat-plane variant
            return bf ? launch_bulk<7, true, false, false, 2>(g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits)
                      : launch_bulk<7, false, false, false, 2>(g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits);
        const int sel = (g.w == 7 ? 0 : 4) + (bf ? 2 : 0) + (mode == 2 ? 1 : 0);
        switch (sel) {
        case 0: return launch_bulk_v<7, false, false>(extras, g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits);
        case 1: return launch_bulk_v<7, false, true>(extras, g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits);
        case 2: return launch_bulk_v<7, true, false>(extras, g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits);
        case 3: return launch_bulk_v<7, true, true>(extras, g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits);
        case 4: return launch_bulk_v<14, false, false>(extras, g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits);
        case 5: return launch_bulk_v<14, false, true>(extras, g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits);
        case 6: return launch_bulk_v<14, true, false>(extras, g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits);
        default: return launch_bulk_v<14, true, true>(extras, g, tl, x, T, Tl, y, reverse, stream, bias, ident_bits);
        }
    }
    if (Tl || bias || ident_bits) return cudaErrorNotSupported;      // hierarchical / fused variants exist in the bulk kernel only
    *path = WBMM_PATH_TC_GATHER;
    if (g.w == 7)
        return bf ? launch_generic<7, true>(g, tl, x, T, y, reverse, stream)
                  : launch_generic<7, false>(g, tl, x, T, y, reverse, stream);
    return bf ? launch_generic<14, true>(g, tl, x, T, y, reverse, stream)
              : launch_generic<14, false>(g, tl, x, T, y, reverse, stream);
}

// Cached-M mode (WBMM-C): the per-channel matrices are given, nothing is built from a table.
cudaError_t tc_forward_matrix(const Geom& g, int dtype, const void* x, const void* M, const void* bias, void* y,
                              bool transpose, cudaStream_t stream, int* launches, int* path)
{
    TcTiles tl;
    if (!tc_tiles(g, &tl)) return cudaErrorNotSupported;
    if (tl.ntiles == 0) return cudaSuccess;
    *launches += 1;
    const bool bf = dtype == WBMM_DTYPE_BF16;
    if (g.w == 7) {
        // w = 7: the pipelined kernel holds the whole 8 KB W_c in shared memory anyway -- the given matrix takes its place
        const int mode = bulk_mode<7>(g, tl, x, y);
        if (mode != 0) {
            *path = WBMM_PATH_TC_TMA;
            if (mode == 2 && tl.nstrips > 1)
                return bf ? launch_bulk<7, true, true, true, 1>(g, tl, x, nullptr, M, y, transpose, stream, bias, 0u)
                          : launch_bulk<7, false, true, true, 1>(g, tl, x, nullptr, M, y, transpose, stream, bias, 0u);
            if (mode == 2)
                return bf ? launch_bulk<7, true, true, false, 1>(g, tl, x, nullptr, M, y, transpose, stream, bias, 0u)
                          : launch_bulk<7, false, true, false, 1>(g, tl, x, nullptr, M, y, transpose, stream, bias, 0u);
            if (g.H == 7 && g.W == 7)
                return bf ? launch_bulk<7, true, false, false, 2>(g, tl, x, nullptr, M, y, transpose, stream, bias, 0u)
                          : launch_bulk<7, false, false, false, 2>(g, tl, x, nullptr, M, y, transpose, stream, bias, 0u);
            return bf ? launch_bulk<7, true, false, false, 1>(g, tl, x, nullptr, M, y, transpose, stream, bias, 0u)
                      : launch_bulk<7, false, false, false, 1>(g, tl, x, nullptr, M, y, transpose, stream, bias, 0u);
        }
    }
    if (g.w == 14) {
        // w = 14: the given matrix (100 KB in the row-padded operand layout) takes the place of the Toeplitz library in
        // the same pipelined kernel, where a tile and a half of input plus a tile of output still fit beside it
        const int mode = bulk_mode<14>(g, tl, x, y);
        int ns_ = 0, no_ = 0;
        if (mode != 0 && !(mode == 2 && tl.nstrips > 1) && bulk_slots<14>(tl, tl.NSY * g.nww, &ns_, &no_, 1, BulkSmem<14>::FULL_EXTRA)) {
            *path = WBMM_PATH_TC_TMA;
            cudaError_t e;
            if (mode == 2)
                e = bf ? launch_bulk<14, true, true, false, 2>(g, tl, x, nullptr, nullptr, y, transpose, stream, bias, 0u, M)
                       : launch_bulk<14, false, true, false, 2>(g, tl, x, nullptr, nullptr, y, transpose, stream, bias, 0u, M);
            else
                e = bf ? launch_bulk<14, true, false, false, 2>(g, tl, x, nullptr, nullptr, y, transpose, stream, bias, 0u, M)
                       : launch_bulk<14, false, false, false, 2>(g, tl, x, nullptr, nullptr, y, transpose, stream, bias, 0u, M);
            if (e != cudaErrorInvalidConfiguration) return e;
            cudaGetLastError();          // (the ring did not fit after all: the gather kernel below)
        }
    }
    *path = WBMM_PATH_TC_GATHER;
    if (g.w == 7)
        return bf ? launch_generic<7, true>(g, tl, x, nullptr, y, transpose, stream, M, bias)
                  : launch_generic<7, false>(g, tl, x, nullptr, y, transpose, stream, M, bias);
    return bf ? launch_generic<14, true>(g, tl, x, nullptr, y, transpose, stream, M, bias)
              : launch_generic<14, false>(g, tl, x, nullptr, y, transpose, stream, M, bias);
}


}  // namespace wbmm
