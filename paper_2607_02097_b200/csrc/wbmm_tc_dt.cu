// WBMM table gradient on the tensor cores (autograd of Alg. 1):
//     S_c[i, j] = sum over windows n of dY[n, i] * X[n, j]          (tcgen05.mma, fp32 in TMEM)
//     dT[c, k]  = sum over pairs (i, j) with rel(i, j) = k of S_c[i, j]   (Eq. 6-7 as a scatter)
//
// The contraction index of S is the WINDOW, so both operands are "MN-major": thread n writes its
// window's N values as 16-byte vectors of 8 consecutive positions into the no-swizzle core-matrix
// layout  addr(pos, n) = (pos/8)*SBO + (n/8)*128 + (n%8)*16 + (pos%8)*2  -- 32 lanes write 512
// contiguous bytes.  One tile = 128 windows = MMA K of 128 (8 instructions per M-tile).  S stays in
// TMEM while a CTA walks the tiles of one channel; at the end of the channel segment every warp
// folds its 32 rows of S into a private copy of the (2w-1)^2 bins in shared memory (plain
// read-add-write: within one column step the 32 rows of a warp hit 32 different bins), the copies
// are summed and ONE pass of red.global.add.f32 per bin goes to dT.
//
//   warp 0      producer   bulk loads of the x and dy frame images of a tile into the slot ring
//   warp 1      MMA        MT * 8 tcgen05.mma (SS form, both operands MN-major) per tile
//   warps 2-5   x  -> B operand stage;  warps 6-9   dy -> A operand stage;  all eight: the bin epilogue
#include "wbmm_tc_dev.cuh"

#include <cuda.h>

#include <cstring>
#include <mutex>

namespace wbmm {

using namespace tcdev;

namespace {

constexpr int kThreadsD = 320;

template <int WS>
struct DtCfg {
    using Cf = WinCfg<WS>;
    static constexpr int MT = (Cf::N + 127) / 128;     // M tiles of 128 output positions
    static constexpr int NV = (Cf::N + 7) / 8;         // 16-byte vectors a window fills
    static constexpr int NVEC = Cf::N_PAD / 8;         // vectors per operand region
    // The stage is two HALVES of 64 windows (K = 64 each): the repack of one half overlaps the MMAs of the other.
    static constexpr int HW = 64;                      // windows per half
    static constexpr int SBO = HW * 16;                // bytes between position groups (64 windows x 16 B)
    static constexpr int LBO = 128;                    // bytes between groups of 8 windows
    static constexpr int OP_BYTES = NVEC * SBO;        // one operand of one half
    static constexpr int HALF = 2 * OP_BYTES;          // A region then B region; an M-tile's 16 vectors may run into B
    static constexpr int STAGE = 2 * HALF;
    static constexpr int BAR_BYTES = (2 * kMaxSlots + 8) * 8;   // slots + STAGE_FULL[2] + STAGE_EMPTY[2]
    static constexpr int FIXED = (STAGE + BAR_BYTES + 127) / 128 * 128;   // tensor-map boxes land 128-byte aligned
    // Bin fold: a warp's private bins have row pitch BP = WS (mod 32), so the 32 consecutive rows of S a warp
    // updates in one step (bin = ri*BP + ci + const) fall into 32 different banks.
    static constexpr int BP = ((Cf::TW - WS + 31) / 32) * 32 + WS;
    static constexpr int BN = Cf::TW * BP;             // floats per private copy
    static_assert(BP >= Cf::TW && BP % 32 == WS % 32, "bin pitch");
    static_assert(MT * 16 <= 2 * NVEC, "an A M-tile must stay inside the stage");
    // Hierarchical variant: a second set of bins for the (w/2)-window table (row pitch WS: 2*(WS/2)-1 < WS).
    static constexpr int WL = WS / 2, LTW = 2 * WL - 1, LP = WS, LBN = LTW * LP, LNB = LTW * LTW;
    static_assert(8 * (BN + LBN) * 4 <= STAGE, "per-warp bin copies alias the stage");
};

// HIER: S is folded a second time, onto the bins of the local (w/2 x w/2) sub-window table -- only pairs
// (i, j) inside the same sub-window count (Eq. 9: diag_blocks(M_l)).
// STRIP (with GEN): general addressing on strips of window rows held in ROLLED row order (shifted / ragged maps
// whose whole frame images do not fit, or with more than 128 windows per image): the producer moves a strip as up
// to two runs of image rows, so rows never wrap inside the frame and only the columns do (as in tc_bulk_kernel).
// CTAs per SM: two at w = 7 (S is 64 TMEM columns, the operand stage 32 KB, <= 96 registers): the repack / MMA /
// fold latencies of one CTA are hidden by the other's, as in the forward kernel (wbmm_tc.cu).  w = 14 keeps S in
// 416 of the 512 columns: one CTA.
template <int WS>
constexpr int dt_ctas_per_sm() { return WS == 7 ? 2 : 1; }
template <int WS>
constexpr int dt_tmem_cols() { return DtCfg<WS>::MT * 256 <= 256 && WinCfg<WS>::N_PAD <= 128 ? 128 : 512; }

template <int WS, bool BF16, bool GEN, bool HIER, bool STRIP = false>
__global__ void __launch_bounds__(kThreadsD, dt_ctas_per_sm<WS>())
tc_dt_kernel(Geom g, TcTiles tl, TilePart part_, int nslot, const uint16_t* __restrict__ x,
             const uint16_t* __restrict__ dy, float* __restrict__ dT, float* __restrict__ dTl, int box, int pbox,
             const __grid_constant__ CUtensorMap mx, const __grid_constant__ CUtensorMap mg)
{
    using Cf = WinCfg<WS>;
    using Dc = DtCfg<WS>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* stage = smem;                                   // A (dy) region, then B (x) region
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Dc::STAGE);
    uint8_t* ring = smem + Dc::FIXED;
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t bar0 = ptx::smem_u32(bars);
    auto FULL = [&](int s) { return bar0 + 8u * s; };
    auto EMPTY = [&](int s) { return bar0 + 8u * (kMaxSlots + s); };
    const uint32_t STAGE_FULL = bar0 + 8u * (2 * kMaxSlots), STAGE_EMPTY = STAGE_FULL + 16;   // [2 halves] each
    const int wpf = tl.NSY * g.nww;

    if (warp == 1) ptx::tmem_alloc(ptx::smem_u32(&tmem_base_s), dt_tmem_cols<WS>());
    if (tid >= 64 && tid < 64 + nslot) {
        ptx::mbar_init(FULL(tid - 64), 1);
        ptx::mbar_init(EMPTY(tid - 64), box ? box * wpf : wpf);   // box mode: one barrier pair per group of `box` images
        ptx::fence_mbar_init();
    }
    if (tid == 0) {
        for (int hf = 0; hf < 2; ++hf) {
            ptx::mbar_init(STAGE_FULL + 8 * hf, 2 * Dc::HW);      // 64 windows x (x, dy)
            ptx::mbar_init(STAGE_EMPTY + 8 * hf, 1);
        }
        ptx::fence_mbar_init();
    }
    // vectors a window never writes (padding positions) must read as zero / finite
    for (int i = tid; i < Dc::STAGE / 16; i += kThreadsD) reinterpret_cast<uint4*>(stage)[i] = make_uint4(0, 0, 0, 0);
    ptx::fence_proxy_async_smem();
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::tc_fence_after_sync();
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const uint32_t tmem = tmem_base_s;

    const int t0 = part_.start[blockIdx.x], t1 = part_.start[blockIdx.x + 1];
    const int rowB = g.W * 2;
    const long long plane_elems = (long long)g.H * g.W;
    const bool ragged = g.H != g.Hp || g.W != g.Wp;
    const bool flat7 = WS == 7 && !GEN && pbox && g.W == WS && g.H == WS;      // 7 x 7 maps: the plane is the window (wbmm_tc_dev.cuh)

    auto tile_decode = [&](int t, int& c, int& b0, int& wy0, int& np_eff, int& rows_eff) {
        c = t / tl.tiles_per_c;
        const int rem = t - c * tl.tiles_per_c;
        const int gb = rem / tl.nstrips, strip = rem - gb * tl.nstrips;
        b0 = gb * tl.NP;
        wy0 = strip * tl.NSY;
        np_eff = min(tl.NP, g.B - b0);
        rows_eff = GEN ? (!STRIP ? g.H : min(tl.frame_rows, g.Hp - wy0 * WS)) : min(tl.frame_rows, g.H - wy0 * WS);
    };

    if (warp == 0) {
        // ------------------------------------------------------------------ producer
        // ring order per tile: x image 0, dy image 0, x image 1, dy image 1, ...
        uint32_t k = 0;
        for (int t = t0; t < t1; ++t) {
            int c, b0, wy0, np_eff, rows_eff;
            tile_decode(t, c, b0, wy0, np_eff, rows_eff);
            // pbox ("plane boxes", wbmm_tc.cu): the maps are over [B][C*H*W], inner coordinate c*H*W, slot pitch tl.S
            const uint32_t bytes = pbox ? (uint32_t)tl.S : (uint32_t)rows_eff * rowB;
            if (box) {
                // small images: one tensor-map box per group of `box` images and operand; ring order per tile:
                // x group 0, dy group 0, x group 1, dy group 1, ...
                for (int j = lane; j < 2 * np_eff / box; j += 32) {
                    const uint32_t kk = k + j * box;
                    const int slot = kk % nslot;
                    ptx::mbar_wait(EMPTY(slot), ((kk / nslot) & 1) ^ 1);
                    ptx::mbar_arrive_expect_tx(FULL(slot), bytes * box);
                    const int pe0 = c * (int)plane_elems;
                    ptx::tma_load_4d(ptx::smem_u32(ring + (size_t)slot * tl.S), (j & 1) ? &mg : &mx, pbox ? (plane_box_2d(plane_elems) ? 0 : pe0 & ~7) : 0,
                                     pbox && plane_box_2d(plane_elems) ? pe0 >> 3 : 0, pbox ? 0 : c, b0 + (j >> 1) * box, FULL(slot));
                }
            } else if constexpr (STRIP) {
                // The strip's rolled rows are up to two runs of image rows (none when it lies in the padding: the barrier
                // then completes on the arrival alone).  One bulk copy per lane and pass: run A with the byte count of
                // both runs, then run B.  (Two copies issued by the same lane inside one divergent loop body lost copies
                // as soon as four lanes were active -- the reason the first strip variant of this kernel hung.)
                const StripRuns sr = strip_runs(g, wy0 * WS, rows_eff);
                for (int j = lane; j < 2 * np_eff; j += 32) {
                    const uint32_t kk = k + j;
                    const int slot = kk % nslot;
                    ptx::mbar_wait(EMPTY(slot), ((kk / nslot) & 1) ^ 1);
                    const uint16_t* pl0 = ((j & 1) ? dy : x) + ((long long)(b0 + (j >> 1)) * g.C + c) * plane_elems;
                    ptx::mbar_arrive_expect_tx(FULL(slot), (uint32_t)(sr.nA + sr.nB) * rowB);
                    if (sr.nA > 0)
                        ptx::bulk_g2s(ptx::smem_u32(ring + (size_t)slot * tl.S), pl0 + (long long)sr.a0 * g.W, (uint32_t)sr.nA * rowB, FULL(slot));
                }
                __syncwarp();
                if (sr.nB > 0)
                    for (int j = lane; j < 2 * np_eff; j += 32) {
                        const uint32_t kk = k + j;
                        const int slot = kk % nslot;
                        const uint16_t* pl0 = ((j & 1) ? dy : x) + ((long long)(b0 + (j >> 1)) * g.C + c) * plane_elems;
                        ptx::bulk_g2s(ptx::smem_u32(ring + (size_t)slot * tl.S) + sr.n1 * rowB, pl0, (uint32_t)sr.nB * rowB, FULL(slot));
                    }
            } else
            for (int j = lane; j < 2 * np_eff; j += 32) {
                const uint32_t kk = k + j;
                const int slot = kk % nslot;
                const int p = j >> 1;
                ptx::mbar_wait(EMPTY(slot), ((kk / nslot) & 1) ^ 1);
                ptx::mbar_arrive_expect_tx(FULL(slot), bytes);
                const uint16_t* src = ((j & 1) ? dy : x) + ((long long)(b0 + p) * g.C + c) * plane_elems +
                                      (long long)wy0 * WS * g.W;
                ptx::bulk_g2s(ptx::smem_u32(ring + (size_t)slot * tl.S), src, bytes, FULL(slot));
            }
            k += 2 * np_eff;
            __syncwarp();   // no lane starts the next tile's copies before every copy of this tile is issued (see the repack warps)
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer
        if (lane == 0) {
            constexpr uint32_t idesc = ptx::idesc_f16(BF16 ? 1 : 0, 128, Cf::N_PAD) | (1u << 15) | (1u << 16);   // A, B MN-major
            const uint32_t stage_addr = ptx::smem_u32(stage);
            uint32_t lt = 0;
            int cur_c = -1;
            for (int t = t0; t < t1; ++t, ++lt) {
                const int c = t / tl.tiles_per_c;
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    const uint32_t a_addr = stage_addr + hf * Dc::HALF, b_addr = a_addr + Dc::OP_BYTES;
                    ptx::mbar_wait(STAGE_FULL + 8 * hf, lt & 1);
                    ptx::tc_fence_after_sync();
#pragma unroll
                    for (int mt = 0; mt < Dc::MT; ++mt) {
#pragma unroll
                        for (int ks = 0; ks < Dc::HW / 16; ++ks) {
                            const uint64_t ad = ptx::smem_desc_kmajor_noswz(a_addr + mt * 16 * Dc::SBO + ks * 2 * Dc::LBO, Dc::LBO, Dc::SBO);
                            const uint64_t bd = ptx::smem_desc_kmajor_noswz(b_addr + ks * 2 * Dc::LBO, Dc::LBO, Dc::SBO);
                            ptx::mma_ss(tmem + mt * 256, ad, bd, idesc, (c != cur_c && hf == 0 && ks == 0) ? 0u : 1u);
                        }
                    }
                    ptx::mma_commit(STAGE_EMPTY + 8 * hf);
                }
                cur_c = c;
            }
        }
    } else {
        // ------------------------------------------------------------------ operand repack + bin epilogue
        const int ot = tid - 64;            // 0..255
        const int o = ot >> 7;              // 0: x -> B region, 1: dy -> A region
        const int m = ot & 127;             // window of the tile = MMA K index (image-major)
        const int pl = m / wpf, wl = m - pl * wpf;
        const int wyl = wl / g.nww, wx = wl - wyl * g.nww;
        const int win_off = ((wyl * WS) * g.W + wx * WS) * 2;
        const int hf = m >> 6;                                   // half of the stage this window goes to
        uint8_t* dst = stage + hf * Dc::HALF + (o ? 0 : Dc::OP_BYTES) + (m & 63) * 16;
        constexpr bool WG = GEN || (WS % 2 == 1);   // word-granular window addressing (GenAddr)
        GenAddr<WG ? WS : 1> ga;
        if constexpr (STRIP) gen_addr_init_strip<WS>(ga, g, wyl, wx);
        else if constexpr (GEN) gen_addr_init<WS>(ga, g, wyl, wx);
        else if constexpr (WG) gen_addr_init_plain<WS>(ga, g.W, wyl, wx);
        float* bins = reinterpret_cast<float*>(stage);
        float* bw = bins + (ot >> 5) * Dc::BN;          // this warp's private copy of the bins
        const int ew = ot >> 5;                          // 0..7
        const int emt = ew >> 2, eq = warp & 3;          // M-tile and TMEM lane quarter in the epilogue
        const int erow = emt * 128 + eq * 32 + lane;     // row of S = output position i
        const int eri = erow / WS, eci = erow - eri * WS;
        float* lw = bins + 8 * Dc::BN + (ot >> 5) * Dc::LBN;   // HIER: this warp's private local-table bins
        const int erh = eri / Dc::WL, ech = eci / Dc::WL;      // HIER: sub-window of output position i
        uint32_t k = 0, lt = 0;
        for (int t = t0; t < t1; ++t, ++lt) {
            int c, b0, wy0, np_eff, rows_eff;
            tile_decode(t, c, b0, wy0, np_eff, rows_eff);
            // Slot barriers are tested by phase PARITY, and successive fills of one slot are consumed by
            // different threads: a thread may only test fill n once fill n-1 is known to have landed.
            // After this barrier every repack thread has passed its waits of the previous tile, and a
            // slot's previous fill always belongs to an earlier tile (nslot > copies per tile).
            ptx::named_bar_sync(1, 256);
            const bool part = pl < tl.NP && pl < np_eff;
            const bool valid = part && wy0 + wyl < g.nwh;
            if constexpr (STRIP) {
                if (ragged) ga.rowmask = gen_strip_rowmask<WS>(g, wy0 + wyl);
            }
            const uint32_t kk = box ? k + 2 * box * (pl / box) + box * o + pl % box : k + 2 * pl + o;
            const int slot = kk % nslot;
            const int bslot = box ? slot - slot % box : slot;      // the barrier pair that covers this image
            if (part) ptx::mbar_wait(FULL(bslot), (kk / nslot) & 1);
            const uint8_t* img = ring + (size_t)slot * tl.S + (pbox ? ((c * (int)plane_elems) & 7) * 2 : 0);
            {
                uint32_t wv[Dc::NV * 4];
                if (WS == 7 && flat7) {
                    if constexpr (WS == 7) window_to_regs_flat7(ring + (size_t)slot * tl.S, ((c * (int)plane_elems) & 7) * 2, valid, wv);
                } else if constexpr (WG) {
                    if (GEN && ragged) window_to_regs_gen<WS, true>(img, ga, valid, wv);
                    else window_to_regs_gen<WS, false>(img, ga, valid, wv);
                } else {
                    window_to_regs<WS>(valid ? img + win_off : img, valid, rowB, wv);
                    if (WS % 2 == 0 && !valid) {
#pragma unroll
                        for (int e = 0; e < Cf::NW; ++e) wv[e] = 0u;
                    }
                }
#pragma unroll
                for (int e = Cf::NW; e < Dc::NV * 4; ++e) wv[e] = 0u;
                // The window is in registers: its frame image can be refilled, and only the vector stores below have to
                // wait for the MMAs of the previous tile -- the frame reads (the larger part of the repack) overlap them.
                if (part) ptx::mbar_arrive(EMPTY(bslot));
                ptx::mbar_wait(STAGE_EMPTY + 8 * hf, (lt & 1) ^ 1);      // the MMAs of tile lt-1 have read this half
#pragma unroll
                for (int v = 0; v < Dc::NV; ++v)
                    *reinterpret_cast<uint4*>(dst + v * Dc::SBO) = make_uint4(wv[4 * v], wv[4 * v + 1], wv[4 * v + 2], wv[4 * v + 3]);
            }
            ptx::fence_proxy_async_smem();
            ptx::mbar_arrive(STAGE_FULL + 8 * hf);
            k += 2 * np_eff;

            const bool seg_end = t + 1 == t1 || (t + 1) - c * tl.tiles_per_c == tl.tiles_per_c;
            if (seg_end) {
                // ---- S (TMEM) -> bins -> dT[c]
                ptx::mbar_wait(STAGE_EMPTY, lt & 1);        // every MMA of this channel segment has completed
                ptx::mbar_wait(STAGE_EMPTY + 8, lt & 1);
                ptx::tc_fence_after_sync();
                for (int b = lane; b < Dc::BN; b += 32) bw[b] = 0.f;
                if constexpr (HIER)
                    for (int b = lane; b < Dc::LBN; b += 32) lw[b] = 0.f;
                __syncwarp();
                if (emt < Dc::MT) {
                    // Row i = erow of S goes to bins base - rj*TW - cj.  For a fixed column j the 32 rows of
                    // the warp hit 32 different bins; input rows rj and rj + RJ_STRIDE are RJ_STRIDE*w > 31
                    // rows of S apart in bin space, so their updates are independent too: NU read-add-write
                    // chains are in flight per step instead of one.
                    const uint32_t taddr = tmem + emt * 256 + ((uint32_t)(eq * 32) << 16);
                    float* bbase = bw + (eri + WS - 1) * Dc::BP + eci + WS - 1;
                    const bool rowok = erow < Cf::N;
                    float* lbase = lw + (eri + Dc::WL - 1) * Dc::LP + eci + Dc::WL - 1;
                    constexpr int RJ_STRIDE = 31 / WS + 1, NU = (WS + RJ_STRIDE - 1) / RJ_STRIDE;
#pragma unroll
                    for (int g0 = 0; g0 < RJ_STRIDE; ++g0) {
                        // rows rj = g0, g0 + RJ_STRIDE, ... of one pass: NU independent chains
                        uint32_t v[NU][WS];
#pragma unroll
                        for (int u = 0; u < NU; ++u)
                            if (g0 + u * RJ_STRIDE < WS) ptx::tmem_ld_n<WS>(taddr + (g0 + u * RJ_STRIDE) * WS, v[u]);
                        ptx::tmem_wait_ld();
#pragma unroll
                        for (int cj = 0; cj < WS; ++cj) {
                            float old[NU];
#pragma unroll
                            for (int u = 0; u < NU; ++u)
                                if (g0 + u * RJ_STRIDE < WS && rowok) old[u] = bbase[-(g0 + u * RJ_STRIDE) * Dc::BP - cj];
#pragma unroll
                            for (int u = 0; u < NU; ++u)
                                if (g0 + u * RJ_STRIDE < WS && rowok)
                                    bbase[-(g0 + u * RJ_STRIDE) * Dc::BP - cj] = old[u] + __uint_as_float(v[u][cj]);
                            __syncwarp();
                            if constexpr (HIER) {
                                // same S element, local bin (ri - rj + w/2 - 1, ci - cj + w/2 - 1), if j is in i's sub-window
                                const bool colok = rowok && ech == cj / Dc::WL;
#pragma unroll
                                for (int u = 0; u < NU; ++u)
                                    if (g0 + u * RJ_STRIDE < WS && colok && erh == (g0 + u * RJ_STRIDE) / Dc::WL)
                                        old[u] = lbase[-(g0 + u * RJ_STRIDE) * Dc::LP - cj];
#pragma unroll
                                for (int u = 0; u < NU; ++u)
                                    if (g0 + u * RJ_STRIDE < WS && colok && erh == (g0 + u * RJ_STRIDE) / Dc::WL)
                                        lbase[-(g0 + u * RJ_STRIDE) * Dc::LP - cj] = old[u] + __uint_as_float(v[u][cj]);
                                __syncwarp();
                            }
                        }
                    }
                }
                ptx::tc_fence_before_sync();
                ptx::named_bar_sync(1, 256);
                for (int b = ot; b < Cf::NB; b += 256) {
                    float sacc = 0.f;
                    const int bp = (b / Cf::TW) * Dc::BP + b % Cf::TW;
#pragma unroll
                    for (int w8 = 0; w8 < 8; ++w8) sacc += bins[w8 * Dc::BN + bp];
                    atomicAdd(dT + (long long)c * Cf::NB + b, sacc);
                }
                if constexpr (HIER) {
                    const float* lbins = bins + 8 * Dc::BN;
                    for (int b = ot; b < Dc::LNB; b += 256) {
                        float sacc = 0.f;
                        const int bp = (b / Dc::LTW) * Dc::LP + b % Dc::LTW;
#pragma unroll
                        for (int w8 = 0; w8 < 8; ++w8) sacc += lbins[w8 * Dc::LBN + bp];
                        atomicAdd(dTl + (long long)c * Dc::LNB + b, sacc);
                    }
                }
                ptx::named_bar_sync(1, 256);
                // the bins aliased the operand stage: restore the zero padding vectors
                for (int i = ot; i < 8 * (Dc::BN + Dc::LBN) * 4 / 16 + 1; i += 256)
                    if (i * 16 < Dc::STAGE) reinterpret_cast<uint4*>(stage)[i] = make_uint4(0, 0, 0, 0);
                ptx::fence_proxy_async_smem();
                ptx::named_bar_sync(1, 256);
            }
        }
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem, dt_tmem_cols<WS>());
}

template <int WS>
int dt_slots(const TcTiles& tl, int ctas = 1)
{
    const long long room = (ctas == 1 ? 227ll * 1024 : 113ll * 1024) - 1024 - DtCfg<WS>::FIXED;
    long long n = room / tl.S;
    if (n > 6 * tl.NP) n = 6 * tl.NP;
    if (n > kMaxSlots) n = kMaxSlots;
    return (int)n;
}

// 0 = not servable, 1 = aligned form, 2 = general form (shift / ragged)
template <int WS>
int dt_mode(const Geom& g, const TcTiles& tl, const void* x, const void* dy)
{
    if (g.layout != WBMM_LAYOUT_NCHW) return 0;
    const bool pb = ((long long)g.H * g.W * 2) % 16 != 0;       // plane boxes (wbmm_tc.cu), 8, 4 or 2 images per box
    if (pb && plane_box_images(g, tl) == 0) return 0;      // (odd planes: 7 x 7 at w = 7 only -- the flat form)
    if (reinterpret_cast<uintptr_t>(x) % 16 != 0 || reinterpret_cast<uintptr_t>(dy) % 16 != 0) return 0;
    if (tl.ntiles > 0x3fffffffll) return 0;
    if (dt_slots<WS>(tl) < 2 * tl.NP + 1) return 0;
    const bool plain = g.sh == 0 && g.sw == 0 && g.H == g.Hp && g.W == g.Wp;
    if (plain && (pb || (tl.frame_rows * g.W * 2) % 16 == 0) && (WS % 2 == 0 || g.W % 2 == 0 || (pb && g.H == WS && g.W == WS))) return 1;   // odd w: rows must be word-aligned (7 x 7 maps: flat form)
    // general form: whole images in natural layout, word-granular window addressing (W, W' even)
    // (an odd W' -- ragged maps at odd w -- is fine without a column shift: nothing wraps)
    // strips of window rows (maps with more than 128 windows per image, or whose whole images do not fit): rolled-order
    // frames loaded as runs of whole image rows -- rows of 16-byte multiples
    return ((tl.nstrips == 1 || (g.W * 2) % 16 == 0) && g.W % 2 == 0 && (g.Wp % 2 == 0 || g.sw == 0)) ? 2 : 0;
}

// Tiling of the table-gradient kernel.  Its ring holds x AND dy and shares the SM with the 106 KB operand stage,
// so whole frame images of large maps (112 x 112: 25 KB) do not fit 2 * NP + 1 times.  Window-multiple, unshifted
// maps can be cut into strips of window rows instead (the aligned form reads any whole rows): more images per
// tile, fewer rows per image, frame images of ~6 KB as on the 56 x 56 maps.
template <int WS>
bool dt_tiles(const Geom& g, TcTiles* t)
{
    if (!tc_tiles(g, t)) return false;
    const bool plain = g.sh == 0 && g.sw == 0 && g.H == g.Hp && g.W == g.Wp;
    const bool strip_ok = plain || (g.W * 2) % 16 == 0;     // general form on strips: runs of whole image rows
    if (dt_slots<WS>(*t) >= 2 * t->NP + 1) return true;
    auto fewer_images = [&]() {
        // whole images (general addressing without row runs), and tiny maps with more images per tile than the ring has
        // slots for x and dy: fewer images per tile; the windows a tile then lacks are zero columns of the contraction
        TcTiles c = *t;
        while (c.NP > 1 && dt_slots<WS>(c) < 2 * c.NP + 1) c.NP /= 2;
        c.ngb = (g.B + c.NP - 1) / c.NP;
        c.tiles_per_c = c.ngb * c.nstrips;
        c.ntiles = (long long)g.C * c.tiles_per_c;
        if (dt_slots<WS>(c) >= 2 * c.NP + 1) *t = c;
    };
    if (!strip_ok || (t->nstrips == 1 && t->S <= 8192)) {
        if (t->nstrips == 1) fewer_images();
        return true;
    }
    for (int nsy = t->NSY - 1; nsy >= 1; --nsy) {
        // aligned form: whole strips of a window-multiple map, as one copy; general form: any strip, row by row runs
        if (plain && (g.nwh % nsy != 0 || (nsy * g.w * g.W * 2) % 16 != 0)) continue;
        TcTiles c = *t;
        c.NSY = nsy;
        c.NP = 128 / (nsy * g.nww);
        if (c.NP > g.B) c.NP = g.B;
        if (c.NP < 1) continue;
        c.nstrips = (g.nwh + nsy - 1) / nsy;
        c.ngb = (g.B + c.NP - 1) / c.NP;
        c.tiles_per_c = c.ngb * c.nstrips;
        c.frame_rows = nsy * g.w;
        int s16 = (c.frame_rows * g.Wp * 2 + 15) / 16;
        if (s16 % 2 == 0) ++s16;
        c.S = s16 * 16;
        c.ntiles = (long long)g.C * c.tiles_per_c;
        if (c.S <= 8192 && dt_slots<WS>(c) >= 2 * c.NP + 1) {
            *t = c;
            return true;
        }
    }
    if (!plain && t->nstrips == 1) fewer_images();
    return true;    // nothing fits: dt_mode() rejects the original tiling
}

template <int WS, bool BF16, bool GEN, bool HIER = false, bool STRIP = false>
cudaError_t launch_dt(const Geom& g, const TcTiles& tl_in, const void* x, const void* dy, float* dT, cudaStream_t s,
                      float* dTl = nullptr)
{
    auto k = tc_dt_kernel<WS, BF16, GEN, HIER, STRIP>;
    TcTiles tl = tl_in;
    CUtensorMap mx, mg;
    memset(&mx, 0, sizeof(mx));
    memset(&mg, 0, sizeof(mg));
    // small frame images: tensor-map boxes of 8 images per copy (see bulk_box_mode in wbmm_tc.cu)
    int box = 0, pbox = 0;
    if (((long long)g.H * g.W * 2) % 16 != 0) {
        const int dtype = BF16 ? WBMM_DTYPE_BF16 : WBMM_DTYPE_F16;
        box = plane_box_images(g, tl);
        if (box == 0 || !plane_box_map(g, dtype, x, box, &mx) || !plane_box_map(g, dtype, dy, box, &mg))
            return cudaErrorInvalidConfiguration;
        pbox = 1;
        tl.S = (int)(((long long)g.H * g.W + 14) / 8 * 8 * 2);
    } else {
        const long long ib = (long long)g.H * g.W * 2;
        const int dtype = BF16 ? WBMM_DTYPE_BF16 : WBMM_DTYPE_F16;
        if (tl.nstrips == 1 && ib <= 4096 && tl.NP % 8 == 0 && g.B % 8 == 0 && (8 * ib) % 128 == 0 &&
            image_box_map(g, dtype, x, 8, &mx) && image_box_map(g, dtype, dy, 8, &mg)) {
            box = 8;
            tl.S = (int)ib;
        }
    }
    // two CTAs per SM (w = 7) when half the shared memory still holds a tile and a half of x and dy
    int ctas = dt_ctas_per_sm<WS>();
    if (ctas > 1) {
        int n2 = dt_slots<WS>(tl, ctas);
        if (box) n2 -= n2 % (2 * box);
        if (n2 < 3 * tl.NP) ctas = 1;
    }
    int nslot = dt_slots<WS>(tl, ctas);
    if (box) {
        nslot -= nslot % (2 * box);
        if (nslot < 2 * tl.NP) {
            if (pbox) return cudaErrorInvalidConfiguration;
            box = 0;
            tl = tl_in;
            ctas = 1;
            nslot = dt_slots<WS>(tl);
        }
    }
    const size_t smem = (size_t)DtCfg<WS>::FIXED + (size_t)nslot * tl.S;
    static SmemOptIn smem_state;
    cudaError_t e = ensure_dynamic_smem(reinterpret_cast<const void*>(k), smem, &smem_state);
    if (e != cudaSuccess) return e;
    int grid = (int)(tl.ntiles < (long long)num_sms() * ctas ? tl.ntiles : (long long)num_sms() * ctas);
    if (grid > kMaxGrid) grid = kMaxGrid;
    static std::mutex mu;
    static TilePart cached;
    static long long key_n = -1;
    static int key_tpc = -1, key_grid = -1, cached_used = 0;
    TilePart part;
    {
        std::lock_guard<std::mutex> lock(mu);
        if (key_n != tl.ntiles || key_tpc != tl.tiles_per_c || key_grid != grid) {
            cached_used = partition_tiles(tl, grid, 1.5, &cached);   // a channel boundary costs one bin fold (~1.5 tiles)
            key_n = tl.ntiles; key_tpc = tl.tiles_per_c; key_grid = grid;
        }
        part = cached;
        grid = cached_used;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(kThreadsD);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k, g, tl, part, nslot, (const uint16_t*)x, (const uint16_t*)dy, dT, dTl, box, pbox, mx, mg);
}

}  // namespace

bool tc_grad_table_supported(const Geom& g, int dtype, const void* x, const void* dy)
{
    if (dtype != WBMM_DTYPE_BF16 && dtype != WBMM_DTYPE_F16) return false;
    if (g.w != 7 && g.w != 14) return false;
    TcTiles tl;
    if (!(g.w == 7 ? dt_tiles<7>(g, &tl) : dt_tiles<14>(g, &tl))) return false;
    return (g.w == 7 ? dt_mode<7>(g, tl, x, dy) : dt_mode<14>(g, tl, x, dy)) != 0;
}

cudaError_t tc_grad_table(const Geom& g, int dtype, const void* x, const void* dy, float* dT, cudaStream_t stream,
                          int* launches, int* path, float* dTl)
{
    TcTiles tl;
    if (!(g.w == 7 ? dt_tiles<7>(g, &tl) : dt_tiles<14>(g, &tl))) return cudaErrorNotSupported;
    if (tl.ntiles == 0) return cudaSuccess;
    const int mode = g.w == 7 ? dt_mode<7>(g, tl, x, dy) : dt_mode<14>(g, tl, x, dy);
    if (mode == 0) return cudaErrorNotSupported;
    if (dTl && g.w != 14) return cudaErrorNotSupported;
    *launches += 1;
    *path = WBMM_PATH_TC_TMA;
    const bool bf = dtype == WBMM_DTYPE_BF16;
    if (mode == 2 && tl.nstrips > 1) {      // general addressing on strips of window rows
        if (dTl) return bf ? launch_dt<14, true, true, true, true>(g, tl, x, dy, dT, stream, dTl)
                           : launch_dt<14, false, true, true, true>(g, tl, x, dy, dT, stream, dTl);
        if (g.w == 7) return bf ? launch_dt<7, true, true, false, true>(g, tl, x, dy, dT, stream)
                                : launch_dt<7, false, true, false, true>(g, tl, x, dy, dT, stream);
        return bf ? launch_dt<14, true, true, false, true>(g, tl, x, dy, dT, stream)
                  : launch_dt<14, false, true, false, true>(g, tl, x, dy, dT, stream);
    }
    if (dTl) {
        // hierarchical: both table gradients from one pass over (x, dy)
        if (mode == 2) return bf ? launch_dt<14, true, true, true>(g, tl, x, dy, dT, stream, dTl)
                                 : launch_dt<14, false, true, true>(g, tl, x, dy, dT, stream, dTl);
        return bf ? launch_dt<14, true, false, true>(g, tl, x, dy, dT, stream, dTl)
                  : launch_dt<14, false, false, true>(g, tl, x, dy, dT, stream, dTl);
    }
    const int sel = (g.w == 7 ? 0 : 4) + (bf ? 2 : 0) + (mode == 2 ? 1 : 0);
    switch (sel) {
    case 0: return launch_dt<7, false, false>(g, tl, x, dy, dT, stream);
    case 1: return launch_dt<7, false, true>(g, tl, x, dy, dT, stream);
    case 2: return launch_dt<7, true, false>(g, tl, x, dy, dT, stream);
    case 3: return launch_dt<7, true, true>(g, tl, x, dy, dT, stream);
    case 4: return launch_dt<14, false, false>(g, tl, x, dy, dT, stream);
    case 5: return launch_dt<14, false, true>(g, tl, x, dy, dT, stream);
    case 6: return launch_dt<14, true, false>(g, tl, x, dy, dT, stream);
    default: return launch_dt<14, true, true>(g, tl, x, dy, dT, stream);
    }
}




}  // namespace wbmm

#ifdef WBMM_WATCHDOG
// debug build only (wbmm_debug.cuh): the waiters this translation unit's kernels gave up on
extern "C" __attribute__((visibility("default"))) int wbmm_debug_watchdog_dt(unsigned long long* out)
{
    return (int)cudaMemcpyFromSymbol(out, wbmm::ptx::g_watchdog, sizeof(unsigned long long) * 64);
}
#endif
