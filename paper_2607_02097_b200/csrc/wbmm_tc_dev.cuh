// Device-side building blocks shared by the tensor-core WBMM kernels (forward/dX in wbmm_tc.cu,
// table gradient in wbmm_tc_dt.cu): window geometry constants, window <-> frame addressing,
// TMEM transfer helpers, the static tile schedule.  Not part of the C ABI.
#pragma once

#include "wbmm_ptx.cuh"
#include "wbmm_tc.cuh"

namespace wbmm {
namespace tcdev {

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
// without a window write zeros (odd w) or whatever finite-or-not bytes `win` points at (even w:
// unconditional loads -- the caller passes a legal address; row m of D depends on row m of A
// only, and rows of lanes without a window are never stored).
template <int WS>
__device__ __forceinline__ void window_to_tmem(const uint8_t* win, bool valid, int rowB, uint32_t taddr)
{
    using Cf = WinCfg<WS>;
    if constexpr (WS % 2 == 0) {
        // a window row is WS/2 aligned 32-bit words: one running row pointer, immediate offsets
        constexpr int WPR = WS / 2;
        uint32_t v[(Cf::A_COLS + 15) / 16 * 16];
        const uint8_t* p = win;
#pragma unroll
        for (int r = 0; r < WS; ++r) {
#pragma unroll
            for (int k = 0; k < WPR; ++k) v[r * WPR + k] = *reinterpret_cast<const uint32_t*>(p + 4 * k);
            p += rowB;
        }
#pragma unroll
        for (int k = Cf::NW; k < (Cf::A_COLS + 15) / 16 * 16; ++k) v[k] = 0u;
#pragma unroll
        for (int ch = 0; ch < Cf::A_COLS / 16; ++ch) ptx::tmem_st16(taddr + ch * 16, v + ch * 16);
        if constexpr (Cf::A_COLS % 16 != 0) ptx::tmem_st8(taddr + (Cf::A_COLS / 16) * 16, v + (Cf::A_COLS / 16) * 16);
        ptx::tmem_wait_st();
        return;
    }
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

// TMEM D -> rounded 16-bit values in the window's frame position (32 columns per wait).
template <int WS, bool BF16>
__device__ __forceinline__ void tmem_to_window(uint8_t* win, bool valid, int rowB, uint32_t taddr)
{
    using Cf = WinCfg<WS>;
    constexpr int NCH = (Cf::NW + 7) / 8;     // 16-column chunks that hold real outputs
#pragma unroll
    for (int ch = 0; ch < NCH; ch += 2) {
        uint32_t v[32];
        ptx::tmem_ld16(taddr + ch * 16, v);
        if (ch + 1 < NCH) ptx::tmem_ld16(taddr + (ch + 1) * 16, v + 16);
        ptx::tmem_wait_ld();
        if (valid) {
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                const int wi = ch * 8 + e;
                if (wi < Cf::NW && (e < 8 || ch + 1 < NCH))
                    store_word<WS>(win, rowB, wi, pack2<BF16>(v[2 * e], v[2 * e + 1]));
            }
        }
    }
}

// The accumulator is drained in NH column ranges ("halves") so that the epilogue of one half
// overlaps the MMAs of the other: w = 14 splits after output row 8 (112 | 84 positions), w = 7
// is one range.  HalfCfg<WS, h>: first column, MMA N of the half, packed-word range.
template <int WS>
struct HalfSplit {
    using Cf = WinCfg<WS>;
    static constexpr int NH = (WS == 14) ? 2 : 1;
    static constexpr int N0 = (WS == 14) ? 112 : Cf::N_PAD;                 // columns of half 0 (multiple of 16)
    static constexpr int col0(int h) { return h == 0 ? 0 : N0; }
    static constexpr int ncols(int h) { return h == 0 ? N0 : Cf::N_PAD - N0; }
    static constexpr int word0(int h) { return col0(h) / 2; }
    static constexpr int word1(int h) { return (col0(h) + ncols(h)) / 2 < Cf::NW ? (col0(h) + ncols(h)) / 2 : Cf::NW; }
    static_assert(N0 % 16 == 0 && (Cf::N_PAD - N0) % 16 == 0, "halves are MMA-N legal");
    static_assert(WS != 14 || N0 % (2 * WS) == 0, "the split falls on a window-row boundary");
};

// NCOLS fp32 accumulator columns (multiple of 16) -> NCOLS/2 packed 16-bit pairs (RNE).
template <bool BF16, int NCOLS>
__device__ __forceinline__ void tmem_cols_to_packed(uint32_t taddr, uint32_t* pk)
{
    static_assert(NCOLS % 16 == 0, "16-column chunks");
#pragma unroll
    for (int ch = 0; ch < NCOLS / 16; ch += 2) {
        uint32_t v[32];
        ptx::tmem_ld16(taddr + ch * 16, v);
        if (ch + 1 < NCOLS / 16) ptx::tmem_ld16(taddr + (ch + 1) * 16, v + 16);
        ptx::tmem_wait_ld();
#pragma unroll
        for (int e = 0; e < 16; ++e)
            if (e < 8 || ch + 1 < NCOLS / 16) pk[ch * 8 + e] = pack2<BF16>(v[2 * e], v[2 * e + 1]);
    }
}

// Packed words [W0, W1) of a window -> its frame position (aligned form).
template <int WS, int W0, int W1>
__device__ __forceinline__ void packed_to_window(uint8_t* win, int rowB, const uint32_t* pk)
{
    if constexpr (WS % 2 == 0) {
        constexpr int WPR = WS / 2;
        static_assert(W0 % WPR == 0, "starts on a window row");
        uint8_t* p = win + (W0 / WPR) * rowB;
#pragma unroll
        for (int wi = W0; wi < W1; ++wi) {
            *reinterpret_cast<uint32_t*>(p + 4 * (wi % WPR)) = pk[wi - W0];
            if (wi % WPR == WPR - 1) p += rowB;
        }
    } else {
#pragma unroll
        for (int wi = W0; wi < W1; ++wi) store_word<WS>(win, rowB, wi, pk[wi - W0]);
    }
}

// General window addressing for whole-image frames held exactly as they sit in global memory
// (row pitch W): the cyclic shift and the zero padding (Eq. 4-5; A6) become per-thread
// row / column byte offsets plus validity bit masks (bit r / bit cc set = inside H x W).  Offsets
// of padding rows / columns are clamped to 0 so every load address is legal; the value is masked.
template <int WS>
struct GenAddr {
    int rowoff[WS], coloff[WS];
    uint32_t rowmask, colmask;
};

template <int WS>
__device__ __forceinline__ void gen_addr_init(GenAddr<WS>& a, const Geom& g, int wyl, int wx)
{
    a.rowmask = a.colmask = 0;
#pragma unroll
    for (int r = 0; r < WS; ++r) {
        int h = wyl * WS + r + g.sh;
        if (h >= g.Hp) h -= g.Hp;
        a.rowoff[r] = h < g.H ? h * g.W * 2 : 0;
        a.rowmask |= (h < g.H ? 1u : 0u) << r;
    }
#pragma unroll
    for (int cc = 0; cc < WS; ++cc) {
        int v = wx * WS + cc + g.sw;
        if (v >= g.Wp) v -= g.Wp;
        a.coloff[cc] = v < g.W ? v * 2 : 0;
        a.colmask |= (v < g.W ? 1u : 0u) << cc;
    }
}

// RAGGED = false: every window element lies inside H x W (no padding anywhere), masks unused.
template <int WS, bool RAGGED>
__device__ __forceinline__ uint32_t gen_load_word(const uint8_t* img, const GenAddr<WS>& a, uint32_t rm, int wi)
{
    const int e0 = 2 * wi, e1 = 2 * wi + 1;
    uint32_t lo = *reinterpret_cast<const uint16_t*>(img + a.rowoff[e0 / WS] + a.coloff[e0 % WS]);
    if (RAGGED && !((rm >> (e0 / WS)) & (a.colmask >> (e0 % WS)) & 1u)) lo = 0;
    uint32_t hi = 0;
    if (e1 < WS * WS) {
        hi = *reinterpret_cast<const uint16_t*>(img + a.rowoff[e1 / WS] + a.coloff[e1 % WS]);
        if (RAGGED && !((rm >> (e1 / WS)) & (a.colmask >> (e1 % WS)) & 1u)) hi = 0;
    }
    return lo | (hi << 16);
}

template <int WS, bool RAGGED>
__device__ __forceinline__ void gen_store_word(uint8_t* img, const GenAddr<WS>& a, int wi, uint32_t v)
{
    const int e0 = 2 * wi, e1 = 2 * wi + 1;
    if (!RAGGED || ((a.rowmask >> (e0 / WS)) & (a.colmask >> (e0 % WS)) & 1u))
        *reinterpret_cast<uint16_t*>(img + a.rowoff[e0 / WS] + a.coloff[e0 % WS]) = (uint16_t)(v & 0xffffu);
    if (e1 < WS * WS) {
        if (!RAGGED || ((a.rowmask >> (e1 / WS)) & (a.colmask >> (e1 % WS)) & 1u))
            *reinterpret_cast<uint16_t*>(img + a.rowoff[e1 / WS] + a.coloff[e1 % WS]) = (uint16_t)(v >> 16);
    }
}

template <int WS, bool RAGGED>
__device__ __forceinline__ void window_to_tmem_gen_t(const uint8_t* img, const GenAddr<WS>& a, uint32_t rm, uint32_t taddr)
{
    using Cf = WinCfg<WS>;
#pragma unroll
    for (int ch = 0; ch < (Cf::A_COLS + 15) / 16; ++ch) {
        uint32_t v[16];
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            const int wi = ch * 16 + e;
            v[e] = wi < Cf::NW ? gen_load_word<WS, RAGGED>(img, a, rm, wi) : 0u;
        }
        if (ch * 16 + 16 <= Cf::A_COLS) ptx::tmem_st16(taddr + ch * 16, v);
        else ptx::tmem_st8(taddr + ch * 16, v);
    }
}

// tcgen05.st is warp-collective: every lane runs the same instruction stream; a lane without a
// window (or a ragged problem) takes the masked form, chosen warp-uniformly.
template <int WS>
__device__ __forceinline__ void window_to_tmem_gen(const uint8_t* img, const GenAddr<WS>& a, bool valid, bool ragged,
                                                   uint32_t taddr)
{
    const bool masked = ragged || !__all_sync(0xffffffffu, valid);
    if (masked) window_to_tmem_gen_t<WS, true>(img, a, valid ? a.rowmask : 0u, taddr);
    else window_to_tmem_gen_t<WS, false>(img, a, 0u, taddr);
    ptx::tmem_wait_st();
}

template <int WS, bool BF16, bool RAGGED>
__device__ __forceinline__ void tmem_to_window_gen_t(uint8_t* img, const GenAddr<WS>& a, bool valid, uint32_t taddr)
{
    using Cf = WinCfg<WS>;
    constexpr int NCH = (Cf::NW + 7) / 8;
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
        uint32_t v[16];
        ptx::tmem_ld16(taddr + ch * 16, v);
        ptx::tmem_wait_ld();
        if (valid) {
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const int wi = ch * 8 + e;
                if (wi < Cf::NW) gen_store_word<WS, RAGGED>(img, a, wi, pack2<BF16>(v[2 * e], v[2 * e + 1]));
            }
        }
    }
}

template <int WS, int W0, int W1, bool RAGGED>
__device__ __forceinline__ void packed_to_window_gen(uint8_t* img, const GenAddr<WS>& a, const uint32_t* pk)
{
#pragma unroll
    for (int wi = W0; wi < W1; ++wi) gen_store_word<WS, RAGGED>(img, a, wi, pk[wi - W0]);
}

template <int WS, bool BF16>
__device__ __forceinline__ void tmem_to_window_gen(uint8_t* img, const GenAddr<WS>& a, bool valid, bool ragged, uint32_t taddr)
{
    if (ragged) tmem_to_window_gen_t<WS, BF16, true>(img, a, valid, taddr);
    else tmem_to_window_gen_t<WS, BF16, false>(img, a, valid, taddr);
}

constexpr int kThreadsB = 352;
constexpr int kMaxSlots = 96;
constexpr int kMaxGrid = 160;
constexpr int kMaxOutBufs = 16;  // output group buffers of the bulk kernel

// Output hand-off groups of the bulk kernel: the smallest runs of whole epilogue warps that cover
// whole frame images (MMA rows are image-major), so a group's images can be stored as soon as ITS
// warps are done.  lanes per group, groups per tile, frame images per group.
struct OutGroups { int lanes, n, images; };
__host__ __device__ inline OutGroups out_groups(const TcTiles& tl, int wpf)
{
    OutGroups og;
    og.lanes = 128;
    for (int cand = 32; cand < 128; cand += cand)
        if (cand % wpf == 0) { og.lanes = cand; break; }
    og.n = 128 / og.lanes;
    og.images = og.lanes % wpf == 0 ? og.lanes / wpf : tl.NP;
    if (og.images > tl.NP) og.images = tl.NP;
    return og;
}

// Static tile schedule: CTA b owns tiles [start[b], start[b+1]) (channel-major, so W_c is rebuilt
// at most once or twice per CTA).  The host balances tiles + the cost of mid-range W_c rebuilds.
struct TilePart {
    int start[kMaxGrid + 1];
};


#ifdef WBMM_TRACE
// Debug build only: per-tile event timestamps of block 0 (read back with wbmm_debug_trace()).
__device__ long long g_trace[16 * 16];
__device__ long long g_blk[148 * 4];
__device__ __forceinline__ long long gtime() { long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define TRACE(ev, lt) do { if (blockIdx.x == 1 && (lt) < 16) g_trace[(lt) * 16 + (ev)] = gtime(); } while (0)
#else
#define TRACE(ev, lt) do { } while (0)
#endif

}  // namespace tcdev

// Host helpers defined in wbmm_tc.cu.
int num_sms();
// Greedy contiguous partition of the tile sequence over `grid` CTAs minimising the largest cost,
// cost = tiles + switch_cost per channel boundary strictly inside a CTA's range.  Returns the
// number of CTAs used.
int partition_tiles(const TcTiles& tl, int grid, double switch_cost, tcdev::TilePart* part);

}  // namespace wbmm
