// Device-side building blocks shared by the tensor-core WBMM kernels (forward/dX in wbmm_tc.cu,
// table gradient in wbmm_tc_dt.cu): window geometry constants, window <-> frame addressing,
// TMEM transfer helpers, the static tile schedule.  Not part of the C ABI.
#pragma once

#include <atomic>

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

// Aligned form: the window's N values, two per word in row-major in-window order, v[0 .. NW).
// Even w: unconditional loads through one running row pointer (the caller passes a legal address).
template <int WS>
__device__ __forceinline__ void window_to_regs(const uint8_t* win, bool valid, int rowB, uint32_t* v)
{
    using Cf = WinCfg<WS>;
    if constexpr (WS % 2 == 0) {
        constexpr int WPR = WS / 2;
        const uint8_t* p = win;
#pragma unroll
        for (int r = 0; r < WS; ++r) {
#pragma unroll
            for (int k = 0; k < WPR; ++k) v[r * WPR + k] = *reinterpret_cast<const uint32_t*>(p + 4 * k);
            p += rowB;
        }
    } else {
#pragma unroll
        for (int wi = 0; wi < Cf::NW; ++wi) v[wi] = valid ? load_word<WS>(win, rowB, wi) : 0u;
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
__device__ __forceinline__ void tmem_to_window(uint8_t* win, bool valid, int rowB, uint32_t taddr, float bias = 0.f)
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
                    store_word<WS>(win, rowB, wi, pack2<BF16>(__float_as_uint(__uint_as_float(v[2 * e]) + bias),
                                                               __float_as_uint(__uint_as_float(v[2 * e + 1]) + bias)));
            }
        }
    }
}

// W_c from a GIVEN matrix M_c[N][N] (cached-M mode) into the K-major core-matrix layout of
// build_weight: value (i, j) at byte (j/8)*LBO + i*16 + (j%8)*2; transpose: W_c = M_c^T.  Rows / columns >= N zero.
template <int WS>
__device__ __forceinline__ void load_weight(const uint16_t* __restrict__ Mc, bool transpose, uint8_t* Wc, int tid, int nthreads)
{
    using Cf = WinCfg<WS>;
    constexpr int NCHUNK = (Cf::K_PAD / 8) * Cf::N_PAD;
    constexpr int NKC = Cf::K_PAD / 8;
    for (int id = tid; id < NCHUNK; id += nthreads) {
        // neighbouring threads read neighbouring addresses: along a row of M_c, or (transposed) along a column
        const int kc = transpose ? id / Cf::N_PAD : id % NKC, i = transpose ? id % Cf::N_PAD : id / NKC;
        uint32_t pk[4] = {0u, 0u, 0u, 0u};
        if (i < Cf::N) {
            uint32_t v[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const int j = kc * 8 + e;
                v[e] = j < Cf::N ? (uint32_t)(transpose ? Mc[j * Cf::N + i] : Mc[i * Cf::N + j]) : 0u;
            }
#pragma unroll
            for (int e = 0; e < 8; ++e) pk[e >> 1] |= v[e] << ((e & 1) * 16);
        }
        *reinterpret_cast<uint4*>(Wc + kc * Cf::LBO + i * 16) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
    }
}

// Operand geometry of the bulk kernel.
//
// w = 14 ("block-Toeplitz library"): W_c[(ri,ci),(rj,cj)] = T[c, (ri-rj+w-1)(2w-1) + (ci-cj+w-1)] (Eq. 7)
// depends on the rows only through dr = ri - rj, so W_c is 14 x 14 blocks out of just 27 distinct
// 14 x 14 Toeplitz blocks Z[dr].  With every window row padded to 16 positions on both GEMM axes
// (K index = rj*16 + cj, N index = ri*16 + ci; the pads meet zero weights / are never stored), the
// B operand of K-step rj is rows (13 - rj)*16 ... of ONE 432-row array
//     lib[kc][(dr+13)*16 + ci][e] = Z[dr][ci][cj = 8*kc + e]      (K-major core matrices, 16-byte rows)
// i.e. a plain descriptor with a different start address per K-step.  13.5 KB instead of the 86.5 KB
// materialised W_c, and 864 16-byte chunks to build per channel instead of 4900.
//
// w = 7: the full K-major W_c (8 KB), as in WinCfg.
//
// The accumulator is drained in NH column ranges ("halves") so that the epilogue of one half
// overlaps the MMAs of the other.
template <int WS>
struct BulkCfg {
    using Cf = WinCfg<WS>;
    static constexpr bool TOEP = false;
    static constexpr int KSTEPS = Cf::KSTEPS;
    static constexpr int A_COLS = Cf::A_COLS;          // 32-bit TMEM columns of one A buffer
    static constexpr int D_COLS = Cf::N_PAD;
    static constexpr int WC_BYTES = Cf::WC_BYTES;
    static constexpr int LBO = Cf::LBO;
    static constexpr int NH = 1;
    static constexpr int ncols(int) { return D_COLS; }
    static constexpr int col0(int) { return 0; }
    static constexpr int word0(int) { return 0; }
    static constexpr int word1(int) { return Cf::NW; }
    // byte offset of the B operand of K-step ks, half h, inside the weight area
    static constexpr int b_off(int ks, int) { return ks * 2 * LBO; }
    static constexpr int HIER_BYTES = 0;
};

template <>
struct BulkCfg<14> {
    using Cf = WinCfg<14>;
    static constexpr bool TOEP = true;
    static constexpr int RP = 16;                      // padded window row on both GEMM axes
    static constexpr int KSTEPS = 14;                  // one input window row per tcgen05.mma (K = 16)
    static constexpr int A_COLS = 14 * RP / 2;         // 112
    static constexpr int D_COLS = 14 * RP;             // 224
    static constexpr int LIB_ROWS = 27 * RP;           // 432
    static constexpr int LBO = LIB_ROWS * 16;          // bytes between the two K chunks (cj 0-7 | 8-15)
    static constexpr int WC_BYTES = 2 * LBO;           // 13824
    static constexpr int NH = 2;                       // output rows 0-6 | 7-13
    static constexpr int ncols(int) { return 7 * RP; }
    static constexpr int col0(int h) { return h * 7 * RP; }
    static constexpr int word0(int h) { return h * 49; }
    static constexpr int word1(int h) { return (h + 1) * 49; }
    static constexpr int b_off(int ks, int h) { return ((13 - ks) * RP + h * 7 * RP) * 16; }
    // Hierarchical reparameterisation (Eq. 9): inside one half of the window rows
    // (ri/7 == rj/7) the block of the fused matrix is Z_g[dr] + Z_l'[dr], |dr| <= 6, where Z_l' holds the
    // local table on its two 7 x 7 diagonal sub-blocks: a second library of 13 blocks; the two identity
    // shortcuts are a 16 x 16 block 2*I applied by 14 extra N = 16 MMAs (kept out of the 16-bit sums).
    static constexpr int LIBA_ROWS = 13 * RP;          // 208
    static constexpr int LBO_A = LIBA_ROWS * 16;
    static constexpr int LIBA_BYTES = 2 * LBO_A;       // 6656
    static constexpr int LBO_I = RP * 16;
    static constexpr int LIBI_BYTES = 2 * LBO_I;       // 512
    static constexpr int TL_BYTES = 352;               // 13 x 13 local table, staged reversed
    static constexpr int HIER_BYTES = LIBA_BYTES + LIBI_BYTES + TL_BYTES;
    static constexpr int b_off_a(int ks, int h) { return (7 * h - ks + 6) * RP * 16; }   // valid when ks / 7 == h
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

// One half of the accumulator (BulkCfg<WS>::ncols(h) fp32 columns at taddr) -> packed 16-bit pairs
// in row-major in-window order (the 2 pad columns of every padded row are dropped for w = 14).
template <int WS, bool BF16, int H>
__device__ __forceinline__ void accum_half_to_packed(uint32_t taddr, uint32_t* pk)
{
    using Bc = BulkCfg<WS>;
    if constexpr (Bc::TOEP) {
#pragma unroll
        for (int r = 0; r < 7; r += 2) {
            uint32_t v[32];
            ptx::tmem_ld16(taddr + r * 16, v);
            if (r + 1 < 7) ptx::tmem_ld16(taddr + (r + 1) * 16, v + 16);
            ptx::tmem_wait_ld();
#pragma unroll
            for (int e = 0; e < 7; ++e) pk[r * 7 + e] = pack2<BF16>(v[2 * e], v[2 * e + 1]);
            if (r + 1 < 7) {
#pragma unroll
                for (int e = 0; e < 7; ++e) pk[(r + 1) * 7 + e] = pack2<BF16>(v[16 + 2 * e], v[16 + 2 * e + 1]);
            }
        }
    } else {
        tmem_cols_to_packed<BF16, Bc::ncols(H)>(taddr, pk);
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
// (row pitch W elements, W and W' even): the cyclic shift and the zero padding (Eq. 4-5; DESIGN.md
// A6) become per-thread byte offsets of the window's rows and of the NWR aligned 32-bit words that
// cover one window row, plus validity masks.  Window column e of a thread sits at image column
// (c0 + e) mod W', c0 = (wx*w + s_w) mod W'; with `odd` = c0 & 1 the aligned element pairs of the row
// are  f_k = funnelshift_r(word_k, word_k+1, 16*odd).  Offsets of padding rows / words are 0 so that
// every address is legal; their values are masked (loads) or skipped (stores).
template <int WS>
struct GenAddr {
    static constexpr int NWR = WS / 2 + 1;          // image words that can hold one window row
    int rowoff[WS];
    int coloff[NWR];
    uint32_t rowmask, colmask;                      // bit r / bit k set = inside H x W
    uint32_t sh;                                    // 16 * odd
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
    int c0 = wx * WS + g.sw;
    if (c0 >= g.Wp) c0 -= g.Wp;
    a.sh = (c0 & 1) * 16;
    const int wbase = c0 >> 1, wpr = g.Wp >> 1, wreal = g.W >> 1;
#pragma unroll
    for (int k = 0; k < GenAddr<WS>::NWR; ++k) {
        int wi = wbase + k;
        if (g.sw != 0 && wi >= wpr) wi -= wpr;      // columns wrap only under a shift (then W' is even: whole words wrap)
        a.coloff[k] = wi < wreal ? wi * 4 : 0;
        a.colmask |= (wi < wreal ? 1u : 0u) << k;
    }
}

// General addressing on a STRIP of window rows (maps with more than 128 windows per image): the frame holds the
// strip's rows in ROLLED order (frame row i = rolled row wy0*w + i, loaded as up to two runs of image rows), so the
// row offsets are plain and only the columns wrap.  rowmask is per tile (gen_strip_rowmask).
template <int WS>
__device__ __forceinline__ void gen_addr_init_strip(GenAddr<WS>& a, const Geom& g, int wyl, int wx)
{
    gen_addr_init<WS>(a, g, 0, wx);                  // columns as in the whole-image form
#pragma unroll
    for (int r = 0; r < WS; ++r) a.rowoff[r] = (wyl * WS + r) * g.W * 2;
    a.rowmask = 0xffffffffu;
}
template <int WS>
__device__ __forceinline__ uint32_t gen_strip_rowmask(const Geom& g, int wy)
{
    uint32_t m = 0;
#pragma unroll
    for (int r = 0; r < WS; ++r) {
        int h = wy * WS + r + g.sh;
        if (h >= g.Hp) h -= g.Hp;
        m |= (h < g.H ? 1u : 0u) << r;
    }
    return m;
}
// The (at most two) runs of image rows behind the n rolled rows that start at rolled row R0: run A = image rows
// [a0, a0 + nA) -> frame row 0, run B = image rows [0, nB) -> frame row n1.  Rows at or beyond H (padding) are in
// neither run.
struct StripRuns { int a0, nA, n1, nB; };
__device__ __forceinline__ StripRuns strip_runs(const Geom& g, int R0, int n)
{
    StripRuns s;
    s.a0 = R0 + g.sh;
    if (s.a0 >= g.Hp) s.a0 -= g.Hp;
    s.n1 = min(n, g.Hp - s.a0);
    s.nA = max(0, min(s.a0 + s.n1, g.H) - s.a0);
    s.nB = min(n - s.n1, g.H);
    return s;
}

// The same descriptor for the aligned form (no shift, no padding; frame rows relative to the strip):
// used for odd w, whose window rows start on odd columns for every other window.
template <int WS>
__device__ __forceinline__ void gen_addr_init_plain(GenAddr<WS>& a, int W, int wyl, int wx)
{
    a.rowmask = a.colmask = 0xffffffffu;
#pragma unroll
    for (int r = 0; r < WS; ++r) a.rowoff[r] = (wyl * WS + r) * W * 2;
    const int c0 = wx * WS;
    a.sh = (c0 & 1) * 16;
#pragma unroll
    for (int k = 0; k < GenAddr<WS>::NWR; ++k) a.coloff[k] = ((c0 >> 1) + k) * 4;
}

// lo half of the result = half `ha` of a, hi half = half `hb` of b
template <int HA, int HB>
__device__ __forceinline__ uint32_t pick_halves(uint32_t a, uint32_t b)
{
    return __byte_perm(a, b, (HA ? 0x32 : 0x10) | ((HB ? 0x76 : 0x54) << 8));
}

// The window's N values, two per word in row-major in-window order, v[0 .. NW).  RAGGED = false:
// every window element lies inside H x W (no masks).
// PAR: parity of the window's first column when it is known to the caller (0 / 1; for even w it is the
// parity of the column shift, the same for every window), -1 = per thread from a.sh.
template <int WS, bool RAGGED, int PAR = -1>
__device__ __forceinline__ void window_to_regs_gen(const uint8_t* img, const GenAddr<WS>& a, bool valid, uint32_t* v)
{
    constexpr int NWR = GenAddr<WS>::NWR, NF = (WS + 1) / 2;
    const uint32_t rm = valid ? a.rowmask : 0u;
#pragma unroll
    for (int r = 0; r < WS; ++r) {
        const uint8_t* p = img + a.rowoff[r];
        uint32_t w[NWR + 1];
#pragma unroll
        for (int k = 0; k < NWR; ++k) {
            w[k] = *reinterpret_cast<const uint32_t*>(p + a.coloff[k]);
            if (RAGGED && !((rm >> r) & (a.colmask >> k) & 1u)) w[k] = 0u;
        }
        w[NWR] = 0u;
        uint32_t f[NF + 1];                        // aligned element pairs (e_2k, e_2k+1) of this row
#pragma unroll
        for (int k = 0; k < NF; ++k)
            f[k] = PAR == 0 ? w[k] : (PAR == 1 ? __funnelshift_r(w[k], w[k + 1], 16) : __funnelshift_r(w[k], w[k + 1], a.sh));
        f[NF] = 0u;
        // row r starts at linear position L = r*WS
        const int L = r * WS;
        if (L % 2 == 0) {
#pragma unroll
            for (int k = 0; k < WS / 2; ++k) v[L / 2 + k] = f[k];
            if (WS % 2 == 1) v[(L + WS - 1) / 2] = f[NF - 1] & 0xffffu;       // last element; the next row fills the high half
        } else {
            v[(L - 1) / 2] |= f[0] << 16;                                      // first element -> high half of the previous word
#pragma unroll
            for (int k = 0; k < WS / 2; ++k) v[(L + 1) / 2 + k] = __funnelshift_r(f[k], f[k + 1], 16);   // (e_2k+1, e_2k+2)
        }
    }
    if (!RAGGED && !valid) {
#pragma unroll
        for (int k = 0; k < WinCfg<WS>::NW; ++k) v[k] = 0u;
    }
}

// Linear packed window words v[0 .. NW) -> one A buffer of the bulk kernel (tcgen05.st, all 32
// lanes).  w = 14: every window row is padded to 8 words, the last one zero (BulkCfg<14>).
// pad0: the first padding word of the window's K range -- (row 0, columns 14-15) at w = 14, elements N+1, N+2
// otherwise; 1.0 in its low half turns that K index into a column of ones (the fused bias, see build_lib14).
template <int WS>
__device__ __forceinline__ void packed_window_to_tmem(const uint32_t* v, uint32_t taddr, uint32_t pad0 = 0u)
{
    using Bc = BulkCfg<WS>;
    using Cf = WinCfg<WS>;
    constexpr int NV = (Bc::A_COLS + 15) / 16 * 16;
    uint32_t u[NV];
    if constexpr (Bc::TOEP) {
#pragma unroll
        for (int r = 0; r < WS; ++r) {
#pragma unroll
            for (int k = 0; k < 8; ++k) u[r * 8 + k] = k < 7 ? v[r * 7 + k] : (r == 0 ? pad0 : 0u);
        }
    } else {
#pragma unroll
        for (int k = 0; k < NV; ++k) u[k] = k < Cf::NW ? v[k] : (k == Cf::NW ? pad0 : 0u);
    }
#pragma unroll
    for (int ch = 0; ch < Bc::A_COLS / 16; ++ch) ptx::tmem_st16(taddr + ch * 16, u + ch * 16);
    if constexpr (Bc::A_COLS % 16 != 0) ptx::tmem_st8(taddr + (Bc::A_COLS / 16) * 16, u + (Bc::A_COLS / 16) * 16);
    ptx::tmem_wait_st();
}

template <int WS>
__device__ __forceinline__ void window_to_tmem_bulk(const uint8_t* win, bool valid, int rowB, uint32_t taddr, uint32_t pad0 = 0u)
{
    uint32_t v[WinCfg<WS>::NW];
    window_to_regs<WS>(win, valid, rowB, v);
    packed_window_to_tmem<WS>(v, taddr, pad0);
}

template <int WS, int PAR = -1>
__device__ __forceinline__ void window_to_tmem_gen(const uint8_t* img, const GenAddr<WS>& a, bool valid, bool ragged,
                                                   uint32_t taddr, uint32_t pad0 = 0u)
{
    uint32_t v[WinCfg<WS>::NW];
    if (ragged) window_to_regs_gen<WS, true, PAR>(img, a, valid, v);
    else window_to_regs_gen<WS, false, PAR>(img, a, valid, v);
    packed_window_to_tmem<WS>(v, taddr, pad0);
}

// 7 x 7 maps at w = 7 (the S4 stage): the window IS the plane -- 49 contiguous elements, 98 bytes, so
// planes start on odd elements for every other (image, channel).  The plane sits `off` bytes (a multiple of 2) into
// its plane-box slot; its 25 packed words come from 26 aligned words through one funnel shift by the parity.
__device__ __forceinline__ void window_to_regs_flat7(const uint8_t* slot, int off, bool valid, uint32_t* v)
{
    constexpr int NW = WinCfg<7>::NW;
    const uint32_t sh = (uint32_t)(off & 2) * 8u;
    const uint32_t* p = reinterpret_cast<const uint32_t*>(slot + (off & ~3));
    uint32_t w[NW + 1];
#pragma unroll
    for (int k = 0; k < NW; ++k) w[k] = p[k];           // the 49 elements end inside word NW - 1 for either parity
    w[NW] = 0u;
#pragma unroll
    for (int k = 0; k < NW; ++k) v[k] = valid ? __funnelshift_r(w[k], w[k + 1], sh) : 0u;
    v[NW - 1] &= 0xffffu;                               // there is no element 49
}
__device__ __forceinline__ void window_to_tmem_flat7(const uint8_t* slot, int off, bool valid, uint32_t taddr, uint32_t pad0 = 0u)
{
    uint32_t v[WinCfg<7>::NW];
    window_to_regs_flat7(slot, off, valid, v);
    packed_window_to_tmem<7>(v, taddr, pad0);
}

// ... and the result: 25 packed words to the start of the window's output slot (the plane is copied out from there
// element by element; the high half of the last word falls into the slot's padding)
__device__ __forceinline__ void packed_to_flat7(uint8_t* slot, const uint32_t* pk)
{
#pragma unroll
    for (int k = 0; k < WinCfg<7>::NW; ++k) reinterpret_cast<uint32_t*>(slot)[k] = pk[k];
}

// Packed words [W0, W1) of a window (pk[0] = word W0; the range covers whole window rows, or the
// whole window) -> the window's place in the natural-layout frame.
template <int WS, int W0, int W1, bool RAGGED, int PAR = -1>
__device__ __forceinline__ void packed_to_window_gen(uint8_t* img, const GenAddr<WS>& a, const uint32_t* pk)
{
    constexpr int NWR = GenAddr<WS>::NWR, NF = (WS + 1) / 2;
    constexpr int R0 = (2 * W0) / WS, R1 = (2 * W1 + WS - 1) / WS < WS ? (2 * W1 + WS - 1) / WS : WS;
    static_assert((2 * W0) % WS == 0, "the range starts on a window row");
    const int odd = PAR < 0 ? (int)(a.sh >> 4) : PAR;
    const uint32_t sh = PAR < 0 ? a.sh : (uint32_t)PAR * 16u;
#pragma unroll
    for (int r = R0; r < R1; ++r) {
        // aligned element pairs of the row from the linear packed words
        uint32_t f[NF + 2];
        f[0] = 0u;                                  // f[k+1] = (e_2k, e_2k+1); f[0] and f[NF+1] are zero pads
        const int L = r * WS;
#pragma unroll
        for (int k = 0; k < NF; ++k) {
            const int i0 = L + 2 * k, i1 = i0 + 1;                 // linear positions of the pair
            const uint32_t wa = pk[i0 / 2 - W0];
            const uint32_t wb = (2 * k + 1 < WS) ? pk[i1 / 2 - W0] : 0u;
            if (i0 % 2 == 0) f[k + 1] = (2 * k + 1 < WS) ? wa : (wa & 0xffffu);
            else f[k + 1] = (2 * k + 1 < WS) ? __funnelshift_r(wa, wb, 16) : (wa >> 16);
        }
        f[NF + 1] = 0u;
        uint8_t* p = img + a.rowoff[r];
        const bool rv = !RAGGED || ((a.rowmask >> r) & 1u);
#pragma unroll
        for (int k = 0; k < NWR; ++k) {
            // image word k holds window elements ea = 2k - odd (low half) and ea + 1 (high half)
            const uint32_t val = PAR == 0 ? f[k + 1] : __funnelshift_l(f[k], f[k + 1], sh);
            const int ea = 2 * k - odd;
            const bool ok = rv && (!RAGGED || ((a.colmask >> k) & 1u));
            uint8_t* q = p + a.coloff[k];
            if (ok) {
                if (ea >= 0 && ea + 1 < WS) *reinterpret_cast<uint32_t*>(q) = val;
                else if (ea < 0) *reinterpret_cast<uint16_t*>(q + 2) = (uint16_t)(val >> 16);
                else if (ea < WS) *reinterpret_cast<uint16_t*>(q) = (uint16_t)(val & 0xffffu);
            }
        }
    }
}

// ------------------------------------------------------------------------------- weight builders
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


// The table row of a channel is staged in shared memory as two copies of the fully reversed table
// F[q] = T[NB-1-q] (F0 = F, F1 = F shifted by one value), so that any pair (F[q], F[q+1]) is one
// aligned 32-bit load whatever the parity of q.
constexpr int kTabRegs = (WinCfg<14>::NB + 127) / 128;

// The (reversed) table row of one channel, 128 threads -> registers (loads only; no use yet).
__device__ __forceinline__ void table_to_regs14(const uint16_t* __restrict__ Tc, bool reverse, int tid, uint16_t* v)
{
    using Cf = WinCfg<14>;
#pragma unroll
    for (int u = 0; u < kTabRegs; ++u) {
        const int q = tid + u * 128;
        v[u] = q < Cf::NB ? Tc[reverse ? q : Cf::NB - 1 - q] : (uint16_t)0;
    }
}

// w = 7: the table row (169 entries) in the order the W_c builder reads it, two entries per thread.
__device__ __forceinline__ void table_to_regs7(const uint16_t* __restrict__ Tc, bool reverse, int tid, uint16_t* v)
{
    using Cf = WinCfg<7>;
#pragma unroll
    for (int u = 0; u < 2; ++u) {
        const int q = tid + u * 128;
        v[u] = q < Cf::NB ? Tc[reverse ? Cf::NB - 1 - q : q] : (uint16_t)0;
    }
}

// Block-Toeplitz library for w = 14 (BulkCfg<14>) from the two staged copies of the reversed table
// (see build_weight14): chunk (d, ci, kc) = Z[d-13][ci][8kc .. 8kc+7] = F[(26-d)*27 + 13-ci + 8kc + e].
// 128 threads (the repack warps); rows ci = 14, 15 of every block stay zero from the kernel prologue.
__device__ __forceinline__ void build_lib14(const uint16_t* v, uint16_t* F0, uint16_t* F1, uint8_t* lib, int tid, uint32_t bias_bits = 0u)
{
    using Cf = WinCfg<14>;
    using Bc = BulkCfg<14>;
#pragma unroll
    for (int u = 0; u < kTabRegs; ++u) {
        const int q = tid + u * 128;
        if (q < Cf::NB) {
            F0[q] = v[u];
            if (q >= 1) F1[q - 1] = v[u];
        }
    }
    ptx::named_bar_sync(2, 128);
    for (int id = tid; id < 27 * 28; id += 128) {
        const int d = id / 28, rem = id - d * 28, ci = rem >> 1, kc = rem & 1;
        const int q0 = (26 - d) * 27 + 13 - ci + 8 * kc, p0 = q0 & 1;
        const uint32_t* src = reinterpret_cast<const uint32_t*>(reinterpret_cast<const uint8_t*>(p0 ? F1 : F0) + (q0 - p0) * 2);
        // cj = 14, 15 are padding; the fused bias sits at cj = 14 of every block row and meets the column of ones the
        // repack puts at K index (row 0, cj 14) -- the other rows' pads are zero, so it is added exactly once
        const uint32_t w0 = src[0], w1 = src[1], w2 = src[2], w3 = kc ? bias_bits : src[3];
        *reinterpret_cast<uint4*>(lib + kc * Bc::LBO + (d * 16 + ci) * 16) = make_uint4(w0, w1, w2, w3);
    }
}


// Cached-M mode at w = 14: the GIVEN matrix M_c [196][196] as the B operand of the same MMAs, in
// the row-padded index space the Toeplitz form uses on both GEMM axes (K = rj*16 + cj, N = ri*16 + ci; pads are zero):
// 28 K chunks of 8 x 224 rows x 16 bytes = 100 KB, chunk (kc, n) at byte kc * kFullLbo + n * 16.  K-step ks reads
// chunks 2ks, 2ks + 1; output half h rows 112h ...  The A operand and the accumulator keep the Toeplitz form's
// layout, so repack and epilogue are unchanged.  transpose: M_c^T.  bias_bits sits at K index (row 0, cj = 14), where
// the repack puts the column of ones.  128 threads; a warp reads 8 rows x 56 contiguous bytes of M_c per step.
constexpr int kFullLbo = 224 * 16;
constexpr int kFullBytes = 28 * kFullLbo;          // 100352
__device__ __forceinline__ void load_weight14_full(const uint16_t* __restrict__ Mc, bool transpose, uint8_t* wfull, int tid,
                                                   uint32_t bias_bits)
{
    // 49 chunks per thread, seven at a time: all their loads are issued before the first store
    for (int q0 = tid; q0 < 28 * 224; q0 += 7 * 128) {
        uint32_t w[7][4];
#pragma unroll
        for (int u = 0; u < 7; ++u) {
            const int q = q0 + u * 128;
            const int r = q >> 5, kcg = r % 7, kc = 4 * kcg + (q & 3), n = 8 * (r / 7) + ((q >> 2) & 7);
            const int ri = n >> 4, ci = n & 15, rj = kc >> 1, cj0 = (kc & 1) * 8;
            w[u][0] = w[u][1] = w[u][2] = w[u][3] = 0u;
            if (ci < 14) {
                const int i = ri * 14 + ci, j0 = rj * 14 + cj0;
                if (!transpose) {
                    const uint32_t* src = reinterpret_cast<const uint32_t*>(Mc + i * 196 + j0);      // even element offset
                    w[u][0] = src[0]; w[u][1] = src[1]; w[u][2] = src[2];
                    if (cj0 == 0) w[u][3] = src[3];
                } else {
                    uint32_t v[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) v[e] = cj0 + e < 14 ? (uint32_t)Mc[(j0 + e) * 196 + i] : 0u;
#pragma unroll
                    for (int e = 0; e < 8; ++e) w[u][e >> 1] |= v[e] << ((e & 1) * 16);
                }
                if (kc == 1) w[u][3] = bias_bits;           // K index (row 0, cj 14)
            }
        }
#pragma unroll
        for (int u = 0; u < 7; ++u) {
            const int q = q0 + u * 128;
            const int r = q >> 5, kcg = r % 7, kc = 4 * kcg + (q & 3), n = 8 * (r / 7) + ((q >> 2) & 7);
            *reinterpret_cast<uint4*>(wfull + kc * kFullLbo + n * 16) = make_uint4(w[u][0], w[u][1], w[u][2], w[u][3]);
        }
    }
}

// Second library of the hierarchical operator (BulkCfg<14>): libA[da] = lib[da + 7] + Z_l'[da - 6], da = 0..12,
// Z_l'[dr][ci][cj] = [ci/7 == cj/7] * T_l[(dr+6)*13 + (ci-cj+6)]; FL = the local table staged reversed
// (FL[q] = T_l[168 - q], or T_l[q] for the transposed operator).  Sums are rounded (RNE) to the 16-bit type.
// 128 threads, after build_lib14 and a barrier among them.
template <bool BF16>
__device__ __forceinline__ uint32_t add_pairs(uint32_t a, uint32_t b)
{
    if constexpr (BF16) {
        __nv_bfloat162 r = __hadd2(*reinterpret_cast<__nv_bfloat162*>(&a), *reinterpret_cast<__nv_bfloat162*>(&b));
        return *reinterpret_cast<uint32_t*>(&r);
    } else {
        __half2 r = __hadd2(*reinterpret_cast<__half2*>(&a), *reinterpret_cast<__half2*>(&b));
        return *reinterpret_cast<uint32_t*>(&r);
    }
}

template <bool BF16>
__device__ __forceinline__ void build_lib14_local(const uint8_t* lib, const uint16_t* FL, uint8_t* libA, int tid)
{
    using Bc = BulkCfg<14>;
    for (int id = tid; id < 13 * 28; id += 128) {
        const int da = id / 28, rem = id - da * 28, ci = rem >> 1, kc = rem & 1;
        const uint4 g = *reinterpret_cast<const uint4*>(lib + kc * Bc::LBO + ((da + 7) * 16 + ci) * 16);
        uint32_t l[4];
#pragma unroll
        for (int e2 = 0; e2 < 4; ++e2) {
            uint32_t w = 0;
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
                const int cj = 8 * kc + 2 * e2 + hh;
                if (cj < 14 && (ci >= 7) == (cj >= 7)) w |= (uint32_t)FL[(12 - da) * 13 + 6 - ci + cj] << (16 * hh);
            }
            l[e2] = w;
        }
        *reinterpret_cast<uint4*>(libA + kc * Bc::LBO_A + (da * 16 + ci) * 16) =
            make_uint4(add_pairs<BF16>(g.x, l[0]), add_pairs<BF16>(g.y, l[1]), add_pairs<BF16>(g.z, l[2]), add_pairs<BF16>(g.w, l[3]));
    }
}

constexpr int kThreadsB = 352;
constexpr int kMaxSlots = 96;
// plane boxes (wbmm_tc.cu: plane_box_map) of more than 256 padded elements use the two-dimensional view of the row
__host__ __device__ __forceinline__ bool plane_box_2d(long long plane_elems) { return (plane_elems + 14) / 8 * 8 > 256; }
constexpr int kMaxGrid = 320;     // up to two CTAs per SM (w = 7)
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



}  // namespace tcdev

// Host helpers defined in wbmm_tc.cu.
int num_sms();
// Opts a kernel in to `bytes` of dynamic shared memory unless an earlier call already allowed as much on the
// CURRENT device (`state`: one static per kernel instantiation, zero-initialised; per device, safe to use from
// several host threads).
constexpr int kMaxDevices = 64;
struct SmemOptIn { std::atomic<int> bytes[kMaxDevices]; };
cudaError_t ensure_dynamic_smem(const void* kernel, size_t bytes, SmemOptIn* state);
// Greedy contiguous partition of the tile sequence over `grid` CTAs minimising the largest cost,
// cost = tiles + switch_cost per channel boundary strictly inside a CTA's range.  Returns the
// number of CTAs used.
int partition_tiles(const TcTiles& tl, int grid, double switch_cost, tcdev::TilePart* part);

}  // namespace wbmm
