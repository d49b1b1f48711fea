// INT8 forward on the tensor cores (PAPER.md:749 reports INT8 deployments): signed 8-bit x and
// table, exact 32-bit sums (tcgen05.mma kind::i8, accumulator in TMEM), output either the raw sums (int32) or
// requantised 8-bit values q = sat_s8(rne(fp32(sum) * scale[c])) (reading A21).
//
// Per channel the GEMM is the one of wbmm_tc.cu:  D[m, i] = sum_j X[m, j] * W_c[i, j],  m = window, i = output
// position, j = input position (Alg. 1 l.15).
//   * A = X from TMEM ("TS" form): lane m holds window m's N bytes in row-major in-window order, four per 32-bit
//     column; K = 32 per instruction = 8 columns.
//   * B = W_c built in shared memory from the (2w-1)^2 table (Eq. 6-8), K-major no-swizzle core
//     matrices of 8 rows x 16 bytes (16 values); never in HBM.
//   * D: 128 lanes x N_PAD int32 columns, read back with tcgen05.ld.
// Two kernels: tc_i8_bulk_kernel (NCHW, no shift, aligned sizes: bulk copies, two or three CTAs per SM, see there) and
// tc_i8_kernel, block-synchronous (one tile of up to 128 windows at a time: gather -> TMEM -> MMA -> epilogue ->
// scatter), any layout / shift / ragged size: a warp per frame row, or one run per plane strip for aligned NCHW maps.
#include <cuda.h>

#include <type_traits>

#include "wbmm_common.cuh"
#include "wbmm_ptx.cuh"
#include "wbmm_tc.cuh"

namespace wbmm {

namespace {

constexpr int kThreadsI = 256;   // 8 warps; warps 0-3 own the 128 TMEM lanes

template <int WS>
struct I8Cfg {
    static constexpr int N = WS * WS;
    static constexpr int K_PAD = (N + 31) / 32 * 32;     // MMA K: 32 per instruction
    static constexpr int N_PAD = (N + 15) / 16 * 16;     // MMA N: multiple of 16 at M = 128
    static constexpr int KSTEPS = K_PAD / 32;
    static constexpr int A_COLS = K_PAD / 4;
    static constexpr int TW = 2 * WS - 1;
    static constexpr int NB = TW * TW;
    static constexpr int LBO = N_PAD * 16;               // bytes between K chunks (16 values) of W_c
    static constexpr int WC_BYTES = (K_PAD / 16) * LBO;
    static constexpr int D_COL = (A_COLS + 31) / 32 * 32;
    static constexpr int TMEM_COLS = (D_COL + N_PAD) <= 128 ? 128 : ((D_COL + N_PAD) <= 256 ? 256 : 512);
    static constexpr int TS_BYTES = (NB + 15) / 16 * 16;
    static constexpr int FRAME_BYTES = 128 * N + 128 * 32;   // <= 128 windows, plane stride rounded up to 16 * odd bytes
    // pipelined form: A in shared memory (K-major core matrices, 128 rows), D alone in tensor memory
    static constexpr int A_LBO = 128 * 16;
    static constexpr int A_BYTES = (K_PAD / 16) * A_LBO;
};

struct I8Tiles {
    int NP, NSY, nstrips, tiles_per_c;
    int frame_rows, S;       // rows of one frame plane; plane stride in bytes (multiple of 16)
    long long ntiles;
    int bulk;                // plane strips are contiguous 16-byte aligned runs: the bulk-copy kernel serves (see i8_tiles)
    int rot;                 // gather kernel, NCHW with shift on maps without padding: frame rows hold the SOURCE row unrotated
                             // (copied in units of `rot` bytes, 4 or 1); the windows read and write their columns rotated by the shift
    int runs;                // (= rot != 0) a plane strip is TWO contiguous runs of source rows (before / after the row wrap),
                             // copied like the flat form
    int flat;                // gather kernel: a plane strip is ONE contiguous run (NCHW, no shift, H and W multiples of w),
                             // copied by a warp in units of `flat` bytes (4 or 1) without per-element index arithmetic
};

// kind::i8: c_format S32 (2), a / b signed 8-bit (1).  kind::f8f6f4: c_format F32 (1), a / b E4M3 (0).  K-major both.
template <bool F8>
__host__ __device__ constexpr uint32_t idesc_8bit(int M, int N)
{
    return (F8 ? (1u << 4) : ((2u << 4) | (1u << 7) | (1u << 10))) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

template <bool F8>
__device__ __forceinline__ void mma_ts_i8(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    if constexpr (F8)
        asm volatile("{ .reg .pred p; setp.ne.b32 p, %4, 0; tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], [%1], %2, %3, p; }" ::"r"(d_tmem),
                     "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
    else
        asm volatile("{ .reg .pred p; setp.ne.b32 p, %4, 0; tcgen05.mma.cta_group::1.kind::i8 [%0], [%1], %2, %3, p; }" ::"r"(d_tmem),
                     "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}

template <bool F8>
__device__ __forceinline__ void mma_ss_i8(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    if constexpr (F8)
        asm volatile("{ .reg .pred p; setp.ne.b32 p, %4, 0; tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p; }" ::"r"(d_tmem),
                     "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
    else
        asm volatile("{ .reg .pred p; setp.ne.b32 p, %4, 0; tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p; }" ::"r"(d_tmem),
                     "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}

// W_c[i][j] = T[c, rel(i, j)] (Eq. 7) in the K-major core-matrix layout: value (i, j) at byte (j/16)*LBO + i*16 + j%16.
// The table row is staged REVERSED (F[q] = T[NB-1-q]): then rel(i, j) reads F at (w-1-ri+rj)*(2w-1) + (w-1-ci+cj), which
// is one per-thread base plus a compile-time constant of j -- thread i builds row i, all K chunks unrolled, two
// instructions per byte.  Rows i >= N and columns j >= N are zero.
template <int WS>
__device__ __forceinline__ void build_weight_i8(const int8_t* __restrict__ Tc, uint8_t* Ts, uint8_t* Wc, int tid)
{
    using Cf = I8Cfg<WS>;
    for (int k = tid; k < Cf::NB; k += kThreadsI) Ts[k] = (uint8_t)Tc[Cf::NB - 1 - k];
    __syncthreads();
    if (tid < Cf::N_PAD) {
        const int i = tid;
        const int ri = i / WS, ci = i % WS;
        const uint8_t* f = Ts + (i < Cf::N ? (WS - 1 - ri) * Cf::TW + (WS - 1 - ci) : 0);
#pragma unroll
        for (int kc = 0; kc < Cf::K_PAD / 16; ++kc) {
            uint32_t pk[4] = {0u, 0u, 0u, 0u};
            if (i < Cf::N) {
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    const int j = kc * 16 + e;
                    if (j < Cf::N) pk[e >> 2] |= (uint32_t)f[(j / WS) * Cf::TW + (j % WS)] << ((e & 3) * 8);
                }
            }
            *reinterpret_cast<uint4*>(Wc + kc * Cf::LBO + i * 16) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
        }
    }
}

// Bytes [16*KC0, 16*KC1) of a window (row-major order) from the frame into row m of the A tile, 16 bytes per K chunk.
template <int WS, int KC0, int KC1>
__device__ __forceinline__ void stage_window_i8(const uint8_t* win, int rowB, uint8_t* arow)
{
    using Cf = I8Cfg<WS>;
    constexpr int NV = (KC1 - KC0) * 4;
    uint32_t v[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) v[k] = 0u;
    if constexpr (WS % 2 == 0) {
#pragma unroll
        for (int h = KC0 * 8; h < KC1 * 8; ++h)          // halfword h = bytes 2h, 2h+1 (a row is WS/2 aligned halfwords)
            if (2 * h < Cf::N) {
                const uint32_t u = *reinterpret_cast<const uint16_t*>(win + (h / (WS / 2)) * rowB + 2 * (h % (WS / 2)));
                v[(h >> 1) - KC0 * 4] |= u << ((h & 1) * 16);
            }
    } else {
#pragma unroll
        for (int b = KC0 * 16; b < KC1 * 16; ++b)
            if (b < Cf::N) v[(b >> 2) - KC0 * 4] |= (uint32_t)win[(b / WS) * rowB + (b % WS)] << ((b & 3) * 8);
    }
#pragma unroll
    for (int kc = KC0; kc < KC1; ++kc)
        *reinterpret_cast<uint4*>(arow + kc * Cf::A_LBO) =
            make_uint4(v[4 * (kc - KC0)], v[4 * (kc - KC0) + 1], v[4 * (kc - KC0) + 2], v[4 * (kc - KC0) + 3]);
}

// Window -> TMEM A (warp-collective): the N bytes in row-major order, four per column; lanes without a window and
// the K padding write zeros.
template <int WS>
__device__ __forceinline__ void window_to_tmem_i8(const uint8_t* win, bool valid, int rowB, uint32_t taddr)
{
    using Cf = I8Cfg<WS>;
    constexpr int NV = (Cf::A_COLS + 7) / 8 * 8;
    uint32_t v[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) v[k] = 0u;
    if (valid) {
        if constexpr (WS % 2 == 0) {
            // a window row is WS/2 aligned halfwords; halfword q = r*(WS/2) + k of the window lands in word q/2
#pragma unroll
            for (int r = 0; r < WS; ++r)
#pragma unroll
                for (int k = 0; k < WS / 2; ++k) {
                    const int q = r * (WS / 2) + k;
                    const uint32_t h = *reinterpret_cast<const uint16_t*>(win + r * rowB + 2 * k);
                    v[q >> 1] |= h << ((q & 1) * 16);
                }
        } else {
#pragma unroll
            for (int r = 0; r < WS; ++r)
#pragma unroll
                for (int k = 0; k < WS; ++k) {
                    const int q = r * WS + k;
                    v[q >> 2] |= (uint32_t)win[r * rowB + k] << ((q & 3) * 8);
                }
        }
    }
#pragma unroll
    for (int ch = 0; ch < NV / 8; ++ch) ptx::tmem_st8(taddr + ch * 8, v + ch * 8);
    ptx::tmem_wait_st();
}

// q = sat_s8(rne(fp32(sum) * scale)) without the conversion unit (I2F / F2I issue at a quarter of the FP32 rate and were
// the floor of the epilogue): |sum| <= 196 * 128 * 128 < 2^22, so  fp32(sum) = as_float(0x4B400000 + sum) - 1.5 * 2^23
// exactly; one binary32 product (no fma); clamping to [-128, 127] BEFORE rounding gives the same integer as after
// (the bounds are integers, rounding is monotone); adding 1.5 * 2^23 rounds to the nearest integer, ties to even, and
// leaves the two's-complement value in the low mantissa bits.  The low byte of the result is q.
// The same from a frame whose rows hold the source row unrotated: column k of the window is at byte v0 + k of the row, or
// v0 + k - W' once that runs past the row's end (kw = W' - v0 columns come before the wrap; kw >= w: none).
template <int WS>
__device__ __forceinline__ void window_to_tmem_i8_rot(const uint8_t* rows, int v0, int kw, int rowB, bool valid, uint32_t taddr)
{
    using Cf = I8Cfg<WS>;
    constexpr int NV = (Cf::A_COLS + 7) / 8 * 8;
    uint32_t v[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) v[k] = 0u;
    if (valid) {
        int offk[WS];                      // byte of the row that holds the window's column k
#pragma unroll
        for (int k = 0; k < WS; ++k) offk[k] = k < kw ? v0 + k : v0 + k - rowB;
#pragma unroll
        for (int r = 0; r < WS; ++r) {
            const uint8_t* row = rows + r * rowB;
#pragma unroll
            for (int k = 0; k < WS; ++k) {
                const int q = r * WS + k;
                v[q >> 2] |= (uint32_t)row[offk[k]] << ((q & 3) * 8);
            }
            asm volatile("" ::: "memory");      // a row at a time: with all w*w loads hoisted the kernel spilled 764 bytes
        }
    }
#pragma unroll
    for (int ch = 0; ch < NV / 8; ++ch) ptx::tmem_st8(taddr + ch * 8, v + ch * 8);
    ptx::tmem_wait_st();
}

__device__ __forceinline__ uint32_t requant(uint32_t acc_bits, float scale)
{
    const float f = __fsub_rn(__uint_as_float(0x4B400000u + acc_bits), 12582912.0f);
    float r = __fmul_rn(f, scale);
    r = fminf(fmaxf(r, -128.0f), 127.0f);
    return __float_as_uint(__fadd_rn(r, 12582912.0f));
}
// Two values at once with the packed binary32 instructions of sm_100 (sub / mul / add .f32x2: each lane is the scalar
// operation, same rounding); returns q(a0) | q(a1) << 8.
__device__ __forceinline__ uint64_t pack_f2(float lo, float hi)
{
    return (uint64_t)__float_as_uint(lo) | ((uint64_t)__float_as_uint(hi) << 32);
}
__device__ __forceinline__ uint32_t requant2(uint32_t a0, uint32_t a1, uint64_t scale2)
{
    const uint64_t magic2 = pack_f2(12582912.0f, 12582912.0f);
    uint64_t x = (uint64_t)(0x4B400000u + a0) | ((uint64_t)(0x4B400000u + a1) << 32);
    asm("sub.rn.f32x2 %0, %0, %1;\n\tmul.rn.f32x2 %0, %0, %2;" : "+l"(x) : "l"(magic2), "l"(scale2));
    const float r0 = fminf(fmaxf(__uint_as_float((uint32_t)x), -128.0f), 127.0f);
    const float r1 = fminf(fmaxf(__uint_as_float((uint32_t)(x >> 32)), -128.0f), 127.0f);
    uint64_t t = pack_f2(r0, r1);
    asm("add.rn.f32x2 %0, %0, %1;" : "+l"(t) : "l"(magic2));
    return __byte_perm((uint32_t)t, (uint32_t)(t >> 32), 0x0040) & 0xffffu;
}

// FP8 output: E4M3 codes of (sum * scale), round-to-nearest-even, saturating at +-448 (cvt.rn.satfinite.e4m3x2.f32: the
// first source lands in the HIGH byte).  Returns code(a0) | code(a1) << 8.
__device__ __forceinline__ uint32_t to_e4m3x2(uint32_t a0, uint32_t a1, float scale)
{
    const float r0 = __fmul_rn(__uint_as_float(a0), scale), r1 = __fmul_rn(__uint_as_float(a1), scale);
    uint16_t d;
    asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(d) : "f"(r1), "f"(r0));
    return d;
}
// One pair of outputs as two 8-bit codes (int8: requantised; fp8: E4M3), low byte = the first.
template <bool F8>
__device__ __forceinline__ uint32_t out_pair(uint32_t a0, uint32_t a1, float sc, uint64_t sc2)
{
    if constexpr (F8) return to_e4m3x2(a0, a1, sc);
    else return requant2(a0, a1, sc2);
}

// ROT: the rot / runs forms (NCHW with shift or ragged size) are their own instantiation -- in one kernel with the flat and
// row forms the register allocation collapsed (255 registers, 892 bytes of spills)
template <int WS, bool OUT8, bool F8, bool ROT>
__global__ void __launch_bounds__(kThreadsI, 1)
tc_i8_kernel(Geom g, I8Tiles tl, const int8_t* __restrict__ x, const int8_t* __restrict__ T, const float* __restrict__ scale,
             void* __restrict__ yv)
{
    using Cf = I8Cfg<WS>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* Wc = smem;
    uint8_t* Ts = smem + Cf::WC_BYTES;
    uint8_t* frame = smem + Cf::WC_BYTES + Cf::TS_BYTES;
    int32_t* oframe = reinterpret_cast<int32_t*>(frame + Cf::FRAME_BYTES);   // int32 output staging (OUT8: unused)
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
    constexpr uint32_t idesc = idesc_8bit<F8>(128, Cf::N_PAD);

    const long long t0 = tl.ntiles * blockIdx.x / gridDim.x, t1 = tl.ntiles * (blockIdx.x + 1) / gridDim.x;
    const int rowB = g.Wp;
    const int frame_elems = tl.frame_rows * g.Wp;
    int cur_c = -1;
    uint32_t phase = 0;

    // this thread's window (warps 0-3 only): m = wl * NP + pl
    const int m = tid & 127;
    const int wl = m / tl.NP, pl = m % tl.NP;
    const int wyl = wl / g.nww, wx = wl % g.nww;
    const int win_off = (wyl * WS) * g.Wp + wx * WS;
    uint8_t* win = frame + pl * tl.S + win_off;
    // rot mode: this window's rows start at row_off (bytes of the frame plane / elements of the int32 plane), its columns
    // at v0 of the unrotated row, kw of them before the wrap
    const int row_off = (wyl * WS) * g.Wp;
    int v0 = wx * WS + g.sw;
    if (v0 >= g.Wp) v0 -= g.Wp;
    const int kw = g.Wp - v0;

    int8_t* y8 = static_cast<int8_t*>(yv);
    int32_t* y32 = static_cast<int32_t*>(yv);

    for (long long t = t0; t < t1; ++t) {
        const int c = (int)(t / tl.tiles_per_c);
        const int rem = (int)(t % tl.tiles_per_c);
        const int gb = rem / tl.nstrips, strip = rem % tl.nstrips;
        const int b0 = gb * tl.NP, wy0 = strip * tl.NSY;
        const int np_eff = min(tl.NP, g.B - b0);

        if (c != cur_c) {   // (the previous tile's MMAs have completed: every thread waited on mma_bar)
            build_weight_i8<WS>(T + (long long)c * Cf::NB, Ts, Wc, tid);
            cur_c = c;
        }
        const int strip_elems = min(tl.NSY, g.nwh - wy0) * WS * g.Wp;                 // flat mode: the strip's run
        const long long strip_off = (long long)c * g.H * g.W + (long long)wy0 * WS * g.Wp;    // ... inside image b's block
        const long long img_pitch = (long long)g.C * g.H * g.W;
        if (!ROT && tl.flat == 4) {
            const int nu = strip_elems >> 2;
            for (int p = warp; p < np_eff; p += kThreadsI / 32) {
                const uint32_t* sp = reinterpret_cast<const uint32_t*>(x + (b0 + p) * img_pitch + strip_off);
                uint32_t* dp = reinterpret_cast<uint32_t*>(frame + p * tl.S);
                for (int u = lane; u < nu; u += 128) {
                    uint32_t val[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) if (u + 32 * k < nu) val[k] = sp[u + 32 * k];
#pragma unroll
                    for (int k = 0; k < 4; ++k) if (u + 32 * k < nu) dp[u + 32 * k] = val[k];
                }
            }
        } else if (!ROT && tl.flat == 1) {
            for (int p = warp; p < np_eff; p += kThreadsI / 32) {
                const int8_t* sp = x + (b0 + p) * img_pitch + strip_off;
                uint8_t* dp = frame + p * tl.S;
                for (int u = lane; u < strip_elems; u += 128) {
                    uint8_t val[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) if (u + 32 * k < strip_elems) val[k] = (uint8_t)sp[u + 32 * k];
#pragma unroll
                    for (int k = 0; k < 4; ++k) if (u + 32 * k < strip_elems) dp[u + 32 * k] = val[k];
                }
            }
        } else if (ROT && tl.runs) {
            // shift without padding: frame rows [0, lenA) <- source rows [s0, s0 + lenA), frame rows [lenA, R) <- source rows
            // [0, R - lenA): two contiguous runs per plane, a warp per plane
            const int R = strip_elems / g.W;
            int s0 = wy0 * WS + g.sh;
            if (s0 >= g.Hp) s0 -= g.Hp;
            const int lenA = min(R, g.Hp - s0);
            const int nA = lenA * g.W / tl.rot, nB = (R - lenA) * g.W / tl.rot;
            for (int p = warp; p < np_eff; p += kThreadsI / 32) {
                const int8_t* pb = x + (b0 + p) * img_pitch + (long long)c * g.H * g.W;
#pragma unroll
                for (int run = 0; run < 2; ++run) {
                    const int nu = run ? nB : nA;
                    const int8_t* sp = pb + (run ? 0 : (long long)s0 * g.W);
                    uint8_t* dp = frame + p * tl.S + (run ? lenA * g.W : 0);
                    for (int u = lane; u < nu; u += 128) {
                        uint32_t val[4];
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            if (u + 32 * k < nu) val[k] = tl.rot == 4 ? reinterpret_cast<const uint32_t*>(sp)[u + 32 * k] : (uint32_t)(uint8_t)sp[u + 32 * k];
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            if (u + 32 * k < nu) {
                                if (tl.rot == 4) reinterpret_cast<uint32_t*>(dp)[u + 32 * k] = val[k];
                                else dp[u + 32 * k] = (uint8_t)val[k];
                            }
                    }
                }
            }
        } else if (!ROT) {
            // general form: a warp per frame row -- the row's source (shifted row, padding) is worked out once, the lanes
            // walk its columns (column shift and crop by a compare; NHWC by the element stride): no division per element
            const int nrows = np_eff * tl.frame_rows;
            const int estride = g.layout == WBMM_LAYOUT_NCHW ? 1 : g.C;
            const long long rowstride = (long long)g.W * estride;
            const int8_t* xb = x + act_offset(g, b0, c, 0, 0);           // element (b0 + p, c, h, v) = xb[p * img_pitch + h * rowstride + v * estride]
            // eight consecutive rows per warp and step, all their loads issued before the first shared-memory store (a row
            // at a time is one global-memory latency per row); (plane, row) advance by additions -- a division per row and
            // the general offset arithmetic made this loop 100 M of the kernel's 174 M instructions
            constexpr int RB = 8;
            for (int r0 = warp * RB; r0 < nrows; r0 += RB * (kThreadsI / 32)) {
                const int p0 = r0 / tl.frame_rows, hh0 = r0 - p0 * tl.frame_rows;
                for (int vv0 = 0; vv0 < g.Wp; vv0 += 64) {
                    uint8_t val[RB][2];
                    int p = p0, hh = hh0;
#pragma unroll
                    for (int j = 0; j < RB; ++j) {
                        const int hp = wy0 * WS + hh;
                        int h = hp + g.sh;
                        if (h >= g.Hp) h -= g.Hp;
                        const bool rowok = r0 + j < nrows && hp < g.Hp && h < g.H;
                        const int8_t* srow = xb + (rowok ? p * img_pitch + h * rowstride : 0);
#pragma unroll
                        for (int k = 0; k < 2; ++k) {
                            const int vv = vv0 + lane + 32 * k;
                            int v = vv + g.sw;
                            if (v >= g.Wp) v -= g.Wp;
                            val[j][k] = (rowok && vv < g.Wp && v < g.W) ? (uint8_t)srow[v * estride] : (uint8_t)0;
                        }
                        if (++hh == tl.frame_rows) { hh = 0; ++p; }
                    }
                    p = p0; hh = hh0;
#pragma unroll
                    for (int j = 0; j < RB; ++j) {
                        if (r0 + j < nrows) {
                            uint8_t* drow = frame + p * tl.S + hh * g.Wp;
#pragma unroll
                            for (int k = 0; k < 2; ++k) {
                                const int vv = vv0 + lane + 32 * k;
                                if (vv < g.Wp) drow[vv] = val[j][k];
                            }
                        }
                        if (++hh == tl.frame_rows) { hh = 0; ++p; }
                    }
                }
            }
        }
        ptx::fence_proxy_async_smem();   // W_c (generic-proxy stores) -> tcgen05.mma operand reads
        __syncthreads();

        // the next tile's planes -> L2 while this one is multiplied (one CTA per SM and plain loads: without it every tile
        // waits out a DRAM round trip; whole-image tiles of the run-copy forms only)
        if ((tl.flat || tl.runs) && tl.nstrips == 1 && t + 1 < t1) {
            const int c2 = (int)((t + 1) / tl.tiles_per_c);
            const int b2 = (int)((t + 1) % tl.tiles_per_c) * tl.NP;
            const int np2 = min(tl.NP, g.B - b2);
            const int pbytes = g.H * g.W, lines = (pbytes + 127) >> 7;
            for (int i = tid; i < np2 * lines; i += kThreadsI) {
                const int p = i / lines, l = i - p * lines;
                const int8_t* a = x + (b2 + p) * img_pitch + (long long)c2 * pbytes + min(l << 7, pbytes - 1);
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
            }
        }

        const bool valid = wl < tl.NSY * g.nww && pl < np_eff && wy0 + wyl < g.nwh;
        if (warp < 4) {
            if constexpr (ROT) window_to_tmem_i8_rot<WS>(frame + pl * tl.S + row_off, v0, kw, rowB, valid, tmem_a + ((uint32_t)(warp * 32) << 16));
            else window_to_tmem_i8<WS>(win, valid, rowB, tmem_a + ((uint32_t)(warp * 32) << 16));
            ptx::tc_fence_before_sync();
        }
        __syncthreads();
        if (warp == 4 && lane == 0) {
            ptx::tc_fence_after_sync();
            const uint32_t wc_addr = ptx::smem_u32(Wc);
#pragma unroll
            for (int ks = 0; ks < Cf::KSTEPS; ++ks) {
                const uint64_t bdesc = ptx::smem_desc_kmajor_noswz(wc_addr + ks * 2 * Cf::LBO, Cf::LBO, 128);
                mma_ts_i8<F8>(tmem_d, tmem_a + ks * 8, bdesc, idesc, ks > 0 ? 1u : 0u);
            }
            ptx::mma_commit(bar);
        }
        ptx::mbar_wait(bar, phase);
        phase ^= 1;
        ptx::tc_fence_after_sync();
        if (warp < 4) {
            const uint32_t td = tmem_d + ((uint32_t)(warp * 32) << 16);
            const float sc = OUT8 ? scale[c] : 0.f;
            int32_t* owin = oframe + pl * frame_elems + win_off;
            int offk[WS];                  // ROT: byte / element of the unrotated row that holds the window's column k
#pragma unroll
            for (int k = 0; k < WS; ++k) offk[k] = k < kw ? v0 + k : v0 + k - rowB;
#pragma unroll
            for (int ch = 0; ch < Cf::N_PAD / 16; ++ch) {
                uint32_t v[16];
                ptx::tmem_ld16(td + ch * 16, v);
                ptx::tmem_wait_ld();
                if (valid) {
#pragma unroll
                    for (int e = 0; e < 16; ++e) {
                        const int i = ch * 16 + e;
                        if (i < Cf::N) {
                            const int r = i / WS, k = i % WS;
                            if constexpr (ROT) {      // column k of the window sits at v0 + k of the unrotated row, wrapped
                                const int col = r * rowB + offk[k];
                                if constexpr (!OUT8) oframe[pl * frame_elems + row_off + col] = (int32_t)v[e];
                                else frame[pl * tl.S + row_off + col] = (uint8_t)(F8 ? to_e4m3x2(v[e], 0u, sc) : requant(v[e], sc));
                            } else if constexpr (!OUT8) {
                                owin[r * rowB + k] = (int32_t)v[e];
                            } else if constexpr (WS % 2 == 0) {
                                if ((k & 1) == 0)   // (i and i+1 are in the same chunk: 16 and WS are even)
                                    *reinterpret_cast<uint16_t*>(win + r * rowB + k) =
                                        (uint16_t)out_pair<F8>(v[e], v[e + 1], sc, pack_f2(sc, sc));
                            } else {
                                win[r * rowB + k] = (uint8_t)(F8 ? to_e4m3x2(v[e], 0u, sc) : requant(v[e], sc));
                            }
                        }
                    }
                }
            }
            ptx::tc_fence_before_sync();
        }
        __syncthreads();
        // y <- frame (un-shift, crop)
        if (!ROT && tl.flat) {
            constexpr int ES = OUT8 ? 1 : 4;
            const bool words = !OUT8 || tl.flat == 4;
            const int nu = words ? strip_elems * ES / 4 : strip_elems;
            for (int p = warp; p < np_eff; p += kThreadsI / 32) {
                uint8_t* dp = static_cast<uint8_t*>(yv) + ((b0 + p) * img_pitch + strip_off) * ES;
                const uint8_t* sp = OUT8 ? frame + p * tl.S : reinterpret_cast<const uint8_t*>(oframe + p * frame_elems);
                if (words) {
                    for (int u = lane; u < nu; u += 32) reinterpret_cast<uint32_t*>(dp)[u] = reinterpret_cast<const uint32_t*>(sp)[u];
                } else {
                    for (int u = lane; u < nu; u += 32) dp[u] = sp[u];
                }
            }
        } else if (ROT && tl.runs) {
            constexpr int ES = OUT8 ? 1 : 4;
            const int R = strip_elems / g.W;
            int s0 = wy0 * WS + g.sh;
            if (s0 >= g.Hp) s0 -= g.Hp;
            const int lenA = min(R, g.Hp - s0);
            const bool words = !OUT8 || tl.rot == 4;
            for (int p = warp; p < np_eff; p += kThreadsI / 32) {
                uint8_t* pb = static_cast<uint8_t*>(yv) + ((b0 + p) * img_pitch + (long long)c * g.H * g.W) * ES;
                const uint8_t* fb = OUT8 ? frame + p * tl.S : reinterpret_cast<const uint8_t*>(oframe + p * frame_elems);
#pragma unroll
                for (int run = 0; run < 2; ++run) {
                    const int nbytes = (run ? R - lenA : lenA) * g.W * ES;
                    uint8_t* dp = pb + (run ? 0 : (long long)s0 * g.W * ES);
                    const uint8_t* sp = fb + (run ? lenA * g.W * ES : 0);
                    if (words) for (int u = lane; u < nbytes / 4; u += 32) reinterpret_cast<uint32_t*>(dp)[u] = reinterpret_cast<const uint32_t*>(sp)[u];
                    else for (int u = lane; u < nbytes; u += 32) dp[u] = sp[u];
                }
            }
        } else if (!ROT) {
            const int nrows = np_eff * tl.frame_rows;
            const int estride = g.layout == WBMM_LAYOUT_NCHW ? 1 : g.C;
            const long long rowstride = (long long)g.W * estride;
            const long long yb = act_offset(g, b0, c, 0, 0);
            int p = warp / tl.frame_rows, hh = warp - p * tl.frame_rows;       // row rr = warp, warp + 8, ...: (p, hh) by additions
            for (int rr = warp; rr < nrows; rr += kThreadsI / 32) {
                const int hp = wy0 * WS + hh;
                int h = hp + g.sh;
                if (h >= g.Hp) h -= g.Hp;
                if (hp < g.Hp && h < g.H) {                                   // padding rows are cropped
                    const long long rbase = yb + p * img_pitch + h * rowstride;
                    const int fo = p * (OUT8 ? tl.S : frame_elems) + hh * g.Wp;
                    for (int vv = lane; vv < g.Wp; vv += 32) {
                        int v = vv + g.sw;
                        if (v >= g.Wp) v -= g.Wp;
                        if (v < g.W) {
                            if constexpr (OUT8) y8[rbase + v * estride] = (int8_t)frame[fo + vv];
                            else y32[rbase + v * estride] = oframe[fo + vv];
                        }
                    }
                }
                hh += kThreadsI / 32;
                while (hh >= tl.frame_rows) { hh -= tl.frame_rows; ++p; }
            }
        }
        __syncthreads();
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 0) ptx::tmem_dealloc(tmem, Cf::TMEM_COLS);
}

// ------------------------------------------------------------------------------------------------
// Bulk-copy form: NCHW, no shift, H and W multiples of w, plane strips that are 16-byte aligned runs.  A plane strip
// moves global <-> shared memory as ONE 1-D bulk copy (cp.async.bulk, TMA engine); the next tile's planes are in
// flight while the current tile is multiplied and requantised.  A is staged in shared memory (tcgen05.mma "SS" form)
// so that tensor memory holds D only (208 columns at w = 14 -> 256 allocated): two CTAs share an SM (three at w = 7)
// and fill each other's barrier waits.  Per tile:
//   wait full | windows: frame -> registers -> A (16-byte chunks, conflict-free) | sync | load of tile t+1 starts
//   7 (w = 14) / 2 (w = 7) MMAs | tcgen05.ld -> requantise -> output planes (over the A tile) | sync | 16-byte stores
// (A bulk store would have to be waited for before the next A tile overwrites its source: measured 2.5 us per tile.)
// MT: 128-window sub-tiles per tile.  At w = 7 a 128-window tile is 6 KB and its fixed costs (barriers, MMA round trip,
// tile arithmetic) dominate: four sub-tiles share them (4 x 64 TMEM columns, two CTAs per SM).
template <int WS, bool OUT8>
constexpr int i8_mt() { return (WS == 7 && OUT8) ? 4 : 1; }
template <int WS, bool OUT8>
constexpr int i8_ctas() { return WS == 7 ? (OUT8 ? 2 : 3) : (OUT8 ? 2 : 1); }

template <int WS, bool OUT8>
struct I8Fast {
    using Cf = I8Cfg<WS>;
    static constexpr int MT = i8_mt<WS, OUT8>();
    static constexpr int FRAME_BYTES = MT * Cf::FRAME_BYTES;
    static constexpr int OUT_BYTES = OUT8 ? FRAME_BYTES : MT * 128 * Cf::N * 4;
    static constexpr int AO_BYTES = (MT * Cf::A_BYTES > OUT_BYTES ? MT * Cf::A_BYTES : OUT_BYTES);
    static constexpr int D_COLS = MT * Cf::N_PAD <= 32 ? 32 : (MT * Cf::N_PAD <= 64 ? 64 : (MT * Cf::N_PAD <= 128 ? 128 : (MT * Cf::N_PAD <= 256 ? 256 : 512)));
    static constexpr int OFF_TS = Cf::WC_BYTES;
    static constexpr int OFF_FRAME = (OFF_TS + Cf::TS_BYTES + 127) / 128 * 128;
    static constexpr int OFF_AO = (OFF_FRAME + FRAME_BYTES + 127) / 128 * 128;
    static constexpr int SMEM = OFF_AO + AO_BYTES;
};

template <int WS, bool OUT8, bool F8>
__global__ void __launch_bounds__(kThreadsI, i8_ctas<WS, OUT8>())
tc_i8_bulk_kernel(Geom g, I8Tiles tl, const int8_t* __restrict__ x, const int8_t* __restrict__ T,
                  const float* __restrict__ scale, void* __restrict__ yv)
{
    using Cf = I8Cfg<WS>;
    using Sm = I8Fast<WS, OUT8>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* Wc = smem;
    uint8_t* Ts = smem + Sm::OFF_TS;
    uint8_t* frame = smem + Sm::OFF_FRAME;
    uint8_t* ao = smem + Sm::OFF_AO;          // the A tile, then the tile's output planes
    __shared__ __align__(8) uint64_t bars[2];
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t mma_bar = ptx::smem_u32(&bars[0]), full_bar = ptx::smem_u32(&bars[1]);
    constexpr int MT = Sm::MT;
    if (warp == 0) ptx::tmem_alloc(ptx::smem_u32(&tmem_base_s), Sm::D_COLS);
    if (tid == 32) {
        ptx::mbar_init(mma_bar, 1);
        ptx::mbar_init(full_bar, 1);
        ptx::fence_mbar_init();
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::tc_fence_after_sync();
    const uint32_t tmem_d = tmem_base_s;
    constexpr uint32_t idesc = idesc_8bit<F8>(128, Cf::N_PAD);

    const long long t0 = tl.ntiles * blockIdx.x / gridDim.x, t1 = tl.ntiles * (blockIdx.x + 1) / gridDim.x;
    const int rowB = g.W;
    const int frame_elems = tl.frame_rows * g.W;
    const long long plane = (long long)g.H * g.W;
    const int So = OUT8 ? tl.S : frame_elems * 4;        // output plane stride in shared memory (bytes)
    int cur_c = -1;
    uint32_t phase = 0;

    // this thread's windows: row m of sub-tile s is window m + 128 s of the tile = (wl, pl) with m + 128 s = wl * NP + pl
    // (recomputed where used: held in registers across the tile loop -- plain or packed -- they push the kernels with
    // 80 or 128 registers into spills inside the hot loops: int32-out 59 -> 88 us at w = 7, 87 -> 97 us at w = 14)
    const int m = tid & 127;
    struct Win { int pl, wyl, off; bool in; };
    auto window_of = [&](int s) -> Win {
        const int ms = m + 128 * s;
        const int wl = ms / tl.NP;
        Win w;
        w.pl = ms - wl * tl.NP;
        w.wyl = wl / g.nww;
        w.in = wl < tl.NSY * g.nww;
        w.off = w.in ? (w.wyl * WS) * g.W + (wl - w.wyl * g.nww) * WS : 0;
        return w;
    };

    struct Tile { int c, b0, wy0, np, bytes; };
    auto tile_at = [&](long long t) -> Tile {
        Tile q;
        q.c = (int)(t / tl.tiles_per_c);
        const int rem = (int)(t % tl.tiles_per_c);
        const int gb = rem / tl.nstrips, strip = rem % tl.nstrips;
        q.b0 = gb * tl.NP;
        q.wy0 = strip * tl.NSY;
        q.np = min(tl.NP, g.B - q.b0);
        q.bytes = min(tl.NSY, g.nwh - q.wy0) * WS * g.W;
        return q;
    };
    auto load_tile = [&](const Tile& q) {    // one thread
        ptx::mbar_arrive_expect_tx(full_bar, (uint32_t)(q.np * q.bytes));
        const int8_t* src = x + ((long long)q.b0 * g.C + q.c) * plane + (long long)q.wy0 * WS * g.W;
        for (int p = 0; p < q.np; ++p)
            ptx::bulk_g2s(ptx::smem_u32(frame + p * tl.S), src + (long long)p * g.C * plane, (uint32_t)q.bytes, full_bar);
    };
    if (tid == 0 && t0 < t1) load_tile(tile_at(t0));

    for (long long t = t0; t < t1; ++t) {
        const Tile q = tile_at(t);
        if (q.c != cur_c) {   // (the previous tile's MMAs have completed: every thread waited on mma_bar)
            build_weight_i8<WS>(T + (long long)q.c * Cf::NB, Ts, Wc, tid);
            cur_c = q.c;
        }
        ptx::mbar_wait(full_bar, phase);
        // this thread's window -> registers (row-major bytes, four per word) -> row m of A; warps 0-3 take the first
        // half of the K chunks, warps 4-7 the rest
        {
            constexpr int KCH = (Cf::K_PAD / 16 + 1) / 2;
#pragma unroll
            for (int s = 0; s < MT; ++s) {
                const Win wn = window_of(s);
                const uint8_t* win = frame + wn.pl * tl.S + wn.off;
                if (warp < 4) stage_window_i8<WS, 0, KCH>(win, rowB, ao + s * Cf::A_BYTES + m * 16);
                else stage_window_i8<WS, KCH, Cf::K_PAD / 16>(win, rowB, ao + s * Cf::A_BYTES + m * 16);
            }
        }
        ptx::fence_proxy_async_smem();   // A and W_c (generic-proxy stores) -> tcgen05.mma operand reads
        __syncthreads();                 // the frame has been read: the next tile may land in it
        if (tid == 0 && t + 1 < t1) load_tile(tile_at(t + 1));
        if (warp == 4 && lane == 0) {
            ptx::tc_fence_after_sync();
            const uint32_t wc_addr = ptx::smem_u32(Wc), a_addr = ptx::smem_u32(ao);
#pragma unroll
            for (int s = 0; s < MT; ++s)
#pragma unroll
                for (int ks = 0; ks < Cf::KSTEPS; ++ks) {
                    const uint64_t adesc = ptx::smem_desc_kmajor_noswz(a_addr + s * Cf::A_BYTES + ks * 2 * Cf::A_LBO, Cf::A_LBO, 128);
                    const uint64_t bdesc = ptx::smem_desc_kmajor_noswz(wc_addr + ks * 2 * Cf::LBO, Cf::LBO, 128);
                    mma_ss_i8<F8>(tmem_d + s * Cf::N_PAD, adesc, bdesc, idesc, ks > 0 ? 1u : 0u);
                }
            ptx::mma_commit(mma_bar);
        }
        ptx::mbar_wait(mma_bar, phase);
        phase ^= 1;
        ptx::tc_fence_after_sync();
        // all 8 warps: warp w and warp w+4 share the TMEM lanes of windows 32(w%4) .. +31 and take half the columns each
#pragma unroll
        for (int s = 0; s < MT; ++s) {
            const Win wn = window_of(s);
            const bool valid = wn.in && wn.pl < q.np && q.wy0 + wn.wyl < g.nwh;
            const uint32_t td = tmem_d + s * Cf::N_PAD + ((uint32_t)((warp & 3) * 32) << 16);
            const float sc = OUT8 ? scale[q.c] : 0.f;
            const uint64_t sc2 = pack_f2(sc, sc);
            uint8_t* owin = ao + wn.pl * So + wn.off * (OUT8 ? 1 : 4);
            constexpr int NCH = Cf::N_PAD / 16, CH_SPLIT = (NCH + 1) / 2;
#pragma unroll
            for (int ch = 0; ch < NCH; ++ch) {
                if ((ch < CH_SPLIT) != (warp < 4)) continue;
                uint32_t v[16];
                ptx::tmem_ld16(td + ch * 16, v);
                ptx::tmem_wait_ld();
                if (valid) {
#pragma unroll
                    for (int e = 0; e < 16; ++e) {
                        const int i = ch * 16 + e;
                        if (i < Cf::N) {
                            const int r = i / WS, k = i % WS;
                            if constexpr (!OUT8) {
                                *reinterpret_cast<uint32_t*>(owin + (r * rowB + k) * 4) = v[e];
                            } else if constexpr (WS % 2 == 0) {
                                if ((k & 1) == 0)
                                    *reinterpret_cast<uint16_t*>(owin + r * rowB + k) = (uint16_t)out_pair<F8>(v[e], v[e + 1], sc, sc2);
                            } else {
                                owin[r * rowB + k] = (uint8_t)(F8 ? to_e4m3x2(v[e], 0u, sc) : requant(v[e], sc));
                            }
                        }
                    }
                }
            }
            ptx::tc_fence_before_sync();
        }
        __syncthreads();
        {   // output planes -> y: every plane strip is one 16-byte aligned run; all threads, 16 bytes each
            constexpr int ES = OUT8 ? 1 : 4;
            uint8_t* dst = static_cast<uint8_t*>(yv) + (((long long)q.b0 * g.C + q.c) * plane + (long long)q.wy0 * WS * g.W) * ES;
            const int per = q.bytes * ES / 16;                  // 16-byte units per plane strip
            const long long dpitch = (long long)g.C * plane * ES;
            for (int p = warp; p < q.np; p += kThreadsI / 32) {    // a warp per plane, four units in flight per lane
                const uint8_t* sp = ao + p * So;
                uint8_t* dp = dst + p * dpitch;
                for (int o = lane; o < per; o += 128) {
                    uint4 val[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u)
                        if (o + 32 * u < per) val[u] = *reinterpret_cast<const uint4*>(sp + (o + 32 * u) * 16);
#pragma unroll
                    for (int u = 0; u < 4; ++u)
                        if (o + 32 * u < per) *reinterpret_cast<uint4*>(dp + (o + 32 * u) * 16) = val[u];
                }
            }
        }
        __syncthreads();   // the A tile of the next iteration overwrites these planes
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 0) ptx::tmem_dealloc(tmem_d, Sm::D_COLS);
}

// cap: windows per tile (128, or 128 * MT for the bulk-copy kernel's sub-tiled form)
bool i8_tiles(const Geom& g, const void* x, const void* y, bool out8, I8Tiles* t, int cap = 128)
{
    if (g.nww > 128 || g.nww < 1) return false;
    t->NSY = g.nwh < cap / g.nww ? g.nwh : cap / g.nww;
    t->NP = t->NSY == g.nwh ? cap / (g.nwh * g.nww) : 1;
    if (t->NP < 1) t->NP = 1;
    if (t->NP > g.B) t->NP = g.B > 0 ? g.B : 1;
    t->nstrips = (g.nwh + t->NSY - 1) / t->NSY;
    t->tiles_per_c = (g.B + t->NP - 1) / t->NP * t->nstrips;
    t->frame_rows = t->NSY * g.w;
    t->S = (t->frame_rows * g.Wp + 15) / 16 * 16;
    if ((t->S / 16) % 2 == 0) t->S += 16;          // 16 * odd: planes start on different banks
    t->ntiles = (long long)g.C * t->tiles_per_c;
    const bool al = reinterpret_cast<uintptr_t>(x) % 4 == 0 && (!out8 || reinterpret_cast<uintptr_t>(y) % 4 == 0);
    // bulk-copy kernel: every plane strip is one contiguous run whose address and size are multiples of 16 bytes
    const bool al16 = reinterpret_cast<uintptr_t>(x) % 16 == 0 && reinterpret_cast<uintptr_t>(y) % 16 == 0;
    const long long plane = (long long)g.H * g.W;
    const bool plain = g.layout == WBMM_LAYOUT_NCHW && g.sh == 0 && g.sw == 0 && g.Hp == g.H && g.Wp == g.W;
    t->flat = !plain ? 0 : ((plane % 4 == 0 && (g.w * g.W) % 4 == 0 && al) ? 4 : 1);
    // (ragged sizes stay on the row form: whole-row copies into an unrotated frame measured slower there, 366 vs 299 us)
    t->rot = (plain || g.layout != WBMM_LAYOUT_NCHW || g.Hp != g.H || g.Wp != g.W) ? 0 : ((g.W % 4 == 0 && al) ? 4 : 1);
    t->runs = t->rot ? 1 : 0;
    t->bulk = (g.layout == WBMM_LAYOUT_NCHW && g.sh == 0 && g.sw == 0 && g.Hp == g.H && g.Wp == g.W && al16 && plane % 16 == 0 &&
               (t->nstrips == 1 || (g.w * g.W) % 16 == 0) && x != nullptr) ? 1 : 0;
    return true;
}

template <int WS, bool OUT8, bool F8>
cudaError_t launch_i8(const Geom& g, const I8Tiles& tl, const int8_t* x, const int8_t* T, const float* scale, void* y,
                      cudaStream_t stream, int* launches)
{
    using Cf = I8Cfg<WS>;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (tl.bulk) {
        const size_t smem = I8Fast<WS, OUT8>::SMEM;
        auto kern = tc_i8_bulk_kernel<WS, OUT8, F8>;
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        const long long cap = (long long)sms * i8_ctas<WS, OUT8>();
        const long long grid = tl.ntiles < cap ? tl.ntiles : cap;
        kern<<<(unsigned)grid, kThreadsI, smem, stream>>>(g, tl, x, T, scale, y);
        ++*launches;
        return cudaGetLastError();
    }
    const size_t smem = Cf::WC_BYTES + Cf::TS_BYTES + Cf::FRAME_BYTES + (OUT8 ? 0 : 128 * Cf::N * 4);
    auto kern = tl.rot ? tc_i8_kernel<WS, OUT8, F8, true> : tc_i8_kernel<WS, OUT8, F8, false>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long grid = tl.ntiles < sms ? tl.ntiles : sms;
    kern<<<(unsigned)grid, kThreadsI, smem, stream>>>(g, tl, x, T, scale, y);
    ++*launches;
    return cudaGetLastError();
}

}  // namespace

bool tc_i8_supported(const Geom& g)
{
    if (g.w != 7 && g.w != 14) return false;
    I8Tiles tl;
    return i8_tiles(g, nullptr, nullptr, false, &tl);
}

cudaError_t tc_i8_forward(const Geom& g, const int8_t* x, const int8_t* T, const float* scale, void* y, cudaStream_t stream,
                          int* launches, int* path, bool fp8)
{
    I8Tiles tl;
    if (!i8_tiles(g, x, y, scale != nullptr, &tl)) return cudaErrorInvalidValue;
    if (tl.bulk && g.w == 7) {          // the sub-tiled form: 4 (8-bit output) or 2 (32-bit output) x 128 windows per tile
        I8Tiles t4;
        const int mt = scale ? i8_mt<7, true>() : i8_mt<7, false>();
        if (i8_tiles(g, x, y, scale != nullptr, &t4, 128 * mt) && t4.bulk) tl = t4;
        else tl.bulk = 0;
    }
    *path = tl.bulk ? WBMM_PATH_TC_TMA : WBMM_PATH_TC_GATHER;
    if (tl.ntiles == 0) return cudaSuccess;
    auto go = [&](auto ws, auto f8) -> cudaError_t {
        constexpr int WS = decltype(ws)::value;
        constexpr bool F8 = decltype(f8)::value;
        return scale ? launch_i8<WS, true, F8>(g, tl, x, T, scale, y, stream, launches)
                     : launch_i8<WS, false, F8>(g, tl, x, T, scale, y, stream, launches);
    };
    using I14 = std::integral_constant<int, 14>;
    using I7 = std::integral_constant<int, 7>;
    if (g.w == 14) return fp8 ? go(I14{}, std::true_type{}) : go(I14{}, std::false_type{});
    return fp8 ? go(I7{}, std::true_type{}) : go(I7{}, std::false_type{});
}

}  // namespace wbmm
