// WBMM forward / dX for FP32 activations on the tensor cores (the paper's own
// precision: "All experiments use FP32 precision", Table 13).
//
// The 5th-generation tensor cores have no fp32 operand type, and one TF32 pass (10-bit mantissa) misses the
// 1e-4 bar.  Instead every fp32 value is split EXACTLY into three bf16 terms
//     v = v1 + v2 + v3 (+ less than 2^-24 |v|),   v1 = bf16(v), v2 = bf16(v - v1), v3 = bf16(v - v1 - v2)
// (each residual is exact in fp32), for the windows and for the table alike, and the product is expanded
// into the six cross terms whose weight is at least 2^-16:
//     x*t ~= x1 t1 + x1 t2 + x2 t1 + x1 t3 + x2 t2 + x3 t1            (dropped terms <= 3 * 2^-24 |x t|)
// -- six tcgen05.mma.kind::f16 passes with fp32 accumulation in TMEM per K-step, smallest terms first.  The same
// block-Toeplitz library as the 16-bit kernel (wbmm_tc_dev.cuh, BulkCfg<14>) is built once per split of
// the table; the three window splits sit side by side in TMEM as the A operands.  Everything else is the
// 16-bit pipeline (wbmm_tc.cu): TMA-engine bulk copies of whole frame images into a ring of slots, window =
// address offset inside the frame (Alg. 1 l.3-4, l.17), weights built in shared memory from the table
// (Eq. 6-8).  fp32 frames are twice the size of the 16-bit ones, so there is no room for a whole tile of output
// beside the input ring: the accumulator is drained in chunks of output rows, each chunk goes through one of two
// small staging buffers laid out as natural image rows and leaves as bulk copies of those row runs (w = 14: four
// window rows = 4 * W * 4 bytes per window row of the tile; w = 7: whole frame images).  (8-byte stores straight
// from the epilogue registers measured 1.4x SLOWER than even in-place staging: 32 sectors per warp instruction.)
//
//   warp 0      producer   cp.async.bulk  x -> ring slot                       FULL / EMPTY
//   warp 1      MMA        NT chunks x 6 terms x KSTEPS tcgen05.mma per tile   A_FULL / A_EMPTY, D_FULL / D_EMPTY
//   warps 2-5   repack     slot -> registers -> split -> tcgen05.st A1|A2|A3;  libraries on a channel change
//   warps 6-9   epilogue   tcgen05.ld D chunk -> staging buffer in image layout                      OUT_FULL / OUT_EMPTY
//   warp 10     store      cp.async.bulk staging -> y (un-partition + crop + inverse roll as address arithmetic)
#include "wbmm_tc.cuh"

#include <cuda.h>

#include <mutex>

#include "wbmm_tc_dev.cuh"
#include "wbmm_tc_f32.cuh"

namespace wbmm {

using namespace tcdev;

namespace {

constexpr int kThreadsF = 352;
constexpr int kSplit = 3;

template <int WS>
struct F32Cfg;

// w = 14: block-Toeplitz library per split; the accumulator is drained in four chunks of output rows
// (4, 4, 4, 2 rows = 64, 64, 64, 32 columns) that rotate through two TMEM buffers, so that the epilogue of one
// chunk overlaps the MMAs of the next.  TMEM: 3 x 112 (A) + 2 x 64 (D) = 464 columns.  Four rows of any even
// width are a multiple of 16 bytes, so a chunk's rows of one window row leave as one bulk copy.
template <>
struct F32Cfg<14> {
    using Bc = BulkCfg<14>;
    static constexpr int A_COLS = Bc::A_COLS;            // 112 per split
    static constexpr int KSTEPS = Bc::KSTEPS;            // 14
    static constexpr int W_BYTES = Bc::WC_BYTES;         // 13824 per split
    static constexpr int LBO = Bc::LBO;
    static constexpr int NT = 4;
    static constexpr int D_BUF = 64;
    static constexpr int CH_ROWS = 4;                    // staging rows per window row and chunk
    static constexpr int TMEM_COLS = 512;
    static constexpr int row0(int q) { return 4 * q; }
    static constexpr int nrows(int q) { return q < 3 ? 4 : 2; }
    static constexpr int ncols(int q) { return nrows(q) * 16; }
    static constexpr int b_off(int ks, int q) { return ((13 - ks) * 16 + row0(q) * 16) * 16; }
    static constexpr int TAB_BYTES = 2 * (((WinCfg<14>::NB + 2) * 2 + 15) / 16 * 16);   // F0 | F1 staging (one split at a time)
};

// w = 7: the full K-major W_c (8 KB) per split, one chunk.  TMEM: 3 x 32 (A) + 2 x 64 (D) = 224 columns.
template <>
struct F32Cfg<7> {
    using Cf = WinCfg<7>;
    static constexpr int A_COLS = Cf::A_COLS;            // 32 per split
    static constexpr int KSTEPS = Cf::KSTEPS;            // 4
    static constexpr int W_BYTES = Cf::WC_BYTES;         // 8192 per split
    static constexpr int LBO = Cf::LBO;
    static constexpr int NT = 1;
    static constexpr int D_BUF = Cf::N_PAD;              // 64
    static constexpr int CH_ROWS = 7;
    static constexpr int TMEM_COLS = 256;
    static constexpr int row0(int) { return 0; }
    static constexpr int nrows(int) { return 7; }
    static constexpr int ncols(int) { return Cf::N_PAD; }
    static constexpr int b_off(int ks, int) { return ks * 2 * LBO; }
    static constexpr int TAB_BYTES = (Cf::NB * 2 + 15) / 16 * 16;
};

template <int WS>
struct F32Smem {
    using Fc = F32Cfg<WS>;
    static constexpr int BAR_BYTES = (2 * kMaxSlots + 10) * 8;      // FULL | EMPTY per slot, A_FULL A_EMPTY D_FULL[2] D_EMPTY[2] OUT_FULL[2] OUT_EMPTY[2]
    static constexpr int FIXED = (kSplit * Fc::W_BYTES + Fc::TAB_BYTES + BAR_BYTES + 127) / 128 * 128;
};

template <int WS, bool GEN>
__global__ void __launch_bounds__(kThreadsF, 1)
tc_f32_kernel(Geom g, TcTiles tl, TilePart part_, int nslot, int out_bytes, const float* __restrict__ x, const float* __restrict__ T,
              float* __restrict__ y, int reverse)
{
    using Cf = WinCfg<WS>;
    using Fc = F32Cfg<WS>;
    using Sm = F32Smem<WS>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* Wc = smem;                                                          // kSplit weight operands
    uint16_t* tab = reinterpret_cast<uint16_t*>(smem + kSplit * Fc::W_BYTES);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kSplit * Fc::W_BYTES + Fc::TAB_BYTES);
    uint8_t* ring = smem + Sm::FIXED;
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t bar0 = ptx::smem_u32(bars);
    auto FULL = [&](int s) { return bar0 + 8u * s; };
    auto EMPTY = [&](int s) { return bar0 + 8u * (kMaxSlots + s); };
    const uint32_t A_FULL = bar0 + 8u * (2 * kMaxSlots), A_EMPTY = A_FULL + 8, D_FULL = A_FULL + 16, D_EMPTY = A_FULL + 32,
                   OUT_FULL = A_FULL + 48, OUT_EMPTY = A_FULL + 64;
    uint8_t* outb = ring + (size_t)nslot * tl.S;             // two staging buffers of out_bytes

    const int wpf = tl.NSY * g.nww;   // windows per frame image
    if (warp == 1) ptx::tmem_alloc(ptx::smem_u32(&tmem_base_s), Fc::TMEM_COLS);
    if (tid >= 64 && tid < 64 + nslot) {
        ptx::mbar_init(FULL(tid - 64), 1);
        ptx::mbar_init(EMPTY(tid - 64), wpf);
        ptx::fence_mbar_init();
    }
    if (tid == 0) {
        ptx::mbar_init(A_FULL, 128);
        ptx::mbar_init(A_EMPTY, 1);
        for (int b = 0; b < 2; ++b) {
            ptx::mbar_init(D_FULL + 8 * b, 1);
            ptx::mbar_init(D_EMPTY + 8 * b, 128);
            ptx::mbar_init(OUT_FULL + 8 * b, 128);
            ptx::mbar_init(OUT_EMPTY + 8 * b, 1);
        }
        ptx::fence_mbar_init();
    }
    // the library builders never write the padding rows / columns: zero the weight operands once
    for (int i = tid; i < (kSplit * Fc::W_BYTES + Fc::TAB_BYTES) / 16; i += kThreadsF) reinterpret_cast<uint4*>(Wc)[i] = make_uint4(0, 0, 0, 0);
    ptx::fence_proxy_async_smem();
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::tc_fence_after_sync();
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const uint32_t tmem = tmem_base_s;
    const uint32_t tmem_d = tmem + kSplit * Fc::A_COLS;
    static_assert(kSplit * Fc::A_COLS + 2 * Fc::D_BUF <= Fc::TMEM_COLS, "TMEM budget");

    const int t0 = part_.start[blockIdx.x], t1 = part_.start[blockIdx.x + 1];
    const int rowB = g.W * 4;
    const long long plane_elems = (long long)g.H * g.W;

    int it_c = t0 / tl.tiles_per_c, it_gb, it_strip;
    {
        const int rem = t0 - it_c * tl.tiles_per_c;
        it_gb = rem / tl.nstrips;
        it_strip = rem - it_gb * tl.nstrips;
    }
    auto tile_decode = [&](int& c, int& b0, int& wy0, int& np_eff, int& rows_eff) {
        c = it_c;
        b0 = it_gb * tl.NP;
        wy0 = it_strip * tl.NSY;
        np_eff = min(tl.NP, g.B - b0);
        rows_eff = GEN ? g.H : min(tl.frame_rows, g.H - wy0 * WS);
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
        if (t1 > t0) {   // pull this CTA's table rows into L2 ahead of the weight builds
            const int c_first = t0 / tl.tiles_per_c, c_last = (t1 - 1) / tl.tiles_per_c;
            const char* base = reinterpret_cast<const char*>(T + (long long)c_first * Cf::NB);
            const long long nbytes = (long long)(c_last - c_first + 1) * Cf::NB * 4;
            for (long long off = lane * 128ll; off < nbytes; off += 32 * 128)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(base + off));
        }
        uint32_t k = 0;
        for (int t = t0; t < t1; ++t) {
            int c, b0, wy0, np_eff, rows_eff;
            tile_decode(c, b0, wy0, np_eff, rows_eff);
            const uint32_t bytes = (uint32_t)rows_eff * rowB;
            for (int p = lane; p < np_eff; p += 32) {
                const uint32_t kk = k + p;
                const int slot = kk % nslot;
                ptx::mbar_wait(EMPTY(slot), ((kk / nslot) & 1) ^ 1);      // every window of the slot's previous image is in TMEM
                ptx::mbar_arrive_expect_tx(FULL(slot), bytes);
                const float* src = x + ((long long)(b0 + p) * g.C + c) * plane_elems + (long long)wy0 * WS * g.W;
                ptx::bulk_g2s(ptx::smem_u32(ring + (size_t)slot * tl.S), src, bytes, FULL(slot));
            }
            k += np_eff;
            __syncwarp();
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer
        // The whole warp walks the loop; one elected lane issues.  The operand descriptors differ from a base
        // value by compile-time constants in their address field (shared-memory addresses fit its 14 bits), so
        // an issue costs one add instead of a descriptor rebuild: 336 instructions of 16-32 tensor cycles each
        // per tile must not wait for their own issue.
        const uint32_t wc_addr = ptx::smem_u32(Wc);
        const uint64_t bdesc0 = ptx::smem_desc_kmajor_noswz(wc_addr, Fc::LBO, 128);
        const uint32_t b_hi = (uint32_t)(bdesc0 >> 32), b_lo = (uint32_t)bdesc0;
        uint32_t lt = 0, nd = 0;       // nd: running count of accumulator chunks (buffer nd & 1, use nd >> 1)
        for (int t = t0; t < t1; ++t, ++lt) {
            ptx::mbar_wait(A_FULL, lt & 1);
#pragma unroll
            for (int q = 0; q < Fc::NT; ++q, ++nd) {
                const uint32_t db = nd & 1;
                ptx::mbar_wait(D_EMPTY + 8 * db, ((nd >> 1) & 1) ^ 1);     // the epilogue has drained this buffer's previous chunk
                ptx::tc_fence_after_sync();
                if (ptx::elect_one()) {
                    const uint32_t idesc = ptx::idesc_f16(1, 128, Fc::ncols(q));
                    const uint32_t dcol = tmem_d + db * Fc::D_BUF;
                    // (window split, table split) pairs, smallest products first
                    constexpr int SA[6] = {2, 1, 0, 1, 0, 0};
                    constexpr int SB[6] = {0, 1, 2, 0, 1, 0};
#pragma unroll
                    for (int term = 0; term < 6; ++term) {
#pragma unroll
                        for (int ks = 0; ks < Fc::KSTEPS; ++ks) {
                            const uint32_t lo = b_lo + (uint32_t)((SB[term] * Fc::W_BYTES + Fc::b_off(ks, q)) >> 4);
                            const uint64_t bdesc = ((uint64_t)b_hi << 32) | lo;
                            ptx::mma_ts(dcol, tmem + SA[term] * Fc::A_COLS + ks * 8, bdesc, idesc, (term | ks) ? 1u : 0u);
                        }
                    }
                    ptx::mma_commit(D_FULL + 8 * db);
                    if (q == Fc::NT - 1) ptx::mma_commit(A_EMPTY);
                }
                __syncwarp();
            }
        }
    } else if (warp < 6) {
        // ------------------------------------------------------------------ repack (+ weight builder)
        const int q = warp & 3;
        const int m = q * 32 + lane;
        const int rt = (warp - 2) * 32 + lane;          // 0..127 among the repack threads
        const int pl = m / wpf, wl = m % wpf;           // image-major
        const int wyl = wl / g.nww, wx = wl % g.nww;
        const int win_off = ((wyl * WS) * g.W + wx * WS) * 4;
        GenAddrF<GEN ? WS : 1> ga;
        if constexpr (GEN) gen_addr_f32<WS>(ga, g, wyl, wx);
        const uint32_t ta = tmem + ((uint32_t)(q * 32) << 16);
        uint32_t k = 0, lt = 0;
        int cur_c = -1;
        for (int t = t0; t < t1; ++t, ++lt) {
            int c, b0, wy0, np_eff, rows_eff;
            tile_decode(c, b0, wy0, np_eff, rows_eff);
            // A is single-buffered: the MMAs of tile lt-1 have completed, so every repack thread has finished tile
            // lt-1 and every fill of its slots has landed -- a slot's previous fill belongs to an earlier tile
            // (nslot >= images per tile), which makes the parity test of this tile's fill unambiguous.
            ptx::mbar_wait(A_EMPTY, (lt & 1) ^ 1);
            if (c != cur_c) {
                // ---- weights of channel c (Eq. 6-8), one operand per bf16 split of the table row
                const float* Tc = T + (long long)c * Cf::NB;
                if constexpr (WS == 14) {
                    uint16_t tv[kSplit][kTabRegs];
#pragma unroll
                    for (int u = 0; u < kTabRegs; ++u) {
                        const int qq = rt + u * 128;
                        uint16_t s3[3] = {0, 0, 0};
                        if (qq < Cf::NB) split3_one(Tc[reverse ? qq : Cf::NB - 1 - qq], s3);
#pragma unroll
                        for (int s = 0; s < kSplit; ++s) tv[s][u] = s3[s];
                    }
#pragma unroll
                    for (int s = 0; s < kSplit; ++s) {
                        if (s > 0) ptx::named_bar_sync(2, 128);      // the previous split's reads of the staging tables are done
                        build_lib14(tv[s], tab, tab + Fc::TAB_BYTES / 4, Wc + s * Fc::W_BYTES, rt);
                    }
                } else {
#pragma unroll 1
                    for (int s = 0; s < kSplit; ++s) {
                        if (s > 0) ptx::named_bar_sync(2, 128);
                        for (int kk = rt; kk < Cf::NB; kk += 128) {
                            uint16_t s3[3];
                            split3_one(Tc[reverse ? Cf::NB - 1 - kk : kk], s3);
                            tab[kk] = s3[s];
                        }
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
                                    if (j < Cf::N) v = tab[(ri - rj + WS - 1) * Cf::TW + (ci - cj + WS - 1)];   // Eq. 7
                                    pk[e >> 1] |= v << ((e & 1) * 16);
                                    ++j;
                                    if (++cj == WS) { cj = 0; ++rj; }
                                }
                            }
                            *reinterpret_cast<uint4*>(Wc + s * Fc::W_BYTES + kc * Cf::LBO + i * 16) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
                        }
                    }
                }
                ptx::fence_proxy_async_smem();
                cur_c = c;
            }
            const bool part = wl < wpf && pl < np_eff;                 // this thread's frame image was loaded
            const bool valid = part && wy0 + wyl < g.nwh;
            const uint32_t kk = k + pl;
            const int slot = kk % nslot;
            if (part) ptx::mbar_wait(FULL(slot), (kk / nslot) & 1);
            const uint8_t* img = ring + (size_t)(part ? slot : 0) * tl.S;
            if constexpr (WS == 14) {
                const uint8_t* p = img + (valid ? win_off : 0);
                const uint32_t rm = valid ? ga.rowmask : 0u;
#pragma unroll
                for (int r = 0; r < 14; ++r) {
                    float f[14];
                    if constexpr (GEN) {
#pragma unroll
                        for (int e = 0; e < 14; ++e) {
                            f[e] = *reinterpret_cast<const float*>(img + ga.rowoff[r] + ga.coloff[e]);
                            if (!((rm >> r) & (ga.colmask >> e) & 1u)) f[e] = 0.f;
                        }
                    } else {
#pragma unroll
                        for (int e2 = 0; e2 < 7; ++e2) {
                            const float2 v2 = *reinterpret_cast<const float2*>(p + 8 * e2);
                            f[2 * e2] = v2.x;
                            f[2 * e2 + 1] = v2.y;
                        }
                        p += rowB;
                    }
                    uint32_t s0[8], s1[8], s2[8];
#pragma unroll
                    for (int e2 = 0; e2 < 7; ++e2) split3(f[2 * e2], f[2 * e2 + 1], s0[e2], s1[e2], s2[e2]);
                    s0[7] = s1[7] = s2[7] = 0u;                            // the two pad positions of the K row
                    ptx::tmem_st8(ta + r * 8, s0);
                    ptx::tmem_st8(ta + Fc::A_COLS + r * 8, s1);
                    ptx::tmem_st8(ta + 2 * Fc::A_COLS + r * 8, s2);
                }
            } else {
                // w = 7: linear in-window order, two positions per column, no row padding
                float f[Cf::N + 1];
                const uint32_t rm = valid ? ga.rowmask : 0u;
#pragma unroll
                for (int r = 0; r < WS; ++r) {
#pragma unroll
                    for (int e = 0; e < WS; ++e) {
                        if constexpr (GEN) {
                            f[r * WS + e] = *reinterpret_cast<const float*>(img + ga.rowoff[r] + ga.coloff[e]);
                            if (!((rm >> r) & (ga.colmask >> e) & 1u)) f[r * WS + e] = 0.f;
                        } else {
                            f[r * WS + e] = *reinterpret_cast<const float*>(img + (valid ? win_off : 0) + r * rowB + e * 4);
                        }
                    }
                }
                f[Cf::N] = 0.f;
                uint32_t s0[Fc::A_COLS], s1[Fc::A_COLS], s2[Fc::A_COLS];
#pragma unroll
                for (int wi = 0; wi < Fc::A_COLS; ++wi) {
                    if (wi < Cf::NW) split3(f[2 * wi], f[2 * wi + 1], s0[wi], s1[wi], s2[wi]);
                    else s0[wi] = s1[wi] = s2[wi] = 0u;
                }
                if (!GEN && !valid) {
#pragma unroll
                    for (int wi = 0; wi < Fc::A_COLS; ++wi) s0[wi] = s1[wi] = s2[wi] = 0u;
                }
#pragma unroll
                for (int ch = 0; ch < Fc::A_COLS / 16; ++ch) {
                    ptx::tmem_st16(ta + ch * 16, s0 + ch * 16);
                    ptx::tmem_st16(ta + Fc::A_COLS + ch * 16, s1 + ch * 16);
                    ptx::tmem_st16(ta + 2 * Fc::A_COLS + ch * 16, s2 + ch * 16);
                }
            }
            ptx::tmem_wait_st();
            if (part) ptx::mbar_arrive(EMPTY(slot));      // (the loads above have returned: their values were stored to TMEM)
            ptx::tc_fence_before_sync();
            ptx::mbar_arrive(A_FULL);
            k += np_eff;
        }
    } else if (warp < 10) {
        // ------------------------------------------------------------------ epilogue (accumulator -> staging)
        const int q = warp & 3;
        const int m = q * 32 + lane;
        const int pl = m / wpf, wl = m % wpf;
        const int wyl = wl / g.nww, wx = wl % g.nww;
        GenAddrF<GEN ? WS : 1> ga;
        if constexpr (GEN) gen_addr_f32<WS>(ga, g, wyl, wx);
        const uint32_t lane_off = (uint32_t)(q * 32) << 16;
        // w = 14: staging rows of this window = (image, window row of the tile) x CH_ROWS natural image rows
        // w = 7:  staging = the tile's frame images (pitch tl.S), the window at its frame position
        const uint32_t st_off = WS == 14 ? (uint32_t)((pl * tl.NSY + wyl) * Fc::CH_ROWS) * rowB + (GEN ? 0u : (uint32_t)wx * WS * 4u)
                                         : (uint32_t)pl * tl.S + (GEN ? 0u : (uint32_t)((wyl * WS) * g.W + wx * WS) * 4u);
        uint32_t nd = 0;
        for (int t = t0; t < t1; ++t) {
            int c, b0, wy0, np_eff, rows_eff;
            tile_decode(c, b0, wy0, np_eff, rows_eff);
            const bool valid = wl < wpf && pl < np_eff && wy0 + wyl < g.nwh;
#pragma unroll
            for (int qc = 0; qc < Fc::NT; ++qc, ++nd) {
                const uint32_t db = nd & 1;
                uint32_t v[Fc::D_BUF];
                ptx::mbar_wait(D_FULL + 8 * db, (nd >> 1) & 1);
                ptx::tc_fence_after_sync();
                const uint32_t td = tmem_d + db * Fc::D_BUF + lane_off;
#pragma unroll
                for (int ch = 0; ch < Fc::ncols(qc) / 16; ++ch) ptx::tmem_ld16(td + ch * 16, v + ch * 16);
                ptx::tmem_wait_ld();
                ptx::tc_fence_before_sync();
                ptx::mbar_arrive(D_EMPTY + 8 * db);
                ptx::mbar_wait(OUT_EMPTY + 8 * db, ((nd >> 1) & 1) ^ 1);     // the copy engine has read this buffer's previous chunk out
                uint8_t* stg = outb + (size_t)db * out_bytes + st_off;
                if (valid) {
                    if constexpr (WS == 14) {
#pragma unroll
                        for (int rr = 0; rr < Fc::nrows(qc); ++rr) {
                            uint8_t* p = stg + rr * rowB;
                            if constexpr (GEN) {
#pragma unroll
                                for (int e = 0; e < 14; ++e)
                                    if ((ga.colmask >> e) & 1u) *reinterpret_cast<uint32_t*>(p + ga.coloff[e]) = v[rr * 16 + e];
                            } else {
#pragma unroll
                                for (int e2 = 0; e2 < 7; ++e2)
                                    *reinterpret_cast<uint2*>(p + 8 * e2) = make_uint2(v[rr * 16 + 2 * e2], v[rr * 16 + 2 * e2 + 1]);
                            }
                        }
                    } else {
#pragma unroll
                        for (int r = 0; r < WS; ++r) {
#pragma unroll
                            for (int e = 0; e < WS; ++e) {
                                if constexpr (GEN) {
                                    if ((ga.rowmask >> r) & (ga.colmask >> e) & 1u)
                                        *reinterpret_cast<uint32_t*>(stg + ga.rowoff[r] + ga.coloff[e]) = v[r * WS + e];
                                } else {
                                    *reinterpret_cast<uint32_t*>(stg + r * rowB + e * 4) = v[r * WS + e];
                                }
                            }
                        }
                    }
                }
                ptx::fence_proxy_async_smem();      // generic-proxy writes -> the bulk store's async-proxy reads
                ptx::mbar_arrive(OUT_FULL + 8 * db);
            }
        }
    } else {
        // ------------------------------------------------------------------ store
        uint32_t nd = 0;
        for (int t = t0; t < t1; ++t) {
            int c, b0, wy0, np_eff, rows_eff;
            tile_decode(c, b0, wy0, np_eff, rows_eff);
#pragma unroll
            for (int qc = 0; qc < Fc::NT; ++qc, ++nd) {
                const uint32_t db = nd & 1;
                ptx::mbar_wait(OUT_FULL + 8 * db, (nd >> 1) & 1);
                const uint32_t src0 = ptx::smem_u32(outb + (size_t)db * out_bytes);
                if constexpr (WS == 14) {
                    // one run of the chunk's rows per (image, window row of the tile); rolled rows -> up to two runs of image rows
                    const int nr = Fc::nrows(qc);
                    for (int i = lane; i < np_eff * tl.NSY; i += 32) {
                        const int p = i / tl.NSY, wyl = i - p * tl.NSY;
                        if (wy0 + wyl >= g.nwh) continue;
                        float* pl0 = y + ((long long)(b0 + p) * g.C + c) * plane_elems;
                        const uint32_t src = src0 + (uint32_t)(i * Fc::CH_ROWS) * rowB;
                        const int R0 = (wy0 + wyl) * WS + Fc::row0(qc);
                        if constexpr (GEN) {
                            const StripRuns sr = strip_runs(g, R0, nr);
                            if (sr.nA > 0) ptx::bulk_s2g(pl0 + (long long)sr.a0 * g.W, src, (uint32_t)sr.nA * rowB);
                            if (sr.nB > 0) ptx::bulk_s2g(pl0, src + sr.n1 * rowB, (uint32_t)sr.nB * rowB);
                        } else {
                            ptx::bulk_s2g(pl0 + (long long)R0 * g.W, src, (uint32_t)nr * rowB);
                        }
                    }
                } else {
                    const uint32_t bytes = (uint32_t)rows_eff * rowB;
                    for (int p = lane; p < np_eff; p += 32) {
                        float* dst = y + ((long long)(b0 + p) * g.C + c) * plane_elems + (long long)wy0 * WS * g.W;
                        ptx::bulk_s2g(dst, src0 + (uint32_t)p * tl.S, bytes);
                    }
                }
                ptx::bulk_commit();
                ptx::bulk_wait_read<0>();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(OUT_EMPTY + 8 * db);
            }
        }
        ptx::bulk_wait_all<0>();
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem, Fc::TMEM_COLS);
}

// Tiles as in tc_tiles (wbmm_tc.cu) with 4-byte elements, shrunk until a tile fits the ring beside the two
// staging buffers: fewer images per tile, then fewer window rows per strip (half-filled MMA tiles).
template <int WS>
int f32_out_bytes(const Geom& g, const TcTiles& t)
{
    const long long b = WS == 14 ? (long long)t.NP * t.NSY * F32Cfg<WS>::CH_ROWS * g.W * 4 : (long long)t.NP * t.S;
    return (int)((b + 127) / 128 * 128);
}

template <int WS>
bool f32_tiles(const Geom& g, TcTiles* t, int* nslot)
{
    const int wpp = g.nwh * g.nww;
    if (g.nww > 128) return false;
    if (wpp <= 128) {
        t->NSY = g.nwh;
        t->NP = 128 / wpp;
        if (t->NP > 64) t->NP = 64;
        if (t->NP > g.B) t->NP = g.B;
    } else {
        t->NP = 1;
        t->NSY = 128 / g.nww;
    }
    long long room = 0;
    for (;;) {
        t->frame_rows = t->NSY * g.w;
        int s16 = (t->frame_rows * g.Wp * 4 + 15) / 16;
        if (s16 % 2 == 0) ++s16;
        t->S = s16 * 16;
        room = 227ll * 1024 - 1024 - F32Smem<WS>::FIXED - 2ll * f32_out_bytes<WS>(g, *t);
        if ((long long)t->NP * t->S <= room) break;
        if (t->NP > 1) t->NP = (t->NP + 1) / 2;
        else if (t->NSY > 1) t->NSY = (t->NSY + 1) / 2;
        else return false;
    }
    t->nstrips = (g.nwh + t->NSY - 1) / t->NSY;
    t->ngb = (g.B + t->NP - 1) / t->NP;
    t->tiles_per_c = t->ngb * t->nstrips;
    t->ntiles = (long long)g.C * t->tiles_per_c;
    long long n = room / t->S;
    if (n > 2 * t->NP + 2) n = 2 * t->NP + 2;       // two tiles in flight are plenty
    if (n > kMaxSlots) n = kMaxSlots;
    *nslot = (int)n;
    return n >= t->NP && t->ntiles <= 0x3fffffffll;
}

// 0 = not servable, 1 = aligned form, 2 = general form (shift / ragged, whole images)
template <int WS>
int f32_mode(const Geom& g, const TcTiles& tl, const void* x, const void* y)
{
    if (g.layout != WBMM_LAYOUT_NCHW) return 0;
    if (reinterpret_cast<uintptr_t>(x) % 16 != 0 || reinterpret_cast<uintptr_t>(y) % 16 != 0) return 0;
    if (((long long)g.H * g.W * 4) % 16 != 0) return 0;                 // every plane starts on a 16-byte boundary
    const bool plain = g.sh == 0 && g.sw == 0 && g.H == g.Hp && g.W == g.Wp;
    if (plain && (tl.nstrips == 1 || ((long long)tl.frame_rows * g.W * 4) % 16 == 0)) return 1;   // (w = 14: W is even, 4-row runs are 16-byte multiples)
    // general form: whole images in natural layout; w = 14 stores runs of single image rows
    return (tl.nstrips == 1 && (WS == 7 || g.W % 4 == 0)) ? 2 : 0;
}

template <int WS, bool GEN>
cudaError_t launch_f32(const Geom& g, const TcTiles& tl, int nslot, const void* x, const void* T, void* y, bool reverse,
                       cudaStream_t s)
{
    auto k = tc_f32_kernel<WS, GEN>;
    const int out_bytes = f32_out_bytes<WS>(g, tl);
    const size_t smem = (size_t)F32Smem<WS>::FIXED + (size_t)nslot * tl.S + 2 * (size_t)out_bytes;
    static SmemOptIn smem_state;
    static std::mutex mu;
    static TilePart cached;
    static long long key_n = -1;
    static int key_tpc = -1, key_grid = -1, cached_used = 0;
    int grid = (int)(tl.ntiles < num_sms() ? tl.ntiles : num_sms());
    if (grid > kMaxGrid) grid = kMaxGrid;
    TilePart part;
    {
        std::lock_guard<std::mutex> lock(mu);
        cudaError_t e = ensure_dynamic_smem(reinterpret_cast<const void*>(k), smem, &smem_state);
        if (e != cudaSuccess) return e;
        if (key_n != tl.ntiles || key_tpc != tl.tiles_per_c || key_grid != grid) {
            cached_used = partition_tiles(tl, grid, 0.3, &cached);
            key_n = tl.ntiles; key_tpc = tl.tiles_per_c; key_grid = grid;
        }
        part = cached;
        grid = cached_used;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(kThreadsF);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k, g, tl, part, nslot, out_bytes, (const float*)x, (const float*)T, (float*)y, reverse ? 1 : 0);
}

}  // namespace

bool tc_f32_supported(const Geom& g, const void* x, const void* y)
{
    if (g.w != 7 && g.w != 14) return false;
    TcTiles tl;
    int nslot;
    if (!(g.w == 7 ? f32_tiles<7>(g, &tl, &nslot) : f32_tiles<14>(g, &tl, &nslot))) return false;
    return (g.w == 7 ? f32_mode<7>(g, tl, x, y) : f32_mode<14>(g, tl, x, y)) != 0;
}

cudaError_t tc_f32_forward(const Geom& g, const void* x, const void* T, void* y, bool reverse, cudaStream_t stream,
                           int* launches)
{
    TcTiles tl;
    int nslot;
    if (!(g.w == 7 ? f32_tiles<7>(g, &tl, &nslot) : f32_tiles<14>(g, &tl, &nslot))) return cudaErrorNotSupported;
    if (tl.ntiles == 0) return cudaSuccess;
    const int mode = g.w == 7 ? f32_mode<7>(g, tl, x, y) : f32_mode<14>(g, tl, x, y);
    if (mode == 0) return cudaErrorNotSupported;
    *launches += 1;
    if (g.w == 7)
        return mode == 2 ? launch_f32<7, true>(g, tl, nslot, x, T, y, reverse, stream)
                         : launch_f32<7, false>(g, tl, nslot, x, T, y, reverse, stream);
    return mode == 2 ? launch_f32<14, true>(g, tl, nslot, x, T, y, reverse, stream)
                     : launch_f32<14, false>(g, tl, nslot, x, T, y, reverse, stream);
}

}  // namespace wbmm
