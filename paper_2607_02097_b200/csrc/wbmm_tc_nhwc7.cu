// WBMM forward / dX for NHWC activations, w = 7, in ONE pass straight from NHWC memory (BASELINE.json north_star (a),
// configs[3]): no transposition kernels, no scratch, warp-specialised like the NCHW kernel (wbmm_tc.cu).
//
// In NHWC the channel -- the BATCH index of the per-channel GEMM (Alg. 1 l.15) -- is the contiguous
// axis, and the copy engine moves a box of [pixels][CGT channels] at ~13 GB/s per SM when a pixel is 16 bytes, 18-24
// at 32 bytes and 30+ at 64 bytes (measured).  A tile is therefore a GROUP of CGT = 32 (16, 8)
// channels x 128 / NOCT windows, NOCT = CGT / 8 octets of channels:
//
//   * one 4-D tensor-map box {CGT channels, W', 7 rows, 1 image} per window row of a frame image lands as
//     [row][column][CGT channels] with the 64-byte (32-byte) swizzle (padding rows / columns are zero-filled by the
//     copy engine on the way in and clipped on the way out: Eq. 4-5); the window is an address
//     offset inside the strip (Alg. 1 l.3-4, l.17);
//   * TMEM lane m = octet * (128 / NOCT) + window: the repack warp of a lane quarter reads the 16 bytes of ITS octet
//     of each pixel with one load (conflict-free under the swizzle), separates the eight channels with byte permutes
//     and writes the eight A operands of its lanes (8 x 32 columns) -- the strip is read once for the whole group;
//   * channel c = 8 * octet + i is one group of 4 tcgen05.mma over A operand i (two input window rows per K = 16
//     step, N = 64 = 8 padded output rows); its accumulator is meaningful in the lanes of its octet only.  The weights
//     are the 13 distinct 7 x 7 Toeplitz blocks of W_c (Eq. 6-8 depend on the rows only through ri - rj), one
//     128-byte core matrix each: 1.9 KB per channel, all CGT live in shared memory;
//   * the epilogue warps of an octet drain its channels, keep the first channel of a pair in registers, interleave it
//     with the second and write 32 bits per pixel back IN PLACE; the store warp moves a finished strip out with one
//     tensor-map store and hands its slot back to the producer.
//
// w = 14 has no such kernel: one group of 8 channels x 128 windows x 196 positions is 400 KB, the accumulators of 8
// channels are 1792 TMEM columns, and eight 13.5 KB weight libraries take 108 KB -- see DESIGN.md section 7.2.
// Shifted NHWC maps keep the transposition route as well (a box cannot wrap).
#include "wbmm_tc.cuh"

#include <cuda.h>

#include <cstring>
#include <mutex>

#include "wbmm_tc_dev.cuh"

namespace wbmm {

using namespace tcdev;

namespace {

constexpr int kThreadsP = 352;
constexpr int WS = 7;
constexpr int kACols = 32;                   // TMEM columns of one A operand: 4 K-steps x (row 2s+1 | row 2s) x 8 values
constexpr int kDCols = 64;                   // accumulator columns: 8 padded output rows x 8 padded positions
constexpr int kLibBlocks = 15;               // one padding block, the 13 Toeplitz blocks dr = -6..6, one padding block
constexpr int kLibBytes = kLibBlocks * 128;  // per channel
constexpr int kNB = 169;

template <int NOCT>
struct PipeCfg {
    static constexpr int CGT = 8 * NOCT;                              // channels per group
    static constexpr int PX = 16 * NOCT;                              // bytes per pixel in the frame
    static constexpr int WT = 128 / NOCT;                             // windows per tile
    static constexpr uint32_t SWZ = NOCT == 4 ? 3u : (NOCT == 2 ? 1u : 0u);   // 16-byte chunk bits XORed with address bits 7..
    static constexpr int LIB = CGT * kLibBytes + 256;                 // + readable zeros behind the last library
    static constexpr int BAR_BYTES = (3 * kMaxSlots + 12) * 8;        // FULL | EMPTY | OUT_FULL per slot, A_FULL[2] A_EMPTY[2] D_FULL[4] D_EMPTY[4]
    static constexpr int FIXED = (LIB + BAR_BYTES + 1023) / 1024 * 1024;
};

// byte offset of 16-byte chunk `oct` of pixel p under the tensor map's swizzle (slot bases are 1024-byte aligned)
template <int NOCT>
__device__ __forceinline__ uint32_t px_addr(uint32_t p, uint32_t oct)
{
    const uint32_t a = p * PipeCfg<NOCT>::PX + 16u * oct;
    return a ^ (((a >> 7) & PipeCfg<NOCT>::SWZ) << 4);
}

template <bool BF16, int NOCT>
__global__ void __launch_bounds__(kThreadsP, 1)
tc_nhwc7_kernel(Geom g, TcTiles tl, TilePart part_, int nslot, const __grid_constant__ CUtensorMap mx,
                const __grid_constant__ CUtensorMap my, const uint16_t* __restrict__ T, int reverse)
{
    using Pc = PipeCfg<NOCT>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* lib = smem;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Pc::LIB);
    uint8_t* ring = smem + Pc::FIXED;
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t bar0 = ptx::smem_u32(bars);
    auto FULL = [&](int s) { return bar0 + 8u * s; };
    auto EMPTY = [&](int s) { return bar0 + 8u * (kMaxSlots + s); };
    auto OUT_FULL = [&](int s) { return bar0 + 8u * (2 * kMaxSlots + s); };
    const uint32_t A_FULL = bar0 + 8u * (3 * kMaxSlots), A_EMPTY = A_FULL + 16, D_FULL = A_FULL + 32, D_EMPTY = A_FULL + 64;

    // a slot holds ONE window row of one frame image for the whole channel group: 7 rows x W' pixels x CGT channels
    const int spi = tl.NSY;                                   // slots (window rows) per frame image
    const int wpf = tl.NSY * g.nww;                           // windows per frame image
    if (warp == 1) ptx::tmem_alloc(ptx::smem_u32(&tmem_base_s), 512);
    if (tid >= 64 && tid < 64 + nslot) {
        ptx::mbar_init(FULL(tid - 64), 1);
        ptx::mbar_init(EMPTY(tid - 64), 1);
        ptx::mbar_init(OUT_FULL(tid - 64), g.nww * NOCT);     // every lane that owns a window of the row, in every octet
        ptx::fence_mbar_init();
    }
    if (tid == 0) {
        // the A operands are written and consumed in two halves of four channels per octet (i = 0..3 | 4..7), each
        // half with its own buffer: the repack of one half overlaps the MMAs / epilogue of the other
        for (int h = 0; h < 2; ++h) {
            ptx::mbar_init(A_FULL + 8 * h, 128);
            ptx::mbar_init(A_EMPTY + 8 * h, 1);
        }
        // Four accumulators; channel number nd (running over tiles) uses accumulator nd & 3, which therefore always
        // belongs to the same octet of channels: one group of epilogue warps walks ALL phases of its barriers (a
        // waiter that skipped phases, or shared a barrier with a slower group, could mistake one parity for another).
        for (int b = 0; b < 4; ++b) {
            ptx::mbar_init(D_FULL + 8 * b, 1);
            ptx::mbar_init(D_EMPTY + 8 * b, 128 / NOCT);      // the lanes of the accumulator's octet
        }
        ptx::fence_mbar_init();
        ptx::tma_prefetch_desc(&mx);
        ptx::tma_prefetch_desc(&my);
    }
    for (int i = tid; i < Pc::LIB / 16; i += kThreadsP) reinterpret_cast<uint4*>(lib)[i] = make_uint4(0, 0, 0, 0);
    ptx::fence_proxy_async_smem();
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::tc_fence_after_sync();
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const uint32_t tmem = tmem_base_s;
    const uint32_t tmem_d = tmem + 8 * kACols;       // 8 A operands (256 columns), then four accumulators (256 columns)

    const int t0 = part_.start[blockIdx.x], t1 = part_.start[blockIdx.x + 1];

    auto tile_decode = [&](int t, int& cg, int& b0, int& wy0, int& np_eff) {
        cg = t / tl.tiles_per_c;
        const int rem = t - cg * tl.tiles_per_c;
        const int gb = rem / tl.nstrips, strip = rem - gb * tl.nstrips;
        b0 = gb * tl.NP;
        wy0 = strip * tl.NSY;
        np_eff = min(tl.NP, g.B - b0);
    };

    // lane m = octet * WT + window of the tile; window = image-major (pl, window row wyl, wx)
    auto lane_window = [&](int m, int& oct, int& pl, int& wyl, int& wx) {
        oct = m / Pc::WT;
        const int widx = m - oct * Pc::WT;
        pl = widx / wpf;
        const int wl = widx - pl * wpf;
        wyl = wl / g.nww;
        wx = wl - wyl * g.nww;
    };

    // The libraries of a channel group (Eq. 6-8): block 1 + (dr + 6), row ci, 8 values cj = 0..7,
    //     Z[dr][ci][cj] = T[c, (dr + 6) * 13 + (ci - cj + 6)], zero for ci = 7 or cj = 7.
    // One thread per (channel, dr): the 13 table entries of that row offset are loaded once (all loads in flight
    // together) and shifted through the seven rows of the block.
    auto build_lib = [&](int cg, int first, int nthreads) {
        for (int id = first; id < Pc::CGT * 13; id += nthreads) {
            const int ch = id / 13, d = id - ch * 13;
            const uint16_t* Tc = T + (long long)(cg * Pc::CGT + ch) * kNB;
            uint32_t e[13];
#pragma unroll
            for (int j = 0; j < 13; ++j) {
                const int idx = d * 13 + j;
                e[j] = Tc[reverse ? kNB - 1 - idx : idx];
            }
            uint8_t* blk = lib + ch * kLibBytes + (d + 1) * 128;
#pragma unroll
            for (int ci = 0; ci < 7; ++ci) {
                uint32_t pk[4] = {0u, 0u, 0u, 0u};
#pragma unroll
                for (int cj = 0; cj < 7; ++cj) pk[cj >> 1] |= e[ci - cj + 6] << ((cj & 1) * 16);
                *reinterpret_cast<uint4*>(blk + ci * 16) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
            }
        }
    };
    // the first group's libraries: every warp but the producer, while the first boxes are on their way
    int first_cg = -1;
    if (t0 < t1) first_cg = t0 / tl.tiles_per_c;
    if (warp >= 1 && first_cg >= 0) {
        build_lib(first_cg, tid - 32, kThreadsP - 32);
        ptx::fence_proxy_async_smem();
        ptx::named_bar_sync(1, kThreadsP - 32);
    }

    if (warp == 0) {
        // ------------------------------------------------------------------ producer: one box per window row of an image
        uint32_t k = 0;
        for (int t = t0; t < t1; ++t) {
            int cg, b0, wy0, np_eff;
            tile_decode(t, cg, b0, wy0, np_eff);
            for (int i = lane; i < np_eff * spi; i += 32) {
                const int p = i / spi, wyl = i - p * spi;
                const uint32_t kk = k + i;
                const int slot = kk % nslot;
                ptx::mbar_wait(EMPTY(slot), ((kk / nslot) & 1) ^ 1);      // the store warp has read the slot's previous strip out
                ptx::mbar_arrive_expect_tx(FULL(slot), (uint32_t)(WS * g.Wp) * Pc::PX);
                ptx::tma_load_4d(ptx::smem_u32(ring + (size_t)slot * tl.S), &mx, cg * Pc::CGT, 0, (wy0 + wyl) * WS, b0 + p, FULL(slot));
            }
            k += np_eff * spi;
            __syncwarp();
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer (whole warp walks, one lane issues)
        const uint32_t lib_addr = ptx::smem_u32(lib);
        constexpr uint32_t idesc = ptx::idesc_f16(BF16 ? 1 : 0, 128, kDCols);
        uint32_t lt = 0, nd = 0;
        for (int t = t0; t < t1; ++t, ++lt) {
#pragma unroll 1
            for (int i = 0; i < 8; ++i) {
                const int h = i >> 2;
                if ((i & 3) == 0) ptx::mbar_wait(A_FULL + 8 * h, lt & 1);
#pragma unroll
                for (int oct = 0; oct < NOCT; ++oct, ++nd) {
                    const uint32_t db = nd & 3;
                    ptx::mbar_wait(D_EMPTY + 8 * db, ((nd >> 2) & 1) ^ 1);     // this accumulator's previous channel has been drained
                    ptx::tc_fence_after_sync();
                    if (ptx::elect_one()) {
                        // K-step s = input rows (2s+1 | 2s): B chunk 0 = blocks (ri - 2s - 1 + 6) + 1, chunk 1 = the next
                        // block (row 2s), for the 8 output row groups ri = 0..7: consecutive 128-byte core matrices
                        const uint64_t bd0 = ptx::smem_desc_kmajor_noswz(lib_addr + (oct * 8 + i) * kLibBytes, 128, 128);
                        const uint32_t b_hi = (uint32_t)(bd0 >> 32), b_lo = (uint32_t)bd0;
#pragma unroll
                        for (int s = 0; s < 4; ++s) {
                            const uint64_t bdesc = ((uint64_t)b_hi << 32) | (b_lo + (uint32_t)(((6 - 2 * s) * 128) >> 4));
                            ptx::mma_ts(tmem_d + db * kDCols, tmem + i * kACols + s * 8, bdesc, idesc, s > 0 ? 1u : 0u);
                        }
                        ptx::mma_commit(D_FULL + 8 * db);
                        if ((i & 3) == 3 && oct == NOCT - 1) ptx::mma_commit(A_EMPTY + 8 * h);
                    }
                    __syncwarp();
                }
            }
        }
    } else if (warp < 6) {
        // ------------------------------------------------------------------ repack (+ weight builder)
        const int q = warp & 3;
        const int m = q * 32 + lane;
        const int rt = (warp - 2) * 32 + lane;
        int oct, pl, wyl, wx;
        lane_window(m, oct, pl, wyl, wx);
        const uint32_t p0 = (uint32_t)(wx * WS);            // first pixel of the window inside its strip
        const uint32_t ta = tmem + ((uint32_t)(q * 32) << 16);
        // W' a multiple of 8 pixels: a row step does not change the swizzle phase, so the 7 column offsets of the
        // window are per-thread constants and a pixel address is one add
        const bool fastw = g.Wp % 8 == 0;
        uint32_t coff[WS];
#pragma unroll
        for (int c = 0; c < WS; ++c) coff[c] = px_addr<NOCT>(p0 + (uint32_t)c, (uint32_t)oct);
        const uint32_t rowB = (uint32_t)g.Wp * Pc::PX;
        uint32_t k = 0, lt = 0;
        int cur_cg = first_cg;
        for (int t = t0; t < t1; ++t, ++lt) {
            int cg, b0, wy0, np_eff;
            tile_decode(t, cg, b0, wy0, np_eff);
            // Half 0 of the A operands is free once the MMAs of half 0 of tile lt-1 have completed.  The MMA warp issues in
            // order, so every repack thread has then finished tile lt-1's half 0 -- it had waited for all of that tile's
            // fills: a slot's previous fill belongs to an earlier tile (nslot >= slots per tile), which makes the parity
            // test of this tile's fill unambiguous.
            ptx::mbar_wait(A_EMPTY, (lt & 1) ^ 1);
            if (cg != cur_cg) {
                // half 1 of the previous tile still reads the old libraries until its MMAs have completed
                ptx::mbar_wait(A_EMPTY + 8, (lt & 1) ^ 1);
                build_lib(cg, rt, 128);
                ptx::fence_proxy_async_smem();
                cur_cg = cg;
            }
            const bool part = pl < np_eff;
            const bool valid = part && wy0 + wyl < g.nwh;
            const uint32_t kk = k + pl * spi + wyl;
            const int slot = kk % nslot;
            if (part) ptx::mbar_wait(FULL(slot), (kk / nslot) & 1);
            const uint8_t* strip = ring + (size_t)(part ? slot : 0) * tl.S;
            // the octet's channels in two halves (4 channels = 8 bytes of each pixel); rows in K-step order (row 2s+1 | row 2s)
#pragma unroll 1
            for (int hh = 0; hh < 2; ++hh) {
                if (hh == 1) ptx::mbar_wait(A_EMPTY + 8, (lt & 1) ^ 1);
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    uint32_t a[4][8];                   // [channel of the half][column of the K-step]
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int r = 2 * s + 1 - h;    // h = 0: row 2s+1 (columns 0-3), h = 1: row 2s (columns 4-7)
                        if (r < WS) {
                            uint2 e[WS];
#pragma unroll
                            for (int c = 0; c < WS; ++c)
                                e[c] = *reinterpret_cast<const uint2*>(strip + 8 * hh + (fastw ? (uint32_t)r * rowB + coff[c]
                                                                                               : px_addr<NOCT>(p0 + (uint32_t)(r * g.Wp + c), (uint32_t)oct)));
#pragma unroll
                            for (int kp = 0; kp < 2; ++kp) {
#pragma unroll
                                for (int c2 = 0; c2 < 4; ++c2) {
                                    const uint32_t w0 = kp == 0 ? e[2 * c2].x : e[2 * c2].y;
                                    uint32_t w1 = 0u;
                                    if (2 * c2 + 1 < WS) w1 = kp == 0 ? e[2 * c2 + 1].x : e[2 * c2 + 1].y;
                                    a[2 * kp][4 * h + c2] = valid ? __byte_perm(w0, w1, 0x5410) : 0u;
                                    a[2 * kp + 1][4 * h + c2] = valid ? __byte_perm(w0, w1, 0x7632) : 0u;
                                }
                            }
                        } else {
#pragma unroll
                            for (int ch = 0; ch < 4; ++ch)
#pragma unroll
                                for (int c2 = 0; c2 < 4; ++c2) a[ch][4 * h + c2] = 0u;
                        }
                    }
#pragma unroll
                    for (int ch = 0; ch < 4; ++ch) ptx::tmem_st8(ta + (4 * hh + ch) * kACols + s * 8, a[ch]);
                }
                ptx::tmem_wait_st();
                ptx::tc_fence_before_sync();
                ptx::mbar_arrive(A_FULL + 8 * hh);
            }
            k += np_eff * spi;
        }
    } else if (warp < 10) {
        // ------------------------------------------------------------------ epilogue (in place)
        const int q = warp & 3;
        const int m = q * 32 + lane;
        int oct, pl, wyl, wx;
        lane_window(m, oct, pl, wyl, wx);
        const uint32_t p0 = (uint32_t)(wx * WS);
        const uint32_t lane_off = (uint32_t)(q * 32) << 16;
        const bool fastw = g.Wp % 8 == 0;                   // (see the repack warps)
        uint32_t coff[WS];
#pragma unroll
        for (int c = 0; c < WS; ++c) coff[c] = px_addr<NOCT>(p0 + (uint32_t)c, (uint32_t)oct);
        const uint32_t rowB = (uint32_t)g.Wp * Pc::PX;
        uint32_t k = 0, nd = 0;
        for (int t = t0; t < t1; ++t) {
            int cg, b0, wy0, np_eff;
            tile_decode(t, cg, b0, wy0, np_eff);
            const bool part = pl < np_eff;
            const bool valid = part && wy0 + wyl < g.nwh;
            const uint32_t kk = k + pl * spi + wyl;
            const int slot = kk % nslot;
            uint8_t* strip = ring + (size_t)(part ? slot : 0) * tl.S;
#pragma unroll 1
            for (int kp = 0; kp < 4; ++kp) {
                uint32_t keep[28];                   // channel 2kp: packed pairs (c0c1, c2c3, c4c5, c6 .) of the 7 output rows
#pragma unroll
                for (int half = 0; half < 2; ++half) {
                    // this octet's channel i = 2kp + half is channel number nd of the MMA warp's order (i outer, octet inner)
                    const uint32_t ndc = nd + (uint32_t)((2 * kp + half) * NOCT + oct);
                    const uint32_t db = ndc & 3;
                    uint32_t v[kDCols];
                    ptx::mbar_wait(D_FULL + 8 * db, (ndc >> 2) & 1);
                    ptx::tc_fence_after_sync();
                    const uint32_t td = tmem_d + db * kDCols + lane_off;
#pragma unroll
                    for (int chk = 0; chk < kDCols / 16; ++chk) ptx::tmem_ld16(td + chk * 16, v + chk * 16);
                    ptx::tmem_wait_ld();
                    ptx::tc_fence_before_sync();
                    ptx::mbar_arrive(D_EMPTY + 8 * db);
                    if (half == 0) {
#pragma unroll
                        for (int r = 0; r < WS; ++r)
#pragma unroll
                            for (int c2 = 0; c2 < 4; ++c2) keep[r * 4 + c2] = pack2<BF16>(v[r * 8 + 2 * c2], v[r * 8 + 2 * c2 + 1]);
                    } else if (valid) {
#pragma unroll
                        for (int r = 0; r < WS; ++r) {
#pragma unroll
                            for (int c2 = 0; c2 < 4; ++c2) {
                                const uint32_t pa = keep[r * 4 + c2], pb = pack2<BF16>(v[r * 8 + 2 * c2], v[r * 8 + 2 * c2 + 1]);
                                const uint32_t pix = p0 + (uint32_t)(r * g.Wp + 2 * c2);
                                const uint32_t o0 = fastw ? (uint32_t)r * rowB + coff[2 * c2] : px_addr<NOCT>(pix, (uint32_t)oct);
                                *reinterpret_cast<uint32_t*>(strip + o0 + 4 * kp) = __byte_perm(pa, pb, 0x5410);
                                if (2 * c2 + 1 < WS) {
                                    const uint32_t o1 = fastw ? (uint32_t)r * rowB + coff[2 * c2 + 1] : px_addr<NOCT>(pix + 1, (uint32_t)oct);
                                    *reinterpret_cast<uint32_t*>(strip + o1 + 4 * kp) = __byte_perm(pa, pb, 0x7632);
                                }
                            }
                        }
                    }
                }
            }
            nd += 8 * NOCT;
            ptx::fence_proxy_async_smem();      // generic-proxy writes -> the tensor-map store's async-proxy reads
            if (part) ptx::mbar_arrive(OUT_FULL(slot));
            k += np_eff * spi;
        }
    } else {
        // ------------------------------------------------------------------ store
        // Lane (slot mod 32) owns a slot: it stores every fill of it, in order, and hands it back once the copy engine
        // has read it (one owner per barrier: the parity test of fill n is only made after fill n-1 was seen complete).
        uint32_t k = 0;
        for (int t = t0; t < t1; ++t) {
            int cg, b0, wy0, np_eff;
            tile_decode(t, cg, b0, wy0, np_eff);
            for (int i = 0; i < np_eff * spi; ++i) {
                const uint32_t kk = k + i;
                const int slot = kk % nslot;
                if ((slot & 31) != lane) continue;
                const int p = i / spi, wyl = i - p * spi;
                ptx::mbar_wait(OUT_FULL(slot), (kk / nslot) & 1);
                ptx::tma_store_4d(&my, cg * Pc::CGT, 0, (wy0 + wyl) * WS, b0 + p, ptx::smem_u32(ring + (size_t)slot * tl.S));
                ptx::bulk_commit();
                ptx::bulk_wait_read<0>();
                ptx::mbar_arrive(EMPTY(slot));
            }
            k += np_eff * spi;
        }
        ptx::bulk_wait_all<0>();
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem, 512);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn()
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

// x or y viewed as (C, W, H, B), box {CGT channels, W', 7 rows, 1 image}, swizzled over the pixel's 16-byte chunks.
// 64-byte pixels are fetched as 64-byte L2 requests: with 128-byte promotion the other half of each line (the
// neighbouring channel group) came along and was fetched again later (97 MB read for a 77 MB input, 2-5 % slower).
template <int NOCT>
bool make_map(const Geom& g, int dtype, const void* base, CUtensorMap* map)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)g.C, (cuuint64_t)g.W, (cuuint64_t)g.H, (cuuint64_t)g.B};
    const cuuint64_t strides[3] = {(cuuint64_t)g.C * 2, (cuuint64_t)g.C * 2 * g.W, (cuuint64_t)g.C * 2 * g.W * g.H};
    const cuuint32_t box[4] = {(cuuint32_t)PipeCfg<NOCT>::CGT, (cuuint32_t)g.Wp, (cuuint32_t)WS, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUtensorMapSwizzle swz = NOCT == 4 ? CU_TENSOR_MAP_SWIZZLE_64B : (NOCT == 2 ? CU_TENSOR_MAP_SWIZZLE_32B : CU_TENSOR_MAP_SWIZZLE_NONE);
    return fn(map, dtype == WBMM_DTYPE_BF16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 4,
              const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, swz,
              NOCT == 4 ? CU_TENSOR_MAP_L2_PROMOTION_L2_64B : CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// <= 128 / NOCT windows of one channel group per tile: whole frame images, else strips of window rows; a slot is one
// window row of one image (7 x W' pixels of CGT channels).
template <int NOCT>
bool pipe_tiles(const Geom& g, TcTiles* t, int* nslot)
{
    using Pc = PipeCfg<NOCT>;
    if (g.layout != WBMM_LAYOUT_NHWC || g.w != WS || g.C % Pc::CGT != 0 || g.sh != 0 || g.sw != 0) return false;
    if (g.nww > Pc::WT || g.Wp > 256) return false;
    const int wpp = g.nwh * g.nww;
    if (wpp <= Pc::WT) {
        t->NSY = g.nwh;
        t->NP = Pc::WT / wpp;
        if (t->NP > g.B) t->NP = g.B;
    } else {
        t->NP = 1;
        t->NSY = Pc::WT / g.nww;
    }
    t->S = (int)(((long long)WS * g.Wp * Pc::PX + 1023) / 1024 * 1024);      // one window row
    const long long room = 227ll * 1024 - 1024 - Pc::FIXED;
    // strips of >= 4 window rows: one row less when that lets TWO tiles fit the ring (in-place output holds a slot
    // from its load to the end of its store; measured 56 x 56, C = 96: 80 -> 72 us at B = 128)
    if (t->NP == 1 && t->NSY >= 4 && 2 * t->NSY > room / t->S && 2 * (t->NSY - 1) <= room / t->S) t->NSY -= 1;
    t->frame_rows = t->NSY * g.w;
    t->nstrips = (g.nwh + t->NSY - 1) / t->NSY;
    t->ngb = (g.B + t->NP - 1) / t->NP;
    t->tiles_per_c = t->ngb * t->nstrips;                   // per channel GROUP
    t->ntiles = (long long)(g.C / Pc::CGT) * t->tiles_per_c;
    const int per_tile = t->NP * t->NSY;
    long long n = room / t->S;
    if (n > 2 * per_tile) n = 2 * per_tile;
    if (n > kMaxSlots) n = kMaxSlots;
    *nslot = (int)n;
    return n >= per_tile && t->ntiles <= 0x3fffffffll;
}

template <bool BF16, int NOCT>
cudaError_t launch_pipe(const Geom& g, const TcTiles& tl, int nslot, const void* x, const void* T, void* y, bool reverse, cudaStream_t s)
{
    CUtensorMap mx, my;
    const int dtype = BF16 ? WBMM_DTYPE_BF16 : WBMM_DTYPE_F16;
    if (!make_map<NOCT>(g, dtype, x, &mx) || !make_map<NOCT>(g, dtype, y, &my)) return cudaErrorNotSupported;
    auto k = tc_nhwc7_kernel<BF16, NOCT>;
    const size_t smem = (size_t)PipeCfg<NOCT>::FIXED + (size_t)nslot * tl.S;
    static SmemOptIn smem_state;
    cudaError_t e = ensure_dynamic_smem(reinterpret_cast<const void*>(k), smem, &smem_state);
    if (e != cudaSuccess) return e;
    int grid = (int)(tl.ntiles < num_sms() ? tl.ntiles : num_sms());
    if (grid > kMaxGrid) grid = kMaxGrid;
    static std::mutex mu;
    static TilePart cached;
    static long long key_n = -1;
    static int key_tpc = -1, key_grid = -1, cached_used = 0;
    TilePart part;
    {
        std::lock_guard<std::mutex> lock(mu);
        if (key_n != tl.ntiles || key_tpc != tl.tiles_per_c || key_grid != grid) {
            cached_used = partition_tiles(tl, grid, 0.3, &cached);
            key_n = tl.ntiles; key_tpc = tl.tiles_per_c; key_grid = grid;
        }
        part = cached;
        grid = cached_used;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(kThreadsP);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k, g, tl, part, nslot, mx, my, (const uint16_t*)T, reverse ? 1 : 0);
}

// the widest channel group this shape allows: 4 octets (64-byte pixels), else 2, else 1
int pick_octets(const Geom& g, TcTiles* tl, int* nslot)
{
    if (pipe_tiles<4>(g, tl, nslot)) return 4;
    if (pipe_tiles<2>(g, tl, nslot)) return 2;
    if (pipe_tiles<1>(g, tl, nslot)) return 1;
    return 0;
}

}  // namespace

bool tc_nhwc_pipe_supported(const Geom& g, int dtype, const void* x, const void* y)
{
    if (dtype != WBMM_DTYPE_BF16 && dtype != WBMM_DTYPE_F16) return false;
    if (reinterpret_cast<uintptr_t>(x) % 16 != 0 || reinterpret_cast<uintptr_t>(y) % 16 != 0) return false;
    TcTiles tl;
    int nslot;
    return pick_octets(g, &tl, &nslot) != 0 && encode_fn() != nullptr;
}

cudaError_t tc_nhwc_pipe_forward(const Geom& g, int dtype, const void* x, const void* T, void* y, bool reverse,
                                 cudaStream_t stream, int* launches)
{
    TcTiles tl;
    int nslot;
    const int noct = pick_octets(g, &tl, &nslot);
    if (noct == 0) return cudaErrorNotSupported;
    if (tl.ntiles == 0) return cudaSuccess;
    *launches += 1;
    const bool bf = dtype == WBMM_DTYPE_BF16;
    switch (noct) {
    case 4: return bf ? launch_pipe<true, 4>(g, tl, nslot, x, T, y, reverse, stream) : launch_pipe<false, 4>(g, tl, nslot, x, T, y, reverse, stream);
    case 2: return bf ? launch_pipe<true, 2>(g, tl, nslot, x, T, y, reverse, stream) : launch_pipe<false, 2>(g, tl, nslot, x, T, y, reverse, stream);
    default: return bf ? launch_pipe<true, 1>(g, tl, nslot, x, T, y, reverse, stream) : launch_pipe<false, 1>(g, tl, nslot, x, T, y, reverse, stream);
    }
}

}  // namespace wbmm
