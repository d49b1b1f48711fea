// WBMM table gradient for FP32 activations on the tensor cores (SURVEY.md 8(a) row a8 in the paper's own precision,
// PAPER.md:237).  The scheme of wbmm_tc_dt.cu with fp32 frames and split operands:
//     S_c[i, j] = sum over windows n of dY[n, i] * X[n, j]          (tcgen05.mma, fp32 in TMEM)
//     dT[c, k]  = sum over pairs (i, j) with rel(i, j) = k of S_c[i, j]   (Eq. 6-7 as a scatter)
// Every fp32 value is split exactly into bf16 terms v = v1 + v2 (+ v3) (wbmm_tc_f32.cuh) while it is written into the
// MN-major operand stage, and the product is expanded into its leading cross terms:
//     w = 14, two terms per value (a 320 KB stage would be needed for three):  dy1 x1 + dy1 x2 + dy2 x1
//             -- each product is then exact to 2^-16 relative; over the L * mult(k) >= 10^4 products of a bin that is
//                the size of the fp32 accumulation error itself (measured)
//     w = 7,  three terms per value, six cross terms (as the forward kernel).
// A tile is 64 windows of one channel (fp32 frames are twice the size: x and dy of 64 windows are 100 KB at w = 14).
//
//   warp 0      producer   bulk loads of the x and dy frame images of a tile into the slot ring
//   warp 1      MMA        terms x MT x 4 tcgen05.mma (SS form, both operands MN-major) per tile
//   warps 2-9   two threads per (window, operand): frame -> split -> operand stage; all eight: the bin epilogue
#include "wbmm_tc_f32.cuh"

#include <cuda.h>

#include <mutex>

namespace wbmm {

using namespace tcdev;

namespace {

constexpr int kThreadsFD = 320;

template <int WS>
struct FDtCfg {
    using Cf = WinCfg<WS>;
    static constexpr int NS = WS == 14 ? 2 : 3;        // bf16 terms per fp32 value
    static constexpr int NTERM = NS == 2 ? 3 : 6;      // cross terms of weight >= 2^-16
    static constexpr int MT = (Cf::N + 127) / 128;     // M tiles of 128 output positions
    static constexpr int NV = (Cf::N + 7) / 8;         // 16-byte vectors (8 positions) a window fills
    static constexpr int NVEC = Cf::N_PAD / 8;         // vectors per operand region
    static constexpr int HW = 64;                      // windows per tile = MMA K of one stage
    // two CTAs per SM at w = 7 (S is 64 TMEM columns, the stage 48 KB, <= 86 registers), as in wbmm_tc_dt.cu
    static constexpr int CTAS = WS == 7 ? 2 : 1;
    static constexpr int TMEM_COLS = WS == 7 ? 128 : 512;
    static constexpr int SBO = HW * 16;                // bytes between position groups
    static constexpr int LBO = 128;                    // bytes between groups of 8 windows
    static constexpr int OP_BYTES = NVEC * SBO;        // one operand term
    static constexpr int STAGE = 2 * NS * OP_BYTES;    // A (dy) terms, then B (x) terms; an A M-tile's 16 vectors may run into the next region
    static constexpr int BAR_BYTES = (2 * kMaxSlots + 4) * 8;
    static constexpr int FIXED = (STAGE + BAR_BYTES + 127) / 128 * 128;
    // bin fold as in wbmm_tc_dt.cu: a warp's private bins have row pitch BP = WS (mod 32)
    static constexpr int BP = ((Cf::TW - WS + 31) / 32) * 32 + WS;
    static constexpr int BN = Cf::TW * BP;
    static_assert(8 * BN * 4 <= STAGE, "per-warp bin copies alias the stage");
    static_assert(MT * 16 <= 2 * NVEC, "an A M-tile must stay inside the stage");
};

// 8 fp32 values -> NS vectors of 8 bf16 terms each
template <int NS>
__device__ __forceinline__ void split_vec(const float* f, uint4* out)
{
    uint32_t p[3][4];
#pragma unroll
    for (int e2 = 0; e2 < 4; ++e2) split3(f[2 * e2], f[2 * e2 + 1], p[0][e2], p[1][e2], p[2][e2]);
#pragma unroll
    for (int s = 0; s < NS; ++s) out[s] = make_uint4(p[s][0], p[s][1], p[s][2], p[s][3]);
}

template <int WS, bool GEN>
__global__ void __launch_bounds__(kThreadsFD, FDtCfg<WS>::CTAS)
tc_f32_dt_kernel(Geom g, TcTiles tl, TilePart part_, int nslot, const float* __restrict__ x, const float* __restrict__ dy,
                 float* __restrict__ dT)
{
    using Cf = WinCfg<WS>;
    using Dc = FDtCfg<WS>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* stage = smem;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Dc::STAGE);
    uint8_t* ring = smem + Dc::FIXED;
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t bar0 = ptx::smem_u32(bars);
    auto FULL = [&](int s) { return bar0 + 8u * s; };
    auto EMPTY = [&](int s) { return bar0 + 8u * (kMaxSlots + s); };
    const uint32_t STAGE_FULL = bar0 + 8u * (2 * kMaxSlots), STAGE_EMPTY = STAGE_FULL + 8;
    const int wpf = tl.NSY * g.nww;

    if (warp == 1) ptx::tmem_alloc(ptx::smem_u32(&tmem_base_s), Dc::TMEM_COLS);
    if (tid >= 64 && tid < 64 + nslot) {
        ptx::mbar_init(FULL(tid - 64), 1);
        ptx::mbar_init(EMPTY(tid - 64), 2 * wpf);        // two threads per window of the image
        ptx::fence_mbar_init();
    }
    if (tid == 0) {
        ptx::mbar_init(STAGE_FULL, 256);
        ptx::mbar_init(STAGE_EMPTY, 1);
        ptx::fence_mbar_init();
    }
    // vectors a window never writes (padding positions) must read as zero
    for (int i = tid; i < Dc::STAGE / 16; i += kThreadsFD) reinterpret_cast<uint4*>(stage)[i] = make_uint4(0, 0, 0, 0);
    ptx::fence_proxy_async_smem();
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::tc_fence_after_sync();
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const uint32_t tmem = tmem_base_s;

    const int t0 = part_.start[blockIdx.x], t1 = part_.start[blockIdx.x + 1];
    const int rowB = g.W * 4;
    const long long plane_elems = (long long)g.H * g.W;

    auto tile_decode = [&](int t, int& c, int& b0, int& wy0, int& np_eff, int& rows_eff) {
        c = t / tl.tiles_per_c;
        const int rem = t - c * tl.tiles_per_c;
        const int gb = rem / tl.nstrips, strip = rem - gb * tl.nstrips;
        b0 = gb * tl.NP;
        wy0 = strip * tl.NSY;
        np_eff = min(tl.NP, g.B - b0);
        rows_eff = GEN ? g.H : min(tl.frame_rows, g.H - wy0 * WS);
    };

    if (warp == 0) {
        // ------------------------------------------------------------------ producer
        // ring order per tile: x image 0, dy image 0, x image 1, dy image 1, ...
        uint32_t k = 0;
        for (int t = t0; t < t1; ++t) {
            int c, b0, wy0, np_eff, rows_eff;
            tile_decode(t, c, b0, wy0, np_eff, rows_eff);
            const uint32_t bytes = (uint32_t)rows_eff * rowB;
            for (int j = lane; j < 2 * np_eff; j += 32) {
                const uint32_t kk = k + j;
                const int slot = kk % nslot;
                ptx::mbar_wait(EMPTY(slot), ((kk / nslot) & 1) ^ 1);
                ptx::mbar_arrive_expect_tx(FULL(slot), bytes);
                const float* src = ((j & 1) ? dy : x) + ((long long)(b0 + (j >> 1)) * g.C + c) * plane_elems + (long long)wy0 * WS * g.W;
                ptx::bulk_g2s(ptx::smem_u32(ring + (size_t)slot * tl.S), src, bytes, FULL(slot));
            }
            k += 2 * np_eff;
            __syncwarp();   // no lane starts the next tile's copies before every copy of this tile is issued
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer (whole warp walks, one lane issues)
        constexpr uint32_t idesc = ptx::idesc_f16(1, 128, Cf::N_PAD) | (1u << 15) | (1u << 16);   // bf16, A and B MN-major
        const uint32_t stage_addr = ptx::smem_u32(stage);
        // (dy term, x term), smallest products first
        constexpr int SA2[3] = {1, 0, 0}, SB2[3] = {0, 1, 0};
        constexpr int SA3[6] = {2, 1, 0, 1, 0, 0}, SB3[6] = {0, 1, 2, 0, 1, 0};
        uint32_t lt = 0;
        int cur_c = -1;
        for (int t = t0; t < t1; ++t, ++lt) {
            const int c = t / tl.tiles_per_c;
            ptx::mbar_wait(STAGE_FULL, lt & 1);
            ptx::tc_fence_after_sync();
            if (ptx::elect_one()) {
#pragma unroll
                for (int term = 0; term < Dc::NTERM; ++term) {
                    const int sa = Dc::NS == 2 ? SA2[term % 3] : SA3[term], sb = Dc::NS == 2 ? SB2[term % 3] : SB3[term];
                    const uint32_t a_addr = stage_addr + sa * Dc::OP_BYTES, b_addr = stage_addr + (Dc::NS + sb) * Dc::OP_BYTES;
#pragma unroll
                    for (int mt = 0; mt < Dc::MT; ++mt) {
#pragma unroll
                        for (int ks = 0; ks < Dc::HW / 16; ++ks) {
                            const uint64_t ad = ptx::smem_desc_kmajor_noswz(a_addr + mt * 16 * Dc::SBO + ks * 2 * Dc::LBO, Dc::LBO, Dc::SBO);
                            const uint64_t bd = ptx::smem_desc_kmajor_noswz(b_addr + ks * 2 * Dc::LBO, Dc::LBO, Dc::SBO);
                            ptx::mma_ss(tmem + mt * 256, ad, bd, idesc, (c != cur_c && term == 0 && ks == 0) ? 0u : 1u);
                        }
                    }
                }
                ptx::mma_commit(STAGE_EMPTY);
            }
            __syncwarp();
            cur_c = c;
        }
    } else {
        // ------------------------------------------------------------------ operand repack + bin epilogue
        const int ot = tid - 64;            // 0..255
        const int o = ot >> 7;              // 0: x -> B terms, 1: dy -> A terms
        const int hsel = (ot >> 6) & 1;     // which half of the window's position vectors (uniform per warp pair)
        const int m = ot & 63;              // window of the tile = MMA K index (image-major)
        const int pl = m / wpf, wl = m - pl * wpf;
        const int wyl = wl / g.nww, wx = wl - wyl * g.nww;
        const int win_off = ((wyl * WS) * g.W + wx * WS) * 4;
        GenAddrF<GEN ? WS : 1> ga;
        if constexpr (GEN) gen_addr_f32<WS>(ga, g, wyl, wx);
        uint8_t* dst = stage + (o ? 0 : Dc::NS * Dc::OP_BYTES) + m * 16;
        float* bins = reinterpret_cast<float*>(stage);
        float* bw = bins + (ot >> 5) * Dc::BN;          // this warp's private copy of the bins
        const int ew = ot >> 5;                          // 0..7
        const int emt = ew >> 2, eq = warp & 3;          // M-tile and TMEM lane quarter in the epilogue
        const int erow = emt * 128 + eq * 32 + lane;     // row of S = output position i
        const int eri = erow / WS, eci = erow - eri * WS;
        constexpr int NVH = (Dc::NV + 1) / 2;            // vectors [0, NVH) | [NVH, NV)
        uint32_t k = 0, lt = 0;
        for (int t = t0; t < t1; ++t, ++lt) {
            int c, b0, wy0, np_eff, rows_eff;
            tile_decode(t, c, b0, wy0, np_eff, rows_eff);
            // Slot barriers are tested by phase PARITY and successive fills of one slot are consumed by different threads:
            // after this barrier every repack thread has passed its waits of the previous tile, and a slot's previous
            // fill always belongs to an earlier tile (nslot >= copies per tile).
            ptx::named_bar_sync(1, 256);
            const bool part = pl < tl.NP && pl < np_eff;
            const bool valid = part && wy0 + wyl < g.nwh;
            const uint32_t kk = k + 2 * pl + o;
            const int slot = kk % nslot;
            if (part) ptx::mbar_wait(FULL(slot), (kk / nslot) & 1);
            ptx::mbar_wait(STAGE_EMPTY, (lt & 1) ^ 1);      // the MMAs of tile lt-1 have read the stage
            const uint8_t* img = ring + (size_t)(part ? slot : 0) * tl.S;
            const uint32_t rm = (GEN && valid) ? ga.rowmask : 0u;
            auto do_vectors = [&](auto hc) {
                constexpr int V0 = decltype(hc)::value ? NVH : 0, V1 = decltype(hc)::value ? Dc::NV : NVH;
#pragma unroll
                for (int v = V0; v < V1; ++v) {
                    float f[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const int p = 8 * v + e;
                        f[e] = 0.f;
                        if (p < Cf::N) {
                            const int r = p / WS, cc = p % WS;
                            if constexpr (GEN) {
                                const float val = *reinterpret_cast<const float*>(img + ga.rowoff[r] + ga.coloff[cc]);
                                if ((rm >> r) & (ga.colmask >> cc) & 1u) f[e] = val;
                            } else {
                                const float val = *reinterpret_cast<const float*>(img + (valid ? win_off + r * rowB + cc * 4 : 0));
                                if (valid) f[e] = val;
                            }
                        }
                    }
                    uint4 sv[Dc::NS];
                    split_vec<Dc::NS>(f, sv);
#pragma unroll
                    for (int s = 0; s < Dc::NS; ++s) *reinterpret_cast<uint4*>(dst + s * Dc::OP_BYTES + v * Dc::SBO) = sv[s];
                }
            };
            if (hsel == 0) do_vectors(std::integral_constant<int, 0>{});
            else do_vectors(std::integral_constant<int, 1>{});
            ptx::fence_proxy_async_smem();
            ptx::mbar_arrive(STAGE_FULL);
            if (part) ptx::mbar_arrive(EMPTY(slot));
            k += 2 * np_eff;

            const bool seg_end = t + 1 == t1 || (t + 1) - c * tl.tiles_per_c == tl.tiles_per_c;
            if (seg_end) {
                // ---- S (TMEM) -> bins -> dT[c]   (as in wbmm_tc_dt.cu)
                ptx::mbar_wait(STAGE_EMPTY, lt & 1);        // every MMA of this channel segment has completed
                ptx::tc_fence_after_sync();
                for (int b = lane; b < Dc::BN; b += 32) bw[b] = 0.f;
                __syncwarp();
                if (emt < Dc::MT) {
                    // Row i = erow of S goes to bins base - rj*BP - cj.  For a fixed column j the 32 rows of the warp hit
                    // 32 different bins; input rows rj and rj + RJ_STRIDE are independent too: NU chains per step.
                    const uint32_t taddr = tmem + emt * 256 + ((uint32_t)(eq * 32) << 16);
                    float* bbase = bw + (eri + WS - 1) * Dc::BP + eci + WS - 1;
                    const bool rowok = erow < Cf::N;
                    constexpr int RJ_STRIDE = 31 / WS + 1, NU = (WS + RJ_STRIDE - 1) / RJ_STRIDE;
#pragma unroll
                    for (int g0 = 0; g0 < RJ_STRIDE; ++g0) {
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
                ptx::named_bar_sync(1, 256);
                // the bins aliased the operand stage: restore the zero padding vectors
                for (int i = ot; i < 8 * Dc::BN * 4 / 16 + 1; i += 256)
                    if (i * 16 < Dc::STAGE) reinterpret_cast<uint4*>(stage)[i] = make_uint4(0, 0, 0, 0);
                ptx::fence_proxy_async_smem();
                ptx::named_bar_sync(1, 256);
            }
        }
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem, Dc::TMEM_COLS);
}

// Tiles of <= 64 windows of one channel: whole frame images, else strips of window rows (aligned form only); slots
// for x and dy of a tile, two tiles where they fit.  Fewer images per tile when even one tile does not fit.
template <int WS>
bool f32dt_tiles_for(const Geom& g, TcTiles* t, int* nslot, int ctas);

// two CTAs per SM where a tile and a half of x and dy fit half the shared memory, else one
template <int WS>
bool f32dt_tiles(const Geom& g, TcTiles* t, int* nslot, int* ctas)
{
    if (FDtCfg<WS>::CTAS > 1) {
        TcTiles t1;
        int n1 = 0;
        const bool one = f32dt_tiles_for<WS>(g, &t1, &n1, 1);
        if (f32dt_tiles_for<WS>(g, t, nslot, FDtCfg<WS>::CTAS) && *nslot >= 3 * t->NP && (!one || t->NP == t1.NP && t->NSY == t1.NSY)) {
            *ctas = FDtCfg<WS>::CTAS;
            return true;
        }
    }
    *ctas = 1;
    return f32dt_tiles_for<WS>(g, t, nslot, 1);
}

template <int WS>
bool f32dt_tiles_for(const Geom& g, TcTiles* t, int* nslot, int ctas)
{
    using Dc = FDtCfg<WS>;
    if (g.nww > Dc::HW) return false;
    const int wpp = g.nwh * g.nww;
    if (wpp <= Dc::HW) {
        t->NSY = g.nwh;
        t->NP = Dc::HW / wpp;
        if (t->NP > g.B) t->NP = g.B;
    } else {
        t->NP = 1;
        t->NSY = Dc::HW / g.nww;
    }
    const long long room = (ctas == 1 ? 227ll * 1024 : 113ll * 1024) - 1024 - Dc::FIXED;
    for (;;) {
        t->frame_rows = t->NSY * g.w;
        int s16 = (t->frame_rows * g.Wp * 4 + 15) / 16;
        if (s16 % 2 == 0) ++s16;
        t->S = s16 * 16;
        if (2ll * t->NP * t->S <= room) break;
        if (t->NP > 1) t->NP = (t->NP + 1) / 2;
        else if (t->NSY > 1) t->NSY = (t->NSY + 1) / 2;
        else return false;
    }
    t->nstrips = (g.nwh + t->NSY - 1) / t->NSY;
    t->ngb = (g.B + t->NP - 1) / t->NP;
    t->tiles_per_c = t->ngb * t->nstrips;
    t->ntiles = (long long)g.C * t->tiles_per_c;
    long long n = room / t->S;
    if (n > 4 * t->NP) n = 4 * t->NP;
    if (n > kMaxSlots) n = kMaxSlots;
    *nslot = (int)n;
    return n >= 2 * t->NP && t->ntiles <= 0x3fffffffll;
}

// 0 = not servable, 1 = aligned form, 2 = general form (shift / ragged, whole images)
template <int WS>
int f32dt_mode(const Geom& g, const TcTiles& tl, const void* x, const void* dy)
{
    if (g.layout != WBMM_LAYOUT_NCHW) return 0;
    if (reinterpret_cast<uintptr_t>(x) % 16 != 0 || reinterpret_cast<uintptr_t>(dy) % 16 != 0) return 0;
    if (((long long)g.H * g.W * 4) % 16 != 0) return 0;
    const bool plain = g.sh == 0 && g.sw == 0 && g.H == g.Hp && g.W == g.Wp;
    if (plain && (tl.nstrips == 1 || ((long long)tl.frame_rows * g.W * 4) % 16 == 0)) return 1;
    return tl.nstrips == 1 ? 2 : 0;
}

template <int WS, bool GEN>
cudaError_t launch_f32dt(const Geom& g, const TcTiles& tl, int nslot, int ctas, const void* x, const void* dy, float* dT, cudaStream_t s)
{
    auto k = tc_f32_dt_kernel<WS, GEN>;
    const size_t smem = (size_t)FDtCfg<WS>::FIXED + (size_t)nslot * tl.S;
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
            cached_used = partition_tiles(tl, grid, 1.0, &cached);   // a channel boundary costs one bin fold
            key_n = tl.ntiles; key_tpc = tl.tiles_per_c; key_grid = grid;
        }
        part = cached;
        grid = cached_used;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(kThreadsFD);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k, g, tl, part, nslot, (const float*)x, (const float*)dy, dT);
}

}  // namespace

bool tc_f32_grad_table_supported(const Geom& g, const void* x, const void* dy)
{
    if (g.w != 7 && g.w != 14) return false;
    TcTiles tl;
    int nslot, ctas;
    if (!(g.w == 7 ? f32dt_tiles<7>(g, &tl, &nslot, &ctas) : f32dt_tiles<14>(g, &tl, &nslot, &ctas))) return false;
    return (g.w == 7 ? f32dt_mode<7>(g, tl, x, dy) : f32dt_mode<14>(g, tl, x, dy)) != 0;
}

// dT must have been cleared (or hold the values to accumulate into): the kernel adds.
cudaError_t tc_f32_grad_table(const Geom& g, const void* x, const void* dy, float* dT, cudaStream_t stream, int* launches)
{
    TcTiles tl;
    int nslot, ctas;
    if (!(g.w == 7 ? f32dt_tiles<7>(g, &tl, &nslot, &ctas) : f32dt_tiles<14>(g, &tl, &nslot, &ctas))) return cudaErrorNotSupported;
    if (tl.ntiles == 0) return cudaSuccess;
    const int mode = g.w == 7 ? f32dt_mode<7>(g, tl, x, dy) : f32dt_mode<14>(g, tl, x, dy);
    if (mode == 0) return cudaErrorNotSupported;
    *launches += 1;
    if (g.w == 7)
        return mode == 2 ? launch_f32dt<7, true>(g, tl, nslot, ctas, x, dy, dT, stream) : launch_f32dt<7, false>(g, tl, nslot, ctas, x, dy, dT, stream);
    return mode == 2 ? launch_f32dt<14, true>(g, tl, nslot, ctas, x, dy, dT, stream) : launch_f32dt<14, false>(g, tl, nslot, ctas, x, dy, dT, stream);
}

}  // namespace wbmm
