// wbmm_forward_static_scratch (include/wbmm.h): the NHWC transposition route of wbmm_forward (DESIGN.md section 7.2:
// transpose16 -> NCHW tensor-core kernel -> transpose16) for callers that may not allocate -- code under CUDA graph
// capture, serving loops, harnesses that forbid cudaMalloc.  The two temporaries of that route live in ONE file-scope
// device array of fixed size instead of the library's stream-ordered memory pool, so this entry point calls no
// cudaMalloc / cudaFree / cudaMallocAsync and no allocating library routine.
//
//   * Size: kStaticScratchBytes = 32 MiB = two temporaries of 16 MiB.  Every GPU that loads libwbmm.so holds these
//     32 MiB from module load until the process exits, whether or not the entry point is ever called.
//   * In host code the array's NAME is a host-side stand-in, not a device address: its device address is asked for
//     once per device with cudaGetSymbolAddress (with that device current) and only that pointer goes to the kernels.
//   * Every call on a device shares the array and finds the previous call's contents in it.  Nothing has to start at
//     zero: the first transposition writes every element of temporary 0 the NCHW kernel reads, and that kernel writes
//     every element of temporary 1 the second transposition reads (wbmm_forward overwrites its whole output).
//   * Calls that overlap on the GPU (two streams, two host threads on two streams) RACE on the array.  Calls on one
//     stream are ordered by the stream and are safe back to back.
#include <atomic>
#include <mutex>

#include "wbmm_common.cuh"
#include "wbmm_tc.cuh"

namespace wbmm {

namespace {

constexpr size_t kHalfBytes = 16ull << 20;                // one temporary
constexpr size_t kStaticScratchBytes = 2 * kHalfBytes;    // 32 MiB per GPU

static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

constexpr int kMaxDev = 64;
std::mutex g_mu;
unsigned char* g_addr[kMaxDev] = {};      // device address of g_static_scratch on device d (0 = not asked yet)

// Device address of the array on the CURRENT device: cudaGetSymbolAddress once per device, with that device current.
cudaError_t static_scratch_address(unsigned char** out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDev) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_addr[dev]) {
        unsigned char* p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_addr[dev] = p;
    }
    *out = g_addr[dev];
    return cudaSuccess;
}

}  // namespace

size_t static_scratch_limit_bytes() { return kHalfBytes; }

// 0 = served, 1 = not a problem of this route (nothing launched), 2 = larger than the static scratch (nothing launched).
int nhwc_forward_static_scratch(const Geom& g, int dtype, const void* x, const void* T, void* y, cudaStream_t stream,
                                int* launches, int* path, cudaError_t* err)
{
    *err = cudaSuccess;
    if (g.layout != WBMM_LAYOUT_NHWC || (dtype != WBMM_DTYPE_BF16 && dtype != WBMM_DTYPE_F16)) return 1;
    if (g.C % 8 != 0 || ((long long)g.H * g.W) % 8 != 0) return 1;
    Geom gn = g;
    gn.layout = WBMM_LAYOUT_NCHW;
    void* const aligned16 = reinterpret_cast<void*>(256);
    if (!tc_bulk_supported(gn, dtype, aligned16, aligned16) || !transpose16_supported((long long)g.H * g.W, g.C, x, y)) return 1;
    const size_t nbytes = (size_t)g.B * g.C * g.H * g.W * 2;
    if (nbytes > kHalfBytes) return 2;
    unsigned char* base = nullptr;
    *err = static_scratch_address(&base);
    if (*err != cudaSuccess) return 0;
    void* xt = base;                       // [B][C][H*W] copy of x
    void* yt = base + kHalfBytes;          // [B][C][H*W] result
    *err = transpose16(x, xt, g.B, g.H * g.W, g.C, stream, launches);
    if (*err == cudaSuccess) *err = tc_forward(gn, dtype, xt, T, nullptr, yt, false, stream, launches, path, nullptr, 0u);
    if (*err == cudaSuccess) *err = transpose16(yt, y, g.B, g.C, g.H * g.W, stream, launches);
    return 0;
}

}  // namespace wbmm
