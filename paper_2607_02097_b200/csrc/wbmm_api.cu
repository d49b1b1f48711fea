// C ABI of libwbmm.so (include/wbmm.h): argument validation, path selection, host-buffer variants.
// No compute happens here and nothing here can fall back to a CPU implementation.
#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>

#include "wbmm_common.cuh"
#include "wbmm_tc.cuh"

namespace {

thread_local int t_last_path = WBMM_PATH_NONE;
thread_local char t_last_error[256] = "";
std::atomic<uint64_t> g_launches{0};

int set_cuda_error(cudaError_t e, const char* where)
{
    snprintf(t_last_error, sizeof(t_last_error), "%s: %s", where, cudaGetErrorString(e));
    return WBMM_STATUS_CUDA_ERROR;
}

size_t elem_size(int dtype) { return dtype == WBMM_DTYPE_F32 ? 4 : 2; }

constexpr int kMaxDevices = 64;

// Is the CURRENT device an sm_100 part?  Cached per device: 0 = not probed, 1 = yes, -1 = no.
int device_state()
{
    static std::atomic<int> state[kMaxDevices];
    int dev = 0, major = 0, count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count == 0 || cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return -1;
    }
    const bool cached = dev >= 0 && dev < kMaxDevices;
    int s = cached ? state[dev].load(std::memory_order_relaxed) : 0;
    if (s != 0) return s;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        cudaGetLastError();
        return -1;
    }
    s = major == 10 ? 1 : -1;
    if (cached) state[dev].store(s, std::memory_order_relaxed);
    return s;
}

int validate(const wbmm_desc_t* d)
{
    if (!d) return WBMM_STATUS_INVALID_ARGUMENT;
    if (d->B < 0 || d->C < 0 || d->H < 1 || d->W < 1 || d->w < 1) return WBMM_STATUS_INVALID_ARGUMENT;
    if (d->shift_h < 0 || d->shift_w < 0 || d->shift_h >= d->w || d->shift_w >= d->w)
        return WBMM_STATUS_INVALID_ARGUMENT;
    if (d->dtype != WBMM_DTYPE_F32 && d->dtype != WBMM_DTYPE_BF16 && d->dtype != WBMM_DTYPE_F16)
        return WBMM_STATUS_INVALID_ARGUMENT;
    if (d->layout != WBMM_LAYOUT_NCHW && d->layout != WBMM_LAYOUT_NHWC) return WBMM_STATUS_INVALID_ARGUMENT;
    if (d->w > 1024) return WBMM_STATUS_UNSUPPORTED;
    // index arithmetic is 64-bit for elements, 32-bit for per-axis sizes
    long long n = (long long)d->B * d->C;
    if (n > (1ll << 40) / ((long long)d->H * d->W)) return WBMM_STATUS_UNSUPPORTED;
    return WBMM_STATUS_OK;
}

bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

// NHWC through NCHW: stream-ordered temporaries from a memory pool the LIBRARY owns (one per device, created on
// first use, destroyed by wbmm_release).  Freed blocks stay cached in that pool (release threshold = max), so a call
// pays no fresh allocation after the first -- without touching the policy of the device's default pool, which
// belongs to the application (a PyTorch process may run its own allocator on it).
std::mutex g_pool_mutex;
cudaMemPool_t g_pools[kMaxDevices] = {};

cudaError_t scratch_pool(cudaMemPool_t* out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    if (!g_pools[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool;
        e = cudaMemPoolCreate(&pool, &props);
        if (e != cudaSuccess) return e;
        uint64_t keep = ~0ull;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        g_pools[dev] = pool;
    }
    *out = g_pools[dev];
    return cudaSuccess;
}

void scratch_pools_release()
{
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    for (int d = 0; d < kMaxDevices; ++d)
        if (g_pools[d]) {
            cudaMemPoolDestroy(g_pools[d]);
            g_pools[d] = nullptr;
        }
}

struct AsyncScratch {
    void* p = nullptr;
    cudaStream_t s;
    explicit AsyncScratch(cudaStream_t stream) : s(stream) {}
    cudaError_t alloc(size_t n)
    {
        cudaMemPool_t pool;
        cudaError_t e = scratch_pool(&pool);
        if (e != cudaSuccess) return e;
        return cudaMallocFromPoolAsync(&p, n, pool, s);
    }
    ~AsyncScratch() { if (p) cudaFreeAsync(p, s); }
};

bool nhwc_scratch_candidate(const wbmm_desc_t* d, const wbmm::Geom& g)
{
    if (g.layout != WBMM_LAYOUT_NHWC || (d->flags & (WBMM_FLAG_FORCE_SIMT | WBMM_FLAG_NO_SCRATCH))) return false;
    if (d->dtype != WBMM_DTYPE_BF16 && d->dtype != WBMM_DTYPE_F16) return false;
    return g.C % 8 == 0 && ((long long)g.H * g.W) % 8 == 0;
}

// One operator application y = op(x; T) with op = W_c (reverse=false) or W_c^T (reverse=true).
int apply(const wbmm_desc_t* d, const wbmm::Geom& g, const void* x, const void* T, void* y,
          bool reverse, cudaStream_t stream)
{
    int launches = 0;
    cudaError_t e;
    if (g.layout == WBMM_LAYOUT_NHWC && !(d->flags & WBMM_FLAG_FORCE_SIMT) && wbmm::tc_nhwc_pipe_supported(g, d->dtype, x, y)) {
        // w = 7: one pass straight from NHWC memory, no scratch
        e = wbmm::tc_nhwc_pipe_forward(g, d->dtype, x, T, y, reverse, stream, &launches);
        g_launches += launches;
        if (e != cudaSuccess) return set_cuda_error(e, "tc_nhwc_pipe_forward");
        t_last_path = WBMM_PATH_TC_TMA;
        return WBMM_STATUS_OK;
    }
    if (nhwc_scratch_candidate(d, g)) {
        wbmm::Geom gn = g;
        gn.layout = WBMM_LAYOUT_NCHW;
        void* const aligned16 = reinterpret_cast<void*>(256);
        if (wbmm::tc_bulk_supported(gn, d->dtype, aligned16, aligned16) &&
            wbmm::transpose16_supported((long long)g.H * g.W, g.C, x, y)) {
            const size_t nbytes = (size_t)g.B * g.C * g.H * g.W * 2;
            AsyncScratch xt(stream), yt(stream);
            if (xt.alloc(nbytes) == cudaSuccess && yt.alloc(nbytes) == cudaSuccess) {
                int path = WBMM_PATH_NONE;
                e = wbmm::transpose16(x, xt.p, g.B, g.H * g.W, g.C, stream, &launches);
                if (e == cudaSuccess) e = wbmm::tc_forward(gn, d->dtype, xt.p, T, nullptr, yt.p, reverse, stream, &launches, &path);
                if (e == cudaSuccess) e = wbmm::transpose16(yt.p, y, g.B, g.C, g.H * g.W, stream, &launches);
                g_launches += launches;
                if (e != cudaSuccess) return set_cuda_error(e, "NHWC via NCHW scratch");
                t_last_path = WBMM_PATH_TC_TRANSPOSED;
                return WBMM_STATUS_OK;
            }
            cudaGetLastError();      // no stream-ordered allocator / out of memory: in-kernel NHWC path below
        }
    }
    if (g.layout == WBMM_LAYOUT_NHWC && d->dtype == WBMM_DTYPE_F32 && !(d->flags & (WBMM_FLAG_FORCE_SIMT | WBMM_FLAG_NO_SCRATCH)) &&
        wbmm::transpose32_supported((long long)g.H * g.W, g.C, x, y)) {
        // fp32 NHWC: the transposition route around the fp32 tensor-core kernel (the FFMA kernel is 3-5x slower)
        wbmm::Geom gn = g;
        gn.layout = WBMM_LAYOUT_NCHW;
        void* const aligned16 = reinterpret_cast<void*>(256);
        if (wbmm::tc_f32_supported(gn, aligned16, aligned16)) {
            const size_t nbytes = (size_t)g.B * g.C * g.H * g.W * 4;
            AsyncScratch xt(stream), yt(stream);
            if (xt.alloc(nbytes) == cudaSuccess && yt.alloc(nbytes) == cudaSuccess) {
                e = wbmm::transpose32(x, xt.p, g.B, g.H * g.W, g.C, stream, &launches);
                if (e == cudaSuccess) e = wbmm::tc_f32_forward(gn, xt.p, T, yt.p, reverse, stream, &launches);
                if (e == cudaSuccess) e = wbmm::transpose32(yt.p, y, g.B, g.C, g.H * g.W, stream, &launches);
                g_launches += launches;
                if (e != cudaSuccess) return set_cuda_error(e, "fp32 NHWC via NCHW scratch");
                t_last_path = WBMM_PATH_TC_TRANSPOSED;
                return WBMM_STATUS_OK;
            }
            cudaGetLastError();
        }
    }
    if (!(d->flags & WBMM_FLAG_FORCE_SIMT) && wbmm::tc_nhwc_supported(g, d->dtype, x, y)) {
        e = wbmm::tc_nhwc_forward(g, d->dtype, x, T, y, reverse, stream, &launches);
        g_launches += launches;
        if (e != cudaSuccess) return set_cuda_error(e, "tc_nhwc_forward");
        t_last_path = WBMM_PATH_TC_GATHER;
        return WBMM_STATUS_OK;
    }
    // The pipelined kernel where it applies.  Shapes only the block-synchronous gather kernel could take (planes that no
    // copy scheme addresses: 7 x 7, 30 x 30, odd W) go to the FFMA kernels instead when those fit: measured 1.4-2.3x
    // faster there (B128 C256 7x7 w7: 41.8 vs 21.3 us; B64 C96 30x30 w14: 226 vs 164 us).
    const bool pipelined = g.layout == WBMM_LAYOUT_NCHW && wbmm::tc_bulk_supported(g, d->dtype, x, y);
    if (!(d->flags & WBMM_FLAG_FORCE_SIMT) && wbmm::tc_forward_supported(g, d->dtype, x, y) &&
        (pipelined || !wbmm::simt_supported(g))) {
        int path = WBMM_PATH_NONE;
        e = wbmm::tc_forward(g, d->dtype, x, T, nullptr, y, reverse, stream, &launches, &path);
        g_launches += launches;
        if (e != cudaSuccess) return set_cuda_error(e, "tc_forward");
        t_last_path = path;
        return WBMM_STATUS_OK;
    }
    if (d->dtype == WBMM_DTYPE_F32 && !(d->flags & WBMM_FLAG_FORCE_SIMT) && wbmm::tc_f32_supported(g, x, y)) {
        e = wbmm::tc_f32_forward(g, x, T, y, reverse, stream, &launches);
        g_launches += launches;
        if (e != cudaSuccess) return set_cuda_error(e, "tc_f32_forward");
        t_last_path = WBMM_PATH_TC_TMA;
        return WBMM_STATUS_OK;
    }
    if (!wbmm::simt_supported(g)) return WBMM_STATUS_UNSUPPORTED;
    e = wbmm::simt_forward(g, d->dtype, x, T, y, reverse, stream, &launches);
    g_launches += launches;
    if (e != cudaSuccess) return set_cuda_error(e, "simt_forward");
    t_last_path = WBMM_PATH_SIMT;
    return WBMM_STATUS_OK;
}

// The table gradient of wbmm_backward on `stream` (clearing included): returns a wbmm_status_t.
int grad_table_on(const wbmm_desc_t* desc, const wbmm::Geom& g, const void* x, const void* dy, float* dT, cudaStream_t stream)
{
    if (!(desc->flags & WBMM_FLAG_ACCUMULATE_DT) && g.C > 0) {
        int zl = 0;
        cudaError_t e = wbmm::simt_zero_f32(dT, (long long)g.C * g.nb, stream, &zl);
        g_launches += zl;
        if (e != cudaSuccess) return set_cuda_error(e, "zero dT");
    }
    int launches = 0;
    cudaError_t e;
    bool done = false;
    if (nhwc_scratch_candidate(desc, g) && wbmm::transpose16_supported((long long)g.H * g.W, g.C, x, dy)) {
        wbmm::Geom gn = g;
        gn.layout = WBMM_LAYOUT_NCHW;
        void* const aligned16 = reinterpret_cast<void*>(256);
        if (wbmm::tc_grad_table_supported(gn, desc->dtype, aligned16, aligned16)) {
            const size_t nbytes = (size_t)g.B * g.C * g.H * g.W * 2;
            AsyncScratch xt(stream), gt(stream);
            if (xt.alloc(nbytes) == cudaSuccess && gt.alloc(nbytes) == cudaSuccess) {
                int path = WBMM_PATH_NONE;
                e = wbmm::transpose16(x, xt.p, g.B, g.H * g.W, g.C, stream, &launches);
                if (e == cudaSuccess) e = wbmm::transpose16(dy, gt.p, g.B, g.H * g.W, g.C, stream, &launches);
                if (e == cudaSuccess) e = wbmm::tc_grad_table(gn, desc->dtype, xt.p, gt.p, dT, stream, &launches, &path);
                g_launches += launches;
                if (e != cudaSuccess) return set_cuda_error(e, "NHWC dT via NCHW scratch");
                t_last_path = WBMM_PATH_TC_TRANSPOSED;
                done = true;
            } else {
                cudaGetLastError();
            }
        }
    }
    if (!done && g.layout == WBMM_LAYOUT_NHWC && desc->dtype == WBMM_DTYPE_F32 &&
        !(desc->flags & (WBMM_FLAG_FORCE_SIMT | WBMM_FLAG_NO_SCRATCH)) && wbmm::transpose32_supported((long long)g.H * g.W, g.C, x, dy)) {
        wbmm::Geom gn = g;
        gn.layout = WBMM_LAYOUT_NCHW;
        void* const aligned16 = reinterpret_cast<void*>(256);
        if (wbmm::tc_f32_grad_table_supported(gn, aligned16, aligned16)) {
            const size_t nbytes = (size_t)g.B * g.C * g.H * g.W * 4;
            AsyncScratch xt(stream), gt(stream);
            if (xt.alloc(nbytes) == cudaSuccess && gt.alloc(nbytes) == cudaSuccess) {
                e = wbmm::transpose32(x, xt.p, g.B, g.H * g.W, g.C, stream, &launches);
                if (e == cudaSuccess) e = wbmm::transpose32(dy, gt.p, g.B, g.H * g.W, g.C, stream, &launches);
                if (e == cudaSuccess) e = wbmm::tc_f32_grad_table(gn, xt.p, gt.p, dT, stream, &launches);
                g_launches += launches;
                if (e != cudaSuccess) return set_cuda_error(e, "fp32 NHWC dT via NCHW scratch");
                t_last_path = WBMM_PATH_TC_TRANSPOSED;
                done = true;
            } else {
                cudaGetLastError();
            }
        }
    }
    if (done) {
    } else if (!(desc->flags & WBMM_FLAG_FORCE_SIMT) && wbmm::tc_grad_table_supported(g, desc->dtype, x, dy)) {
        int path = WBMM_PATH_NONE;
        e = wbmm::tc_grad_table(g, desc->dtype, x, dy, dT, stream, &launches, &path);
        g_launches += launches;
        if (e != cudaSuccess) return set_cuda_error(e, "tc_grad_table");
        t_last_path = path;
    } else if (desc->dtype == WBMM_DTYPE_F32 && !(desc->flags & WBMM_FLAG_FORCE_SIMT) && wbmm::tc_f32_grad_table_supported(g, x, dy)) {
        e = wbmm::tc_f32_grad_table(g, x, dy, dT, stream, &launches);
        g_launches += launches;
        if (e != cudaSuccess) return set_cuda_error(e, "tc_f32_grad_table");
        t_last_path = WBMM_PATH_TC_TMA;
    } else {
        if (!wbmm::simt_supported(g)) return WBMM_STATUS_UNSUPPORTED;
        e = wbmm::simt_grad_table(g, desc->dtype, x, dy, dT, stream, &launches);
        g_launches += launches;
        if (e != cudaSuccess) return set_cuda_error(e, "simt_grad_table");
        t_last_path = WBMM_PATH_SIMT;
    }
    return WBMM_STATUS_OK;
}

// wbmm_backward with both gradients: dX and dT do not depend on each other, so the table gradient runs on an internal
// stream forked from the caller's and joined back into it -- its CTAs fill the SMs the dX kernel leaves idle at its ramp
// and tail, and at w = 7 one CTA of each kernel shares an SM (cfg5: 61.1 -> 56.2 us for dX + dT, replayed from a
// graph).  One side stream and event pair per host thread and device, created on first use outside stream capture.
struct SideStream {
    cudaStream_t s = nullptr;
    cudaEvent_t fork = nullptr, join = nullptr;
};
thread_local SideStream t_side[kMaxDevices];

SideStream* side_stream(cudaStream_t user)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        cudaGetLastError();
        return nullptr;
    }
    SideStream& ss = t_side[dev];
    if (ss.s) return &ss;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(user, &cap) != cudaSuccess || cap != cudaStreamCaptureStatusNone) {
        cudaGetLastError();
        return nullptr;              // never create resources under capture: this call runs dX and dT in sequence
    }
    cudaStream_t st = nullptr;
    cudaEvent_t a = nullptr, b = nullptr;
    if (cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&a, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&b, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        if (a) cudaEventDestroy(a);
        if (st) cudaStreamDestroy(st);
        return nullptr;
    }
    ss.s = st; ss.fork = a; ss.join = b;
    return &ss;
}

}  // namespace

extern "C" {

int wbmm_forward(const wbmm_desc_t* desc, const void* x, const void* T, void* y, void* cuda_stream)
{
    int st = validate(desc);
    if (st != WBMM_STATUS_OK) return st;
    if (desc->B == 0 || desc->C == 0) return WBMM_STATUS_OK;   // empty problem: nothing to read or write
    if (!x || !T || !y || x == y) return WBMM_STATUS_INVALID_ARGUMENT;
    const size_t es = elem_size(desc->dtype);
    if (!aligned(x, es) || !aligned(T, es) || !aligned(y, es)) return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    wbmm::Geom g = wbmm::make_geom(*desc);
    return apply(desc, g, x, T, y, false, static_cast<cudaStream_t>(cuda_stream));
}

int wbmm_forward_static_scratch(const wbmm_desc_t* desc, const void* x, const void* T, void* y, void* cuda_stream)
{
    int st = validate(desc);
    if (st != WBMM_STATUS_OK) return st;
    if (desc->B == 0 || desc->C == 0) return WBMM_STATUS_OK;
    if (!x || !T || !y || x == y) return WBMM_STATUS_INVALID_ARGUMENT;
    const size_t es = elem_size(desc->dtype);
    if (!aligned(x, es) || !aligned(T, es) || !aligned(y, es)) return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    wbmm::Geom g = wbmm::make_geom(*desc);
    int launches = 0, path = WBMM_PATH_NONE;
    cudaError_t e = cudaSuccess;
    const int r = wbmm::nhwc_forward_static_scratch(g, desc->dtype, x, T, y, static_cast<cudaStream_t>(cuda_stream),
                                                    &launches, &path, &e);
    g_launches += launches;
    if (r == 1) {
        snprintf(t_last_error, sizeof(t_last_error),
                 "wbmm_forward_static_scratch serves NHWC bf16/fp16 activations with w in {7, 14}, C and H*W multiples of 8");
        return WBMM_STATUS_UNSUPPORTED;
    }
    if (r == 2) {
        snprintf(t_last_error, sizeof(t_last_error),
                 "wbmm_forward_static_scratch: the activation has %lld bytes, the static scratch holds %zu bytes per temporary",
                 (long long)desc->B * desc->C * desc->H * desc->W * 2, wbmm::static_scratch_limit_bytes());
        return WBMM_STATUS_TOO_LARGE;
    }
    if (e != cudaSuccess) return set_cuda_error(e, "NHWC via static scratch");
    t_last_path = WBMM_PATH_TC_TRANSPOSED;
    return WBMM_STATUS_OK;
}

int wbmm_backward(const wbmm_desc_t* desc, const void* x, const void* T, const void* dy,
                  void* dx, float* dT, void* cuda_stream)
{
    int st = validate(desc);
    if (st != WBMM_STATUS_OK) return st;
    if (desc->C == 0) return WBMM_STATUS_OK;
    if (desc->B == 0) {   // no windows: dT is all zero, dx is empty
        if (dT && !(desc->flags & WBMM_FLAG_ACCUMULATE_DT)) {
            if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
            size_t n = sizeof(float) * (size_t)desc->C * (2 * desc->w - 1) * (2 * desc->w - 1);
            cudaError_t e = cudaMemsetAsync(dT, 0, n, static_cast<cudaStream_t>(cuda_stream));
            if (e != cudaSuccess) return set_cuda_error(e, "memset dT");
        }
        return WBMM_STATUS_OK;
    }
    if (!dy || (dx && !T) || (dT && !x) || (dx && dx == dy)) return WBMM_STATUS_INVALID_ARGUMENT;
    const size_t es = elem_size(desc->dtype);
    if (!aligned(dy, es) || (x && !aligned(x, es)) || (T && !aligned(T, es)) || (dx && !aligned(dx, es)) ||
        (dT && !aligned(dT, 4)))
        return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    wbmm::Geom g = wbmm::make_geom(*desc);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (dx && dT && !(desc->flags & WBMM_FLAG_NO_FORK)) {
        SideStream* ss = side_stream(stream);
        if (ss && cudaEventRecord(ss->fork, stream) == cudaSuccess && cudaStreamWaitEvent(ss->s, ss->fork, 0) == cudaSuccess) {
            const int st_dt = grad_table_on(desc, g, x, dy, dT, ss->s);
            const int path_dt = t_last_path;
            // dX = W_c^T dY on the caller's stream, then the join -- whatever the two returned
            const int st_dx = apply(desc, g, dy, T, dx, true, stream);
            cudaError_t e = cudaEventRecord(ss->join, ss->s);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, ss->join, 0);
            if (st_dx != WBMM_STATUS_OK) return st_dx;
            if (st_dt != WBMM_STATUS_OK) return st_dt;
            if (e != cudaSuccess) return set_cuda_error(e, "join of the table-gradient stream");
            t_last_path = path_dt;
            return WBMM_STATUS_OK;
        }
        cudaGetLastError();          // no side stream: one after the other below
    }
    if (dx) {
        // dX = W_c^T dY: the forward operator with the table index reversed (k -> nb-1-k)
        st = apply(desc, g, dy, T, dx, true, stream);
        if (st != WBMM_STATUS_OK) return st;
    }
    if (dT) {
        st = grad_table_on(desc, g, x, dy, dT, stream);
        if (st != WBMM_STATUS_OK) return st;
    }
    return WBMM_STATUS_OK;
}

// Rectangular windows: desc->w is w_h, w_w is passed beside it.
static int validate_rect(const wbmm_desc_t* d, int w_w)
{
    if (!d) return WBMM_STATUS_INVALID_ARGUMENT;
    if (d->B < 0 || d->C < 0 || d->H < 1 || d->W < 1 || d->w < 1 || w_w < 1) return WBMM_STATUS_INVALID_ARGUMENT;
    if (d->shift_h < 0 || d->shift_w < 0 || d->shift_h >= d->w || d->shift_w >= w_w) return WBMM_STATUS_INVALID_ARGUMENT;
    if (d->dtype != WBMM_DTYPE_F32 && d->dtype != WBMM_DTYPE_BF16 && d->dtype != WBMM_DTYPE_F16) return WBMM_STATUS_INVALID_ARGUMENT;
    if (d->layout != WBMM_LAYOUT_NCHW && d->layout != WBMM_LAYOUT_NHWC) return WBMM_STATUS_INVALID_ARGUMENT;
    long long n = (long long)d->B * d->C;
    if (n > (1ll << 40) / ((long long)d->H * d->W)) return WBMM_STATUS_UNSUPPORTED;
    return WBMM_STATUS_OK;
}

int wbmm_forward_rect(const wbmm_desc_t* desc, int32_t w_w, const void* x, const void* T, void* y, void* cuda_stream)
{
    if (desc && w_w == desc->w) return wbmm_forward(desc, x, T, y, cuda_stream);      // square: the tensor-core kernels
    int st = validate_rect(desc, w_w);
    if (st != WBMM_STATUS_OK) return st;
    if (desc->B == 0 || desc->C == 0) return WBMM_STATUS_OK;
    if (!x || !T || !y || x == y) return WBMM_STATUS_INVALID_ARGUMENT;
    const size_t es = elem_size(desc->dtype);
    if (!aligned(x, es) || !aligned(T, es) || !aligned(y, es)) return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    if (!wbmm::rect_supported(*desc, w_w)) return WBMM_STATUS_UNSUPPORTED;
    int launches = 0;
    cudaError_t e = wbmm::rect_forward(*desc, w_w, x, T, y, false, static_cast<cudaStream_t>(cuda_stream), &launches);
    g_launches += launches;
    if (e != cudaSuccess) return set_cuda_error(e, "rect_forward");
    t_last_path = WBMM_PATH_SIMT;
    return WBMM_STATUS_OK;
}

int wbmm_backward_rect(const wbmm_desc_t* desc, int32_t w_w, const void* x, const void* T, const void* dy,
                       void* dx, float* dT, void* cuda_stream)
{
    if (desc && w_w == desc->w) return wbmm_backward(desc, x, T, dy, dx, dT, cuda_stream);
    int st = validate_rect(desc, w_w);
    if (st != WBMM_STATUS_OK) return st;
    if (desc->C == 0) return WBMM_STATUS_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const long long nb = (2ll * desc->w - 1) * (2ll * w_w - 1);
    if (dT && !aligned(dT, 4)) return WBMM_STATUS_MISALIGNED;
    if (desc->B > 0 && (!dy || (dx && !T) || (dT && !x) || (dx && dx == dy))) return WBMM_STATUS_INVALID_ARGUMENT;
    const size_t es = elem_size(desc->dtype);
    if (desc->B > 0 && (!aligned(dy, es) || (x && !aligned(x, es)) || (T && !aligned(T, es)) || (dx && !aligned(dx, es))))
        return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    if (desc->B > 0 && !wbmm::rect_supported(*desc, w_w)) return WBMM_STATUS_UNSUPPORTED;
    int launches = 0;
    cudaError_t e = cudaSuccess;
    if (dT && !(desc->flags & WBMM_FLAG_ACCUMULATE_DT)) e = wbmm::simt_zero_f32(dT, (long long)desc->C * nb, stream, &launches);
    if (desc->B > 0) {
        if (e == cudaSuccess && dx) e = wbmm::rect_forward(*desc, w_w, dy, T, dx, true, stream, &launches);
        if (e == cudaSuccess && dT) e = wbmm::rect_grad_table(*desc, w_w, x, dy, dT, stream, &launches);
    }
    g_launches += launches;
    if (e != cudaSuccess) return set_cuda_error(e, "rect backward");
    t_last_path = WBMM_PATH_SIMT;
    return WBMM_STATUS_OK;
}

int wbmm_hier_forward(const wbmm_desc_t* desc, const void* x, const void* Tg, const void* Tl, void* y,
                      int transpose, void* cuda_stream)
{
    int st = validate(desc);
    if (st != WBMM_STATUS_OK) return st;
    if (desc->w % 2 != 0) return WBMM_STATUS_INVALID_ARGUMENT;
    if (desc->B == 0 || desc->C == 0) return WBMM_STATUS_OK;
    if (!x || !Tg || !Tl || !y || x == y) return WBMM_STATUS_INVALID_ARGUMENT;
    const size_t es = elem_size(desc->dtype);
    if (!aligned(x, es) || !aligned(Tg, es) || !aligned(Tl, es) || !aligned(y, es)) return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    wbmm::Geom g = wbmm::make_geom(*desc);
    int launches = 0, path = WBMM_PATH_NONE;
    // what the tensor-core kernel does not take (fp32, w != 14, planes no copy scheme moves, NHWC without scratch): the
    // FFMA kernel of wbmm_rect.cu, the same operator in one pass
    auto ffma = [&]() -> int {
        if (!wbmm::hier_simt_supported(*desc)) return WBMM_STATUS_UNSUPPORTED;
        int l = 0;
        cudaError_t e = wbmm::hier_simt_forward(*desc, x, Tg, Tl, y, transpose != 0, static_cast<cudaStream_t>(cuda_stream), &l);
        g_launches += l;
        if (e != cudaSuccess) return set_cuda_error(e, "hier_simt_forward");
        t_last_path = WBMM_PATH_SIMT;
        return WBMM_STATUS_OK;
    };
    if (desc->flags & WBMM_FLAG_FORCE_SIMT) return ffma();
    if (g.layout == WBMM_LAYOUT_NHWC) {
        // the transposition route of wbmm_forward around the same kernel
        cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
        wbmm::Geom gn = g;
        gn.layout = WBMM_LAYOUT_NCHW;
        void* const aligned16 = reinterpret_cast<void*>(256);
        if (!nhwc_scratch_candidate(desc, g) || !wbmm::tc_hier_supported(gn, desc->dtype, aligned16, aligned16) ||
            !wbmm::transpose16_supported((long long)g.H * g.W, g.C, x, y))
            return ffma();
        const size_t nbytes = (size_t)g.B * g.C * g.H * g.W * 2;
        AsyncScratch xt(stream), yt(stream);
        if (xt.alloc(nbytes) != cudaSuccess || yt.alloc(nbytes) != cudaSuccess) {
            cudaGetLastError();
            return ffma();
        }
        cudaError_t e = wbmm::transpose16(x, xt.p, g.B, g.H * g.W, g.C, stream, &launches);
        if (e == cudaSuccess) e = wbmm::tc_forward(gn, desc->dtype, xt.p, Tg, Tl, yt.p, transpose != 0, stream, &launches, &path);
        if (e == cudaSuccess) e = wbmm::transpose16(yt.p, y, g.B, g.C, g.H * g.W, stream, &launches);
        g_launches += launches;
        if (e != cudaSuccess) return set_cuda_error(e, "hierarchical forward, NHWC via NCHW scratch");
        t_last_path = WBMM_PATH_TC_TRANSPOSED;
        return WBMM_STATUS_OK;
    }
    if (!wbmm::tc_hier_supported(g, desc->dtype, x, y)) return ffma();
    cudaError_t e = wbmm::tc_forward(g, desc->dtype, x, Tg, Tl, y, transpose != 0, static_cast<cudaStream_t>(cuda_stream),
                                     &launches, &path);
    g_launches += launches;
    if (e != cudaSuccess) return set_cuda_error(e, "tc_forward (hierarchical)");
    t_last_path = path;
    return WBMM_STATUS_OK;
}

int wbmm_hier_backward(const wbmm_desc_t* desc, const void* x, const void* Tg, const void* Tl, const void* dy,
                       void* dx, float* dTg, float* dTl, void* cuda_stream)
{
    int st = validate(desc);
    if (st != WBMM_STATUS_OK) return st;
    if (desc->w % 2 != 0) return WBMM_STATUS_INVALID_ARGUMENT;
    if ((dTg == nullptr) != (dTl == nullptr)) return WBMM_STATUS_INVALID_ARGUMENT;   // the two tables go together
    if (desc->C == 0) return WBMM_STATUS_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int wl = desc->w / 2;
    const size_t ng = sizeof(float) * (size_t)desc->C * (2 * desc->w - 1) * (2 * desc->w - 1);
    const size_t nl = sizeof(float) * (size_t)desc->C * (2 * wl - 1) * (2 * wl - 1);
    if (dTg && !aligned(dTg, 4)) return WBMM_STATUS_MISALIGNED;
    if (dTl && !aligned(dTl, 4)) return WBMM_STATUS_MISALIGNED;
    if (dTg && !(desc->flags & WBMM_FLAG_ACCUMULATE_DT)) {
        if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
        int zl = 0;
        cudaError_t e = wbmm::simt_zero_f32(dTg, (long long)(ng / sizeof(float)), stream, &zl);
        if (e == cudaSuccess) e = wbmm::simt_zero_f32(dTl, (long long)(nl / sizeof(float)), stream, &zl);
        g_launches += zl;
        if (e != cudaSuccess) return set_cuda_error(e, "zero dT (hierarchical)");
    }
    if (desc->B == 0) return WBMM_STATUS_OK;
    if (!dy || (dx && (!Tg || !Tl)) || (dTg && !x) || (dx && dx == dy)) return WBMM_STATUS_INVALID_ARGUMENT;
    const size_t es = elem_size(desc->dtype);
    if (!aligned(dy, es) || (x && !aligned(x, es)) || (Tg && !aligned(Tg, es)) || (Tl && !aligned(Tl, es)) ||
        (dx && !aligned(dx, es)))
        return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    wbmm::Geom g = wbmm::make_geom(*desc);
    // check both halves before launching either
    const bool nhwc = g.layout == WBMM_LAYOUT_NHWC;
    wbmm::Geom gn = g;
    gn.layout = WBMM_LAYOUT_NCHW;
    void* const aligned16 = reinterpret_cast<void*>(256);
    bool tc_ok = !(desc->flags & WBMM_FLAG_FORCE_SIMT);
    if (nhwc) {
        if (!nhwc_scratch_candidate(desc, g)) tc_ok = false;
        if (dx && (!wbmm::tc_hier_supported(gn, desc->dtype, aligned16, aligned16) ||
                   !wbmm::transpose16_supported((long long)g.H * g.W, g.C, dy, dx)))
            tc_ok = false;
        if (dTg && (g.w != 14 || !wbmm::tc_grad_table_supported(gn, desc->dtype, aligned16, aligned16) ||
                    !wbmm::transpose16_supported((long long)g.H * g.W, g.C, x, dy)))
            tc_ok = false;
    } else {
        if (dx && !wbmm::tc_hier_supported(g, desc->dtype, dy, dx)) tc_ok = false;
        if (dTg && (g.w != 14 || !wbmm::tc_grad_table_supported(g, desc->dtype, x, dy))) tc_ok = false;
    }
    if (!tc_ok) {
        // the FFMA kernels of wbmm_rect.cu: dx = the transposed operator, both table gradients as windowed correlations
        if (!wbmm::hier_simt_supported(*desc)) return WBMM_STATUS_UNSUPPORTED;
        int l = 0;
        cudaError_t e = cudaSuccess;
        if (dx) e = wbmm::hier_simt_forward(*desc, dy, Tg, Tl, dx, true, stream, &l);
        if (e == cudaSuccess && dTg) e = wbmm::hier_simt_grad_tables(*desc, x, dy, dTg, dTl, stream, &l);
        g_launches += l;
        if (e != cudaSuccess) return set_cuda_error(e, "hierarchical backward (FFMA)");
        t_last_path = WBMM_PATH_SIMT;
        return WBMM_STATUS_OK;
    }
    // both table gradients on `sdt` (dTg, dTl were cleared on the caller's stream above)
    auto table_gradients = [&](cudaStream_t sdt) -> int {
        if (dTg && nhwc) {
            const size_t nbytes = (size_t)g.B * g.C * g.H * g.W * 2;
            AsyncScratch xt(sdt), gt(sdt);
            if (xt.alloc(nbytes) != cudaSuccess || gt.alloc(nbytes) != cudaSuccess) {
                cudaGetLastError();
                return WBMM_STATUS_UNSUPPORTED;
            }
            int launches = 0, path = WBMM_PATH_NONE;
            cudaError_t e = wbmm::transpose16(x, xt.p, g.B, g.H * g.W, g.C, sdt, &launches);
            if (e == cudaSuccess) e = wbmm::transpose16(dy, gt.p, g.B, g.H * g.W, g.C, sdt, &launches);
            if (e == cudaSuccess) e = wbmm::tc_grad_table(gn, desc->dtype, xt.p, gt.p, dTg, sdt, &launches, &path, dTl);
            g_launches += launches;
            if (e != cudaSuccess) return set_cuda_error(e, "hierarchical table gradients, NHWC via NCHW scratch");
            t_last_path = WBMM_PATH_TC_TRANSPOSED;
        } else if (dTg) {
            int launches = 0, path = WBMM_PATH_NONE;
            cudaError_t e = wbmm::tc_grad_table(g, desc->dtype, x, dy, dTg, sdt, &launches, &path, dTl);
            g_launches += launches;
            if (e != cudaSuccess) return set_cuda_error(e, "tc_grad_table (hierarchical)");
            t_last_path = path;
        }
        return WBMM_STATUS_OK;
    };
    if (dx && dTg && !(desc->flags & WBMM_FLAG_NO_FORK)) {
        // as wbmm_backward: the table gradients on the internal stream, forked from and joined into the caller's
        SideStream* ss = side_stream(stream);
        if (ss && cudaEventRecord(ss->fork, stream) == cudaSuccess && cudaStreamWaitEvent(ss->s, ss->fork, 0) == cudaSuccess) {
            const int st_dt = table_gradients(ss->s);
            const int path_dt = t_last_path;
            const int st_dx = wbmm_hier_forward(desc, dy, Tg, Tl, dx, 1, cuda_stream);
            cudaError_t e = cudaEventRecord(ss->join, ss->s);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, ss->join, 0);
            if (st_dx != WBMM_STATUS_OK) return st_dx;
            if (st_dt != WBMM_STATUS_OK) return st_dt;
            if (e != cudaSuccess) return set_cuda_error(e, "join of the table-gradient stream");
            t_last_path = path_dt;
            return WBMM_STATUS_OK;
        }
        cudaGetLastError();
    }
    if (dx) {
        st = wbmm_hier_forward(desc, dy, Tg, Tl, dx, 1, cuda_stream);
        if (st != WBMM_STATUS_OK) return st;
    }
    if (dTg) {
        st = table_gradients(stream);
        if (st != WBMM_STATUS_OK) return st;
    }
    return WBMM_STATUS_OK;
}

int wbmm_forward_fused(const wbmm_desc_t* desc, const void* x, const void* T, const void* bias, float identity,
                       void* y, int transpose, void* cuda_stream)
{
    int st = validate(desc);
    if (st != WBMM_STATUS_OK) return st;
    if (desc->B == 0 || desc->C == 0) return WBMM_STATUS_OK;
    if (!x || !T || !y || x == y) return WBMM_STATUS_INVALID_ARGUMENT;
    if (!(identity == identity) || identity - identity != 0.f) return WBMM_STATUS_INVALID_ARGUMENT;   // NaN / inf
    const size_t es = elem_size(desc->dtype);
    if (!aligned(x, es) || !aligned(T, es) || !aligned(y, es) || (bias && !aligned(bias, es))) return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    // identity rounded to the dtype, as the tensor-core path holds it
    uint32_t ident_bits = 0;
    float ident_f = identity;
    if (identity != 0.f && desc->dtype == WBMM_DTYPE_BF16) { __nv_bfloat16 h = __float2bfloat16_rn(identity); memcpy(&ident_bits, &h, 2); ident_f = __bfloat162float(h); }
    if (identity != 0.f && desc->dtype == WBMM_DTYPE_F16) { __half h = __float2half_rn(identity); memcpy(&ident_bits, &h, 2); ident_f = __half2float(h); }
    // what the pipelined kernel does not take (float32, identity at w != 14, planes no copy scheme moves, NHWC without
    // scratch): the FFMA kernel of wbmm_rect.cu, same operator, one pass
    auto ffma = [&]() -> int {
        if (!wbmm::rect_supported(*desc, desc->w)) return WBMM_STATUS_UNSUPPORTED;
        int l = 0;
        cudaError_t e2 = wbmm::fused_simt_forward(*desc, x, T, bias, ident_f, y, transpose != 0, static_cast<cudaStream_t>(cuda_stream), &l);
        g_launches += l;
        if (e2 != cudaSuccess) return set_cuda_error(e2, "fused_simt_forward");
        t_last_path = WBMM_PATH_SIMT;
        return WBMM_STATUS_OK;
    };
    if ((desc->flags & WBMM_FLAG_FORCE_SIMT) || (desc->dtype != WBMM_DTYPE_BF16 && desc->dtype != WBMM_DTYPE_F16)) return ffma();
    if (identity != 0.f && desc->w != 14) return ffma();              // the identity block exists in the w = 14 library only
    wbmm::Geom g = wbmm::make_geom(*desc);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int launches = 0, path = WBMM_PATH_NONE;
    cudaError_t e;
    if (g.layout == WBMM_LAYOUT_NHWC) {
        // the transposition route of wbmm_forward around the same fused kernel
        wbmm::Geom gn = g;
        gn.layout = WBMM_LAYOUT_NCHW;
        void* const aligned16 = reinterpret_cast<void*>(256);
        if (!nhwc_scratch_candidate(desc, g) || !wbmm::tc_bulk_supported(gn, desc->dtype, aligned16, aligned16) ||
            !wbmm::transpose16_supported((long long)g.H * g.W, g.C, x, y))
            return ffma();
        const size_t nbytes = (size_t)g.B * g.C * g.H * g.W * 2;
        AsyncScratch xt(stream), yt(stream);
        if (xt.alloc(nbytes) != cudaSuccess || yt.alloc(nbytes) != cudaSuccess) {
            cudaGetLastError();
            return ffma();
        }
        e = wbmm::transpose16(x, xt.p, g.B, g.H * g.W, g.C, stream, &launches);
        if (e == cudaSuccess)
            e = wbmm::tc_forward(gn, desc->dtype, xt.p, T, nullptr, yt.p, transpose != 0, stream, &launches, &path, bias, ident_bits);
        if (e == cudaSuccess) e = wbmm::transpose16(yt.p, y, g.B, g.C, g.H * g.W, stream, &launches);
        g_launches += launches;
        if (e != cudaSuccess) return set_cuda_error(e, "fused forward, NHWC via NCHW scratch");
        t_last_path = WBMM_PATH_TC_TRANSPOSED;
        return WBMM_STATUS_OK;
    }
    if (!wbmm::tc_bulk_supported(g, desc->dtype, x, y)) return ffma();
    e = wbmm::tc_forward(g, desc->dtype, x, T, nullptr, y, transpose != 0, stream, &launches, &path, bias, ident_bits);
    g_launches += launches;
    if (e != cudaSuccess) return set_cuda_error(e, "tc_forward (fused)");
    t_last_path = path;
    return WBMM_STATUS_OK;
}

int wbmm_forward_matrix(const wbmm_desc_t* desc, const void* x, const void* M, const void* bias, void* y,
                        int transpose, void* cuda_stream)
{
    int st = validate(desc);
    if (st != WBMM_STATUS_OK) return st;
    if (desc->B == 0 || desc->C == 0) return WBMM_STATUS_OK;
    if (!x || !M || !y || x == y) return WBMM_STATUS_INVALID_ARGUMENT;
    const size_t es = elem_size(desc->dtype);
    if (!aligned(x, es) || !aligned(M, es) || !aligned(y, es) || (bias && !aligned(bias, es))) return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    wbmm::Geom g = wbmm::make_geom(*desc);
    if ((desc->flags & WBMM_FLAG_FORCE_SIMT) || !wbmm::tc_forward_supported(g, desc->dtype, x, y)) {
        // float32, window sizes without a tensor-core kernel: the FFMA kernel of wbmm_rect.cu reads M_c from global memory
        if (!wbmm::rect_supported(*desc, desc->w)) return WBMM_STATUS_UNSUPPORTED;
        int l = 0;
        cudaError_t e2 = wbmm::matrix_simt_forward(*desc, x, M, bias, y, transpose != 0, static_cast<cudaStream_t>(cuda_stream), &l);
        g_launches += l;
        if (e2 != cudaSuccess) return set_cuda_error(e2, "matrix_simt_forward");
        t_last_path = WBMM_PATH_SIMT;
        return WBMM_STATUS_OK;
    }
    int launches = 0, path = WBMM_PATH_NONE;
    cudaError_t e = wbmm::tc_forward_matrix(g, desc->dtype, x, M, bias, y, transpose != 0,
                                            static_cast<cudaStream_t>(cuda_stream), &launches, &path);
    g_launches += launches;
    if (e != cudaSuccess) return set_cuda_error(e, "tc_forward_matrix");
    t_last_path = path;
    return WBMM_STATUS_OK;
}

// 3-D windows (reading A23): desc gives B, C, H, W, w = w_h, shift_h / shift_w, dtype, layout (NCHW = [B][C][D][H][W],
// NHWC = [B][D][H][W][C]); depth, the other two window sides and the depth shift are arguments.
static int validate_win3d(const wbmm_desc_t* d, int D, int w_d, int w_w, int shift_d)
{
    int st = validate_rect(d, w_w);
    if (st != WBMM_STATUS_OK) return st;
    if (D < 1 || w_d < 1 || shift_d < 0 || shift_d >= w_d) return WBMM_STATUS_INVALID_ARGUMENT;
    return WBMM_STATUS_OK;
}

int wbmm_forward_win3d(const wbmm_desc_t* desc, int32_t D, int32_t w_d, int32_t w_w, int32_t shift_d, const void* x, const void* T,
                       void* y, void* cuda_stream)
{
    int st = validate_win3d(desc, D, w_d, w_w, shift_d);
    if (st != WBMM_STATUS_OK) return st;
    if (desc->B == 0 || desc->C == 0) return WBMM_STATUS_OK;
    if (!x || !T || !y || x == y) return WBMM_STATUS_INVALID_ARGUMENT;
    const size_t es = elem_size(desc->dtype);
    if (!aligned(x, es) || !aligned(T, es) || !aligned(y, es)) return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    if (!wbmm::win3d_supported(*desc, D, w_d, w_w)) return WBMM_STATUS_UNSUPPORTED;
    int launches = 0;
    cudaError_t e = wbmm::win3d_forward(*desc, D, w_d, w_w, shift_d, x, T, y, false, static_cast<cudaStream_t>(cuda_stream), &launches);
    g_launches += launches;
    if (e != cudaSuccess) return set_cuda_error(e, "win3d_forward");
    t_last_path = WBMM_PATH_SIMT;
    return WBMM_STATUS_OK;
}

int wbmm_backward_win3d(const wbmm_desc_t* desc, int32_t D, int32_t w_d, int32_t w_w, int32_t shift_d, const void* x, const void* T,
                        const void* dy, void* dx, float* dT, void* cuda_stream)
{
    int st = validate_win3d(desc, D, w_d, w_w, shift_d);
    if (st != WBMM_STATUS_OK) return st;
    if (desc->C == 0) return WBMM_STATUS_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const long long nb = (2ll * w_d - 1) * (2ll * desc->w - 1) * (2ll * w_w - 1);
    if (dT && !aligned(dT, 4)) return WBMM_STATUS_MISALIGNED;
    if (desc->B > 0 && (!dy || (dx && !T) || (dT && !x) || (dx && dx == dy))) return WBMM_STATUS_INVALID_ARGUMENT;
    const size_t es = elem_size(desc->dtype);
    if (desc->B > 0 && (!aligned(dy, es) || (x && !aligned(x, es)) || (T && !aligned(T, es)) || (dx && !aligned(dx, es))))
        return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    if (!wbmm::win3d_supported(*desc, D, w_d, w_w)) return WBMM_STATUS_UNSUPPORTED;
    int launches = 0;
    cudaError_t e = cudaSuccess;
    if (dT && !(desc->flags & WBMM_FLAG_ACCUMULATE_DT)) e = wbmm::simt_zero_f32(dT, (long long)desc->C * nb, stream, &launches);
    if (desc->B > 0) {
        if (e == cudaSuccess && dx) e = wbmm::win3d_forward(*desc, D, w_d, w_w, shift_d, dy, T, dx, true, stream, &launches);
        if (e == cudaSuccess && dT) e = wbmm::win3d_grad_table(*desc, D, w_d, w_w, shift_d, x, dy, dT, stream, &launches);
    }
    g_launches += launches;
    if (e != cudaSuccess) return set_cuda_error(e, "win3d backward");
    t_last_path = WBMM_PATH_SIMT;
    return WBMM_STATUS_OK;
}

// INT8 / FP8 (E4M3) forward: the same kernels and routes, 8-bit elements either way.
static int forward_8bit(const wbmm_desc_t* desc, const int8_t* x, const int8_t* T, const float* scale, void* y, void* cuda_stream, bool fp8)
{
    if (!desc) return WBMM_STATUS_INVALID_ARGUMENT;
    wbmm_desc_t d = *desc;
    d.dtype = WBMM_DTYPE_F32;          // the element type is fixed by this entry point: desc->dtype is not read
    int st = validate(&d);
    if (st != WBMM_STATUS_OK) return st;
    if (d.B == 0 || d.C == 0) return WBMM_STATUS_OK;
    if (!x || !T || !y || static_cast<const void*>(x) == y) return WBMM_STATUS_INVALID_ARGUMENT;
    if ((scale && !aligned(scale, 4)) || (!scale && !aligned(y, 4))) return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    wbmm::Geom g = wbmm::make_geom(d);
    if (!wbmm::tc_i8_supported(g)) {
        snprintf(t_last_error, sizeof(t_last_error),
                 "8-bit forward: w must be 7 or 14 with at most 128 windows across (w = %d, %d windows across)", g.w, g.nww);
        return WBMM_STATUS_UNSUPPORTED;
    }
    int launches = 0, path = WBMM_PATH_NONE;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (g.layout == WBMM_LAYOUT_NHWC && !(desc->flags & WBMM_FLAG_NO_SCRATCH)) {
        // NHWC: transposition passes around the NCHW bulk-copy kernel (a channel-major tile read straight from NHWC
        // touches one 32-byte sector per byte: 755 us against ~100 for the three passes at B128 C96 56x56)
        const long long hw = (long long)g.H * g.W;
        wbmm::Geom gn = g;
        gn.layout = WBMM_LAYOUT_NCHW;
        const bool y_ok = scale ? wbmm::transpose8_supported(g.C, hw, y, y) : wbmm::transpose32_supported(g.C, hw, y, y);
        if (wbmm::transpose8_supported(hw, g.C, x, x) && y_ok) {
            const size_t n = (size_t)g.B * g.C * hw;
            AsyncScratch xt(stream), yt(stream);
            if (xt.alloc(n) == cudaSuccess && yt.alloc(n * (scale ? 1 : 4)) == cudaSuccess) {
                cudaError_t e = wbmm::transpose8(x, xt.p, g.B, (int)hw, g.C, stream, &launches);
                if (e == cudaSuccess) e = wbmm::tc_i8_forward(gn, static_cast<const int8_t*>(xt.p), T, scale, yt.p, stream, &launches, &path, fp8);
                if (e == cudaSuccess)
                    e = scale ? wbmm::transpose8(yt.p, y, g.B, g.C, (int)hw, stream, &launches)
                              : wbmm::transpose32(yt.p, y, g.B, g.C, (int)hw, stream, &launches);
                g_launches += launches;
                if (e != cudaSuccess) return set_cuda_error(e, "int8 NHWC via NCHW scratch");
                t_last_path = WBMM_PATH_TC_TRANSPOSED;
                return WBMM_STATUS_OK;
            }
            cudaGetLastError();      // no stream-ordered allocator / out of memory: the gather kernel below
        }
    }
    cudaError_t e = wbmm::tc_i8_forward(g, x, T, scale, y, stream, &launches, &path, fp8);
    g_launches += launches;
    if (e != cudaSuccess) return set_cuda_error(e, "tc_i8_forward");
    t_last_path = path;
    return WBMM_STATUS_OK;
}

int wbmm_forward_int8(const wbmm_desc_t* desc, const int8_t* x, const int8_t* T, const float* scale, void* y, void* cuda_stream)
{
    return forward_8bit(desc, x, T, scale, y, cuda_stream, false);
}

int wbmm_forward_fp8(const wbmm_desc_t* desc, const void* x, const void* T, const float* scale, void* y, void* cuda_stream)
{
    return forward_8bit(desc, static_cast<const int8_t*>(x), static_cast<const int8_t*>(T), scale, y, cuda_stream, true);
}

int wbmm_fold_dwconv(const wbmm_desc_t* desc, const void* T, const void* K, int ksize, const float* scale,
                     void* Tout, void* cuda_stream)
{
    if (!desc || desc->C < 0 || desc->w < 1 || desc->w > 64) return WBMM_STATUS_INVALID_ARGUMENT;
    if (desc->dtype != WBMM_DTYPE_F32 && desc->dtype != WBMM_DTYPE_BF16 && desc->dtype != WBMM_DTYPE_F16)
        return WBMM_STATUS_INVALID_ARGUMENT;
    if (ksize < 1 || ksize % 2 == 0 || ksize / 2 > desc->w - 1) return WBMM_STATUS_INVALID_ARGUMENT;
    if (desc->C == 0) return WBMM_STATUS_OK;
    if (!T || !K || !Tout) return WBMM_STATUS_INVALID_ARGUMENT;
    const size_t es = elem_size(desc->dtype);
    if (!aligned(T, es) || !aligned(K, es) || !aligned(Tout, es) || (scale && !aligned(scale, 4))) return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    int launches = 0;
    cudaError_t e = wbmm::simt_fold_dwconv(desc->C, desc->w, ksize, desc->dtype, T, K, scale, Tout,
                                           static_cast<cudaStream_t>(cuda_stream), &launches);
    g_launches += launches;
    if (e != cudaSuccess) return set_cuda_error(e, "fold_dwconv");
    t_last_path = WBMM_PATH_SIMT;
    return WBMM_STATUS_OK;
}

int wbmm_materialize_weight(const wbmm_desc_t* desc, const void* T, void* Wout, void* cuda_stream)
{
    if (!desc || desc->C < 0 || desc->w < 1 || desc->w > 64) return WBMM_STATUS_INVALID_ARGUMENT;
    if (desc->dtype != WBMM_DTYPE_F32 && desc->dtype != WBMM_DTYPE_BF16 && desc->dtype != WBMM_DTYPE_F16)
        return WBMM_STATUS_INVALID_ARGUMENT;
    if (!T || !Wout) return WBMM_STATUS_INVALID_ARGUMENT;
    if (!aligned(T, elem_size(desc->dtype)) || !aligned(Wout, elem_size(desc->dtype))) return WBMM_STATUS_MISALIGNED;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    int launches = 0;
    cudaError_t e = wbmm::simt_materialize(desc->C, desc->w, desc->dtype, T, Wout,
                                           static_cast<cudaStream_t>(cuda_stream), &launches);
    g_launches += launches;
    if (e != cudaSuccess) return set_cuda_error(e, "materialize");
    t_last_path = WBMM_PATH_SIMT;
    return WBMM_STATUS_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// Host-buffer variants: device scratch owned by the library, one internal stream.
namespace {

struct Scratch {
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t n)
    {
        if (n <= cap) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr; cap = 0;
        cudaError_t e = cudaMalloc(&p, n);
        if (e == cudaSuccess) cap = n;
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
};

std::mutex g_host_mutex;
Scratch g_sx, g_sT, g_sy, g_sdy, g_sdT;
cudaStream_t g_host_stream = nullptr;

constexpr int kHostChunks = 32;   // at most; see host_chunks()
cudaStream_t g_s_kernel = nullptr, g_s_out = nullptr;
cudaEvent_t g_ev_in[kHostChunks] = {}, g_ev_k[kHostChunks] = {};

// Chunks per call: enough that the un-overlapped head (first upload) and tail (last download) are small, few enough
// that per-copy set-up does not show.
// Measured on cfg3 (77 MB each way, pinned buffers), ms per call: 2 chunks 2.21, 4: 1.96, 8: 1.91-1.97, 12: 1.99,
// 16: 2.04, 32: 2.41.
int host_chunks() { return 8; }

cudaError_t host_pipeline_init()
{
    if (g_s_kernel) return cudaSuccess;
    cudaError_t e = cudaStreamCreateWithFlags(&g_s_kernel, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&g_s_out, cudaStreamNonBlocking);
    for (int i = 0; i < kHostChunks && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&g_ev_in[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&g_ev_k[i], cudaEventDisableTiming);
    }
    return e;
}

void host_pipeline_release()
{
    if (g_s_kernel) { cudaStreamDestroy(g_s_kernel); g_s_kernel = nullptr; }
    if (g_s_out) { cudaStreamDestroy(g_s_out); g_s_out = nullptr; }
    for (int i = 0; i < kHostChunks; ++i) {
        if (g_ev_in[i]) { cudaEventDestroy(g_ev_in[i]); g_ev_in[i] = nullptr; }
        if (g_ev_k[i]) { cudaEventDestroy(g_ev_k[i]); g_ev_k[i] = nullptr; }
    }
}

cudaError_t host_stream(cudaStream_t* s)
{
    if (!g_host_stream) {
        cudaError_t e = cudaStreamCreateWithFlags(&g_host_stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) return e;
    }
    *s = g_host_stream;
    return cudaSuccess;
}

#define WBMM_TRY(expr, where)                                   \
    do {                                                        \
        cudaError_t e_ = (expr);                                \
        if (e_ != cudaSuccess) return set_cuda_error(e_, where); \
    } while (0)

}  // namespace

extern "C" {

int wbmm_forward_host(const wbmm_desc_t* desc, const void* x_host, const void* T_host, void* y_host)
{
    int st = validate(desc);
    if (st != WBMM_STATUS_OK) return st;
    if (!x_host || !T_host || !y_host) return WBMM_STATUS_INVALID_ARGUMENT;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    std::lock_guard<std::mutex> lock(g_host_mutex);
    wbmm::Geom g = wbmm::make_geom(*desc);
    const size_t es = elem_size(desc->dtype);
    const size_t nact = (size_t)g.B * g.C * g.H * g.W * es, ntab = (size_t)g.C * g.nb * es;
    cudaStream_t s;
    WBMM_TRY(host_stream(&s), "stream");
    if (nact == 0) return WBMM_STATUS_OK;
    WBMM_TRY(g_sx.reserve(nact), "cudaMalloc x");
    WBMM_TRY(g_sy.reserve(nact), "cudaMalloc y");
    WBMM_TRY(g_sT.reserve(ntab), "cudaMalloc T");
    // The batch is cut into chunks that flow through three streams -- H2D, kernels, D2H -- so that the
    // upload of chunk i+1, the kernels of chunk i and the download of chunk i-1 overlap (PCIe is full
    // duplex; with pinned host buffers the call takes about max(H2D, D2H) instead of their sum).
    WBMM_TRY(host_pipeline_init(), "streams");
    const int nchunk = nact >= (8u << 20) ? (g.B < host_chunks() ? g.B : host_chunks()) : 1;
    const size_t per_image = nact / (size_t)g.B;
    WBMM_TRY(cudaMemcpyAsync(g_sT.p, T_host, ntab, cudaMemcpyHostToDevice, s), "H2D T");
    for (int i = 0; i < nchunk; ++i) {
        const int b0 = (int)((long long)g.B * i / nchunk), b1 = (int)((long long)g.B * (i + 1) / nchunk);
        if (b1 == b0) continue;
        const size_t off = per_image * b0, len = per_image * (b1 - b0);
        WBMM_TRY(cudaMemcpyAsync((char*)g_sx.p + off, (const char*)x_host + off, len, cudaMemcpyHostToDevice, s), "H2D x");
        WBMM_TRY(cudaEventRecord(g_ev_in[i], s), "event");
        WBMM_TRY(cudaStreamWaitEvent(g_s_kernel, g_ev_in[i], 0), "wait");
        wbmm_desc_t dc = *desc;
        dc.B = b1 - b0;
        wbmm::Geom gc = wbmm::make_geom(dc);
        st = apply(&dc, gc, (char*)g_sx.p + off, g_sT.p, (char*)g_sy.p + off, false, g_s_kernel);
        if (st != WBMM_STATUS_OK) return st;
        WBMM_TRY(cudaEventRecord(g_ev_k[i], g_s_kernel), "event");
        WBMM_TRY(cudaStreamWaitEvent(g_s_out, g_ev_k[i], 0), "wait");
        WBMM_TRY(cudaMemcpyAsync((char*)y_host + off, (char*)g_sy.p + off, len, cudaMemcpyDeviceToHost, g_s_out), "D2H y");
    }
    WBMM_TRY(cudaStreamSynchronize(g_s_out), "sync");
    WBMM_TRY(cudaStreamSynchronize(s), "sync");
    return WBMM_STATUS_OK;
}

int wbmm_backward_host(const wbmm_desc_t* desc, const void* x_host, const void* T_host,
                       const void* dy_host, void* dx_host, float* dT_host)
{
    int st = validate(desc);
    if (st != WBMM_STATUS_OK) return st;
    if (!dy_host || (dx_host && !T_host) || (dT_host && !x_host)) return WBMM_STATUS_INVALID_ARGUMENT;
    if (device_state() < 0) return WBMM_STATUS_NO_DEVICE;
    std::lock_guard<std::mutex> lock(g_host_mutex);
    wbmm::Geom g = wbmm::make_geom(*desc);
    const size_t es = elem_size(desc->dtype);
    const size_t nact = (size_t)g.B * g.C * g.H * g.W * es, ntab = (size_t)g.C * g.nb * es;
    const size_t ngrad = (size_t)g.C * g.nb * sizeof(float);
    cudaStream_t s;
    WBMM_TRY(host_stream(&s), "stream");
    if (nact == 0 || (!dx_host && !dT_host)) {
        if (dT_host && !(desc->flags & WBMM_FLAG_ACCUMULATE_DT)) memset(dT_host, 0, ngrad);
        return WBMM_STATUS_OK;
    }
    WBMM_TRY(g_sdy.reserve(nact), "cudaMalloc dy");
    WBMM_TRY(cudaMemcpyAsync(g_sdy.p, dy_host, nact, cudaMemcpyHostToDevice, s), "H2D dy");
    if (dT_host) {
        WBMM_TRY(g_sx.reserve(nact), "cudaMalloc x");
        WBMM_TRY(g_sdT.reserve(ngrad), "cudaMalloc dT");
        WBMM_TRY(cudaMemcpyAsync(g_sx.p, x_host, nact, cudaMemcpyHostToDevice, s), "H2D x");
        if (desc->flags & WBMM_FLAG_ACCUMULATE_DT)
            WBMM_TRY(cudaMemcpyAsync(g_sdT.p, dT_host, ngrad, cudaMemcpyHostToDevice, s), "H2D dT");
    }
    if (dx_host) {
        WBMM_TRY(g_sT.reserve(ntab), "cudaMalloc T");
        WBMM_TRY(g_sy.reserve(nact), "cudaMalloc dx");
        WBMM_TRY(cudaMemcpyAsync(g_sT.p, T_host, ntab, cudaMemcpyHostToDevice, s), "H2D T");
    }
    st = wbmm_backward(desc, dT_host ? g_sx.p : nullptr, dx_host ? g_sT.p : nullptr, g_sdy.p,
                       dx_host ? g_sy.p : nullptr, dT_host ? (float*)g_sdT.p : nullptr, s);
    if (st != WBMM_STATUS_OK) return st;
    if (dx_host) WBMM_TRY(cudaMemcpyAsync(dx_host, g_sy.p, nact, cudaMemcpyDeviceToHost, s), "D2H dx");
    if (dT_host) WBMM_TRY(cudaMemcpyAsync(dT_host, g_sdT.p, ngrad, cudaMemcpyDeviceToHost, s), "D2H dT");
    WBMM_TRY(cudaStreamSynchronize(s), "sync");
    return WBMM_STATUS_OK;
}

void wbmm_release(void)
{
    std::lock_guard<std::mutex> lock(g_host_mutex);
    g_sx.release(); g_sT.release(); g_sy.release(); g_sdy.release(); g_sdT.release();
    if (g_host_stream) { cudaStreamDestroy(g_host_stream); g_host_stream = nullptr; }
    host_pipeline_release();
    scratch_pools_release();
    // the calling thread's fork / join streams of wbmm_backward (other host threads keep theirs until they exit)
    for (int d = 0; d < kMaxDevices; ++d)
        if (t_side[d].s) {
            cudaEventDestroy(t_side[d].fork);
            cudaEventDestroy(t_side[d].join);
            cudaStreamDestroy(t_side[d].s);
            t_side[d] = SideStream();
        }
}

int wbmm_last_path(void) { return t_last_path; }
uint64_t wbmm_launch_count(void) { return g_launches.load(); }
const char* wbmm_last_error_string(void) { return t_last_error; }
int wbmm_version(void) { return WBMM_VERSION; }

const char* wbmm_status_string(int status)
{
    switch (status) {
    case WBMM_STATUS_OK: return "ok";
    case WBMM_STATUS_INVALID_ARGUMENT: return "invalid argument";
    case WBMM_STATUS_UNSUPPORTED: return "unsupported configuration";
    case WBMM_STATUS_NO_DEVICE: return "no sm_100 CUDA device";
    case WBMM_STATUS_CUDA_ERROR: return "CUDA error";
    case WBMM_STATUS_MISALIGNED: return "misaligned pointer";
    case WBMM_STATUS_TOO_LARGE: return "problem larger than the static scratch";
    default: return "unknown status";
    }
}

const char* wbmm_path_string(int path)
{
    switch (path) {
    case WBMM_PATH_NONE: return "none";
    case WBMM_PATH_SIMT: return "simt";
    case WBMM_PATH_TC_TMA: return "tcgen05+tma";
    case WBMM_PATH_TC_GATHER: return "tcgen05+gather";
    case WBMM_PATH_TC_TRANSPOSED: return "tcgen05+tma via NCHW scratch";
    default: return "unknown path";
    }
}

}  // extern "C"
