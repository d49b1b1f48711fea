/*
 * wbmm.h -- C ABI of libwbmm.so: the WBMM operator (Windowed Batch Matrix Multiplication,
 * arxiv/paper_2607_02097) as hand-written CUDA kernels for NVIDIA B200 (sm_100a).
 *
 * Citations are to the paper text and to DESIGN.md ("Readings").
 *
 * The operator (Algorithm 1, Eq. 4-8; orientation per DESIGN.md reading A1):
 *   the activation x[B,C,H,W] is zero-padded (bottom/right) to multiples of w, cut into
 *   non-overlapping w x w windows of N = w*w positions (row-major inside a window), and every
 *   window of channel c is multiplied by that channel's N x N matrix
 *       W_c[i,j] = T[c, rel(i,j)],   rel(i,j) = (r_i - r_j + w-1)*(2w-1) + (c_i - c_j + w-1)
 *   (Eq. 6-8), i = output position, j = input position:  y_win = W_c * x_win.  W_c is never
 *   written to HBM.  The padding is cropped from the output (Eq. 4-5).
 *   Optional cyclic shift (reading A6):  x^[h,v] = x~[(h+s_h) mod H', (v+s_w) mod W']
 *   on the padded extent before partitioning, inverse roll on the output.
 *   Backward (autograd of Alg. 1):  dX_win = W_c^T * dY_win,
 *       dT[c,k] = sum over images, windows and pairs (i,j) with rel(i,j)=k of dY_win[i]*X_win[j].
 *
 * Conventions for every entry point
 *   - Pointers named x, T, y, dy, dx, dT, Wout are DEVICE pointers unless the function name ends
 *     in _host.  Tensors are dense and contiguous.  The caller owns all buffers and the stream.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *     Calls are asynchronous on that stream; the library never synchronises (the _host variants
 *     do: they return after the result is in host memory).
 *   - Return value: a wbmm_status_t.  Nothing throws or aborts across the ABI.  On a non-zero
 *     status no output buffer has been written.
 *   - NHWC activations (bf16/fp16): w = 7 without shift and C a multiple of 8 is served straight from NHWC memory
 *     by one pipelined kernel (forward and dX; no temporaries).  Other NHWC problems with C and H*W multiples of 8
 *     are served by transposing to NCHW and back around the NCHW kernels; the two temporaries come from a memory
 *     pool the library owns (cudaMallocFromPoolAsync / cudaFreeAsync on the caller's stream: stream-ordered,
 *     capturable in CUDA graphs, released by wbmm_release()) and never outlive the call's work.
 *     WBMM_FLAG_NO_SCRATCH forbids the temporaries; the call is then served by the slower scratch-free kernels.
 *     Every other path allocates nothing.
 *   - float32 activations with w in {7, 14} run on the tensor cores too, each operand split exactly into three
 *     bf16 parts (error <= 1e-6 relative to sum |W||x|); other w use the FFMA kernels.  float32 NHWC
 *     (C and H*W multiples of 4) takes the transposition route with temporaries from the library's pool, as above.
 *   - There is no CPU fallback.  Without a CUDA device of compute capability 10.x every compute
 *     entry point returns WBMM_STATUS_NO_DEVICE.
 */
#ifndef WBMM_H_
#define WBMM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define WBMM_VERSION 100 /* major*10000 + minor*100 + patch */

#if defined(__GNUC__)
#define WBMM_API __attribute__((visibility("default")))
#else
#define WBMM_API
#endif

typedef enum {
    WBMM_STATUS_OK = 0,
    WBMM_STATUS_INVALID_ARGUMENT = 1, /* null pointer, non-positive size, shift not in [0,w), bad enum, y aliases x */
    WBMM_STATUS_UNSUPPORTED = 2,      /* window too large for shared memory, or dtype/path combination not built */
    WBMM_STATUS_NO_DEVICE = 3,        /* no CUDA device, or the device is not sm_100 */
    WBMM_STATUS_CUDA_ERROR = 4,       /* a CUDA runtime/driver call failed; see wbmm_last_error_string() */
    WBMM_STATUS_MISALIGNED = 5,       /* a pointer is not aligned to its element size */
    WBMM_STATUS_TOO_LARGE = 6         /* wbmm_forward_static_scratch: the activation exceeds the static scratch */
} wbmm_status_t;

typedef enum { WBMM_DTYPE_F32 = 0, WBMM_DTYPE_BF16 = 1, WBMM_DTYPE_F16 = 2 } wbmm_dtype_t;
typedef enum { WBMM_LAYOUT_NCHW = 0, WBMM_LAYOUT_NHWC = 1 } wbmm_layout_t;

/* Which kernel family served the last call on this host thread (wbmm_last_path()). */
typedef enum {
    WBMM_PATH_NONE = 0,
    WBMM_PATH_SIMT = 1,      /* general fp32-FFMA kernels: any w, dtype, layout, shift, ragged size */
    WBMM_PATH_TC_TMA = 2,    /* pipelined tcgen05/TMEM tensor-core kernels fed by TMA (bf16/fp16 NCHW, NHWC w = 7,
                                and float32 through the 3-way bf16 split) */
    WBMM_PATH_TC_GATHER = 3, /* block-synchronous tcgen05/TMEM kernels fed by a predicated gather loader (bf16/fp16):
                                wbmm_forward_matrix, and shapes the FFMA kernels cannot take */
    WBMM_PATH_TC_TRANSPOSED = 4 /* NHWC: transposition passes through stream-ordered scratch around the TC_TMA kernels */
} wbmm_path_t;

enum {
    WBMM_FLAG_ACCUMULATE_DT = 1u, /* wbmm_backward: add into dT instead of overwriting it */
    WBMM_FLAG_FORCE_SIMT = 2u,    /* never take a tensor-core path (testing / cross-checks) */
    WBMM_FLAG_NO_FORK = 8u,       /* wbmm_backward with dx AND dT: run the two kernels one after the other on the caller's
                                     stream (default: the table gradient runs on an internal stream forked from and joined
                                     back into the caller's stream -- same ordering guarantees, the two overlap) */
    WBMM_FLAG_NO_SCRATCH = 4u     /* NHWC: never allocate transposition scratch from the library's pool; problems the
                                     one-pass NHWC kernel (w = 7, no shift) does not take then run on the
                                     scratch-free gather / FFMA kernels, which are several times slower */
};

/* Problem descriptor (plain data, passed by pointer, read during the call only). */
typedef struct wbmm_desc {
    int32_t B, C, H, W;       /* logical activation sizes; H, W need not be multiples of w */
    int32_t w;                /* square window side, w >= 1; N = w*w; the table has (2w-1)^2 bins per channel */
    int32_t shift_h, shift_w; /* cyclic shift in [0, w); 0 = none */
    int32_t dtype;            /* wbmm_dtype_t of x, y, dy, dx AND of T.  dT is always float32. */
    int32_t layout;           /* wbmm_layout_t of x, y, dy, dx.  T and dT are [C][(2w-1)^2] row-major. */
    uint32_t flags;           /* WBMM_FLAG_* */
} wbmm_desc_t;

/*
 * Forward, Algorithm 1:  y = WBMM(x; T, w).
 *   x  [in]  B*C*H*W elements of desc->dtype in desc->layout.            Read-only.
 *   T  [in]  C*(2w-1)^2 elements of desc->dtype.                         Read-only.
 *   y  [out] same shape/dtype/layout as x; every element is overwritten, nothing outside it.
 *            Accumulation is fp32; the result is rounded to desc->dtype (RNE).  y must not alias x.
 * bf16/fp16 tensor-core paths multiply some padding lanes by exact zero weights: inputs are
 * assumed finite (a non-finite x may turn neighbouring outputs of the same row strip into NaN).
 */
WBMM_API int wbmm_forward(const wbmm_desc_t *desc, const void *x, const void *T, void *y, void *cuda_stream);

/*
 * wbmm_forward for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): the NHWC transposition route of wbmm_forward (transpose -> NCHW tensor-core kernel -> transpose;
 * same kernels, same results) with its two temporaries in ONE file-scope device array instead of the library's memory
 * pool.  The call allocates and frees nothing (no cudaMalloc, cudaFree, cudaMallocAsync, no allocating library
 * routine); x, T, y are the caller's, as in wbmm_forward.
 *   Serves   NHWC, bf16/fp16, w in {7, 14}, C and H*W multiples of 8 (what the transposition route serves), any shift /
 *            ragged size; anything else: WBMM_STATUS_UNSUPPORTED, nothing launched.  desc->flags is ignored.
 *   Limit    B*C*H*W*2 bytes <= 16 MiB (8 Mi elements; e.g. B = 16, C = 96, 56 x 56).  Beyond it:
 *            WBMM_STATUS_TOO_LARGE with the sizes in wbmm_last_error_string(), nothing launched.
 *   Cost     the array is 32 MiB (two temporaries); every GPU that loads libwbmm.so holds it until the process exits.
 *   Sharing  all calls on a device share the array, which keeps the last call's contents.  Nothing needs clearing:
 *            each call overwrites every byte it later reads.  Calls that OVERLAP on the GPU (different streams) race
 *            on it and give wrong results; calls on one stream are ordered and safe back to back.
 */
WBMM_API int wbmm_forward_static_scratch(const wbmm_desc_t *desc, const void *x, const void *T, void *y, void *cuda_stream);

/*
 * Backward of wbmm_forward:
 *   dx [out, nullable] dX = W_c^T * dY per window, shape/dtype/layout of x, fully overwritten.
 *   dT [out, nullable] float32 [C][(2w-1)^2]; overwritten (zeroed on the stream first) unless
 *                      WBMM_FLAG_ACCUMULATE_DT.  Summation order over windows is not fixed
 *                      (atomics): results are reproducible to rounding, not bitwise.
 *   x, T, dy [in] as in wbmm_forward; dy is treated as zero outside H x W (A11).
 *   x may be NULL when dT is NULL; T may be NULL when dx is NULL.
 * When BOTH dx and dT are asked for, the table gradient runs on an internal stream (one per host thread and device)
 * that waits for everything queued on cuda_stream before the call, and cuda_stream waits for it before anything
 * queued after the call: the ordering seen by the caller is that of a single stream, the call stays asynchronous and
 * capturable, and the two independent kernels overlap (7 % on the config-5 backward).  WBMM_FLAG_NO_FORK keeps both on
 * cuda_stream.
 */
WBMM_API int wbmm_backward(const wbmm_desc_t *desc, const void *x, const void *T, const void *dy,
                  void *dx, float *dT, void *cuda_stream);

/*
 * Rectangular windows w_h x w_w (section 3.1 states the method for a "window size w_h x w_w": d = w_h*w_w
 * positions, table [C][(2w_h-1)(2w_w-1)] row-major; Eq. 4-5 pad H to a multiple of w_h and W to a multiple of w_w;
 * Eq. 6-7  I[i,j] = (dh + w_h - 1)(2w_w - 1) + (dw + w_w - 1)).  w_h = 1 gives the 1-D windows of PAPER.md:909.
 *   desc->w is w_h, w_w is passed beside it; desc->shift_h in [0, w_h), desc->shift_w in [0, w_w).
 *   x, T, y / dy, dx, dT: as wbmm_forward / wbmm_backward with the rectangular table shape.
 * w_w == desc->w is the square operator and is served by wbmm_forward / wbmm_backward (tensor cores).  Other shapes run on
 * FFMA kernels (any dtype / layout / shift / ragged size; wbmm_last_path() = WBMM_PATH_SIMT); w_h*w_w <= 1024 and
 * (2w_h-1)(2w_w-1) <= 4096, else WBMM_STATUS_UNSUPPORTED.  dT: cleared first unless WBMM_FLAG_ACCUMULATE_DT; atomics.
 */
WBMM_API int wbmm_forward_rect(const wbmm_desc_t *desc, int32_t w_w, const void *x, const void *T, void *y, void *cuda_stream);
WBMM_API int wbmm_backward_rect(const wbmm_desc_t *desc, int32_t w_w, const void *x, const void *T, const void *dy,
                       void *dx, float *dT, void *cuda_stream);

/*
 * Hierarchical window reparameterisation, fused (section 3.6, Eq. 9; PAPER.md:862-887
 * Algorithm 3; identical in value to the training form, Algorithm 2):
 *     y_win = (M_g + diag_blocks(M_l) + 2 I) * x_win
 * per global w x w window (desc->w, even), M_g[i,j] = Tg[c, rel_w(i,j)], M_l[i,j] = Tl[c, rel_{w/2}(i,j)]
 * placed on the four diagonal blocks of the 2 x 2 local sub-windows, 2 I = the two identity shortcuts.
 * The fused matrix is never formed: both tables are expanded into block-Toeplitz libraries in shared
 * memory (27 KB instead of the C x 196 x 196 tensor of Algorithm 3).
 *   Tg [in] C*(2w-1)^2, Tl [in] C*(w-1)^2 elements of desc->dtype.  x, y, padding, shift as wbmm_forward.
 *   transpose != 0 applies the transposed fused matrix: dX of the operator for dy in `x`.
 * Gradients: wbmm_hier_backward.
 * Served by the pipelined tensor-core kernel where it applies: w = 14, bf16/fp16, NCHW with 16-byte aligned planes
 * (H*W even ... see wbmm_last_path), or NHWC through the transposition scratch (C and H*W multiples of 8, no
 * WBMM_FLAG_NO_SCRATCH).  Everything else (float32 -- the paper's precision --, other even w, WBMM_FLAG_FORCE_SIMT)
 * runs on FFMA kernels that apply the same fused operator in one pass (wbmm_last_path() = WBMM_PATH_SIMT);
 * w*w > 1024: WBMM_STATUS_UNSUPPORTED.
 */
WBMM_API int wbmm_hier_forward(const wbmm_desc_t *desc, const void *x, const void *Tg, const void *Tl, void *y,
                      int transpose, void *cuda_stream);

/*
 * Backward of wbmm_hier_forward (the gradient of Algorithm 2, term by term; the identity
 * shortcuts carry no parameter):
 *   dx  [out, nullable] the transposed fused operator applied to dy (= wbmm_hier_forward(..., transpose = 1)).
 *   dTg [out, nullable] float32 [C][(2w-1)^2]: sum over windows and pairs (i,j) with rel_w(i,j) = k of dy[i] x[j].
 *   dTl [out, nullable] float32 [C][(w-1)^2]: the same sum restricted to pairs inside one of the 2 x 2 local
 *                       sub-windows, binned by rel_{w/2}.  dTg and dTl are given together or not at all; both
 *                       come from ONE pass over (x, dy): S = dY^T X is accumulated once in tensor memory and
 *                       folded onto both sets of bins.  Overwritten unless WBMM_FLAG_ACCUMULATE_DT.
 *   x may be NULL when the table gradients are not requested; Tg, Tl may be NULL when dx is NULL.
 * Padding, shift and the zero extension of dy as in wbmm_backward.  Tensor-core kernels where wbmm_hier_forward
 * uses them, FFMA kernels otherwise (the local-table gradient is then the table gradient of the (w/2)-window
 * operator on the extent padded for the global window).
 */
WBMM_API int wbmm_hier_backward(const wbmm_desc_t *desc, const void *x, const void *Tg, const void *Tl, const void *dy,
                       void *dx, float *dTg, float *dTl, void *cuda_stream);

/*
 * Eq. 6-8 on their own (test/debug and the WBMM-C "cached M" mode):
 *   Wout [out] [C][N][N] elements of desc->dtype, Wout[c,i,j] = T[c, rel(i,j)] copied bit-exactly.
 * Only C, w and dtype of the descriptor are used.
 */
WBMM_API int wbmm_materialize_weight(const wbmm_desc_t *desc, const void *T, void *Wout, void *cuda_stream);

/*
 * Forward with the neighbouring elementwise steps fused (Eq. 1's beta_c,
 * PAPER.md:848-852 identity shortcut):
 *     y_win = W_c * x_win + identity * x_win + bias_c          (W_c from the table, Eq. 6-8)
 *   bias     [in, nullable] [C] elements of desc->dtype (finite).  Costs nothing: it rides the contraction as one
 *            more K index -- a column of ones in the padding of the A operand against a weight row holding bias_c --
 *            so it is added in the fp32 accumulator, before the single rounding.
 *   identity coefficient of the shortcut, rounded to desc->dtype (1.0 and 2.0 are exact); 0 = none.  Applied by the
 *            16 x 16 block identity * I of the w = 14 weight library (14 extra N = 16 MMAs per tile), never summed
 *            into the 16-bit table values.  w = 14 only.
 *   transpose != 0 applies W_c^T + identity * I (the dX of the fused operator for dy in `x`; pass bias = NULL).
 * Served by the pipelined tensor-core kernel where it applies (bf16/fp16, w in {7, 14} -- identity: w = 14 --, NCHW
 * planes the copy schemes move, or NHWC through the transposition scratch); everything else (float32, identity at
 * other w, other window sizes) by an FFMA kernel that applies the same fused operator in one pass
 * (wbmm_last_path() = WBMM_PATH_SIMT); w*w > 1024: WBMM_STATUS_UNSUPPORTED.
 */
WBMM_API int wbmm_forward_fused(const wbmm_desc_t *desc, const void *x, const void *T, const void *bias, float identity,
                       void *y, int transpose, void *cuda_stream);

/*
 * Cached-M inference mode, "WBMM-C": Algorithm 1 with GIVEN per-channel matrices,
 *     y_win = M_c * x_win (+ bias_c),
 *   M    [in] [C][N][N] elements of desc->dtype, row i = output position, column j = input position (the
 *             layout wbmm_materialize_weight writes); any matrix, not only Eq. 8's.
 *   bias [in, nullable] [C] elements of desc->dtype (Eq. 1's beta_c; the BatchNorm shifts of section 3.7), added
 *             to the fp32 accumulator before the single rounding.
 *   transpose != 0 applies M_c^T (the dX of the cached operator; the bias is still added if given).
 * x, y, padding, shift, layout as wbmm_forward.  With M = wbmm_materialize_weight(T) and no bias the result is
 * wbmm_forward's ("identical outputs") up to the fp32 summation order of the kernel that serves it
 * (at most one 16-bit ulp).  Served by the pipelined tensor-core kernels where wbmm_forward is (NCHW; the matrix takes
 * the place of the weights built from the table), else by the gather tensor-core kernel (w in {7, 14}, bf16/fp16, any
 * layout / shift / ragged size), else (float32, other w with w*w <= 1024) by an FFMA kernel that reads M_c from
 * global memory; otherwise WBMM_STATUS_UNSUPPORTED.  On this design the cached mode is NOT the fast
 * one: the table path rebuilds its weights in shared memory from 1.4 KB per channel while M costs 75 KB per channel
 * of HBM traffic and ~9 us per channel change at w = 14 -- it exists for matrices that are not table-generated.
 */
WBMM_API int wbmm_forward_matrix(const wbmm_desc_t *desc, const void *x, const void *M, const void *bias, void *y,
                        int transpose, void *cuda_stream);

/*
 * 3-D windows w_d x w_h x w_w on volumes (the extension PAPER.md:909 names; reading A23:
 * Eq. 4-7 with one more axis).  desc gives B, C, H, W, w = w_h, shift_h, shift_w, dtype, layout and flags as for
 * wbmm_forward_rect; D (depth), w_d, w_w and shift_d in [0, w_d) are arguments.
 *   layout   WBMM_LAYOUT_NCHW: x, y, dy, dx are [B][C][D][H][W];  WBMM_LAYOUT_NHWC: [B][D][H][W][C].
 *   T, dT    [C][(2w_d-1)(2w_h-1)(2w_w-1)], index ((dz + w_d - 1)(2w_h - 1) + (dh + w_h - 1))(2w_w - 1) + (dw + w_w - 1) with
 *            (dz, dh, dw) = output position - input position inside the window; T in desc->dtype, dT float32.
 *   D, H, W are zero-padded at the far end to multiples of the window; the cyclic shift acts on the padded volume.
 * FFMA kernels with float32 accumulation (wbmm_last_path() = WBMM_PATH_SIMT), any dtype / layout / shift / ragged size;
 * w_d*w_h*w_w <= 1024 and (2w_d-1)(2w_h-1)(2w_w-1) <= 4096, else WBMM_STATUS_UNSUPPORTED.  Pointer rules, nullable dx / dT,
 * WBMM_FLAG_ACCUMULATE_DT as in wbmm_backward_rect.
 */
WBMM_API int wbmm_forward_win3d(const wbmm_desc_t *desc, int32_t D, int32_t w_d, int32_t w_w, int32_t shift_d, const void *x,
                       const void *T, void *y, void *cuda_stream);
WBMM_API int wbmm_backward_win3d(const wbmm_desc_t *desc, int32_t D, int32_t w_d, int32_t w_w, int32_t shift_d, const void *x,
                        const void *T, const void *dy, void *dx, float *dT, void *cuda_stream);

/*
 * INT8 forward (PAPER.md:749 reports INT8 deployments of the operator; reading A21):
 * Algorithm 1 on signed 8-bit activations and tables with exact 32-bit integer sums (|sum| <= w*w*128*128 < 2^31),
 * on the tensor cores (tcgen05.mma kind::i8, accumulator in tensor memory; wbmm_last_path() = WBMM_PATH_TC_TMA for
 * aligned NCHW maps without shift -- the bulk-copy kernel --, WBMM_PATH_TC_GATHER otherwise).
 *   x     [in]  B*C*H*W int8 in desc->layout.  T [in] C*(2w-1)^2 int8.  Device pointers, read-only.
 *   scale [in, nullable] float32 [C], device, finite.
 *   y     [out] scale == NULL: int32, the raw sums (4-byte aligned), same shape / layout as x;
 *               scale != NULL: int8, q = sat_s8(rne(fp32(sum) * scale[c])) -- the sum converted to binary32 (RNE), ONE
 *               binary32 product, rounded to the nearest integer with ties to even, clamped to [-128, 127].
 *               Every element is overwritten, nothing outside it; y must not alias x.
 * desc->dtype is not read (the element types are fixed by this entry point); of desc->flags only WBMM_FLAG_NO_SCRATCH.
 * NHWC with C and H*W multiples of 16 and 16-byte aligned pointers goes through two stream-ordered temporaries from the
 * library's pool (transpose -> NCHW kernel -> transpose; wbmm_last_path() = WBMM_PATH_TC_TRANSPOSED) unless
 * WBMM_FLAG_NO_SCRATCH is set.  Serves w in {7, 14},
 * any shift / ragged size / layout, with at most 128 windows across (W' / w <= 128); anything else:
 * WBMM_STATUS_UNSUPPORTED, nothing launched.  Results are bit-exact against the integer definition.
 */
WBMM_API int wbmm_forward_int8(const wbmm_desc_t *desc, const int8_t *x, const int8_t *T, const float *scale, void *y,
                      void *cuda_stream);

/*
 * FP8 forward (reading A22): Algorithm 1 on E4M3 activations and tables ("fn" flavour:
 * bias 7, no infinities, 0x7f / 0xff NaN), products accumulated in float32 by the tensor cores (tcgen05.mma
 * kind::f8f6f4); the kernels, routes, limits and wbmm_last_path() values of wbmm_forward_int8.
 *   x, T  [in]  E4M3 bytes, shapes as in wbmm_forward_int8.  Inputs are assumed finite (no NaN codes).
 *   scale [in, nullable] float32 [C], device, finite.
 *   y     [out] scale == NULL: float32, the sums (4-byte aligned);
 *               scale != NULL: E4M3 bytes of sum * scale[c] (one binary32 product, round-to-nearest-even, saturating
 *               at +-448).  Every element is overwritten; y must not alias x.
 * The float32 sums agree with the exact real sums to float32 accumulation accuracy (the tensor core's summation order
 * is not specified); a stored code is the nearest E4M3 number to sum * scale except within that error of a midpoint.
 */
WBMM_API int wbmm_forward_fp8(const wbmm_desc_t *desc, const void *x, const void *T, const float *scale, void *y,
                     void *cuda_stream);

/*
 * Multi-kernel fusion for one-window maps (section 3.7): a zero-padded ksize x ksize depthwise
 * conv (Eq. 1, cross-correlation) on an H = W = w map is the WBMM operator with the conv kernel written around
 * the centre of the table, so  Y = WBMM(X) + BN1(DW5(X)) + BN2(DW3(X))  folds into ONE table plus a bias:
 *     Tout[c, (w-1-i)(2w-1) + (w-1-j)] = T[c, same] + scale[c] * K[c, i+k, j+k],   -k <= i, j <= k = ksize/2,
 * every other entry copied.  T, Tout [C][(2w-1)^2] and K [C][ksize][ksize] of desc->dtype (Tout may be T);
 * scale [in, nullable = 1] float32 [C] (BatchNorm's gamma / sigma; its shift goes to wbmm_forward_matrix's bias,
 * or is added by the caller).  fp32 arithmetic, one rounding.  Only C, w and dtype of the descriptor are used;
 * ksize odd, ksize/2 <= w-1.  The fold is exact for maps of one window; on larger maps the conv would cross
 * window borders and the identity does not hold.
 */
WBMM_API int wbmm_fold_dwconv(const wbmm_desc_t *desc, const void *T, const void *K, int ksize, const float *scale,
                     void *Tout, void *cuda_stream);

/*
 * End-to-end variants with HOST buffers (pageable or pinned).  Each call copies its inputs to
 * device scratch owned by the library (grown on demand, reused between calls, freed by
 * wbmm_release()), runs the same kernels as the device entry points on an internal stream,
 * copies the results back and returns when they are in host memory.
 */
WBMM_API int wbmm_forward_host(const wbmm_desc_t *desc, const void *x_host, const void *T_host, void *y_host);
WBMM_API int wbmm_backward_host(const wbmm_desc_t *desc, const void *x_host, const void *T_host,
                       const void *dy_host, void *dx_host /*nullable*/, float *dT_host /*nullable*/);

/* Frees the scratch and cached state held by the library (host-variant buffers, tensor maps). */
WBMM_API void wbmm_release(void);

/* wbmm_path_t of the most recent compute call made by the calling host thread. */
WBMM_API int wbmm_last_path(void);
/* Number of kernels this library has launched since it was loaded (all threads). */
WBMM_API uint64_t wbmm_launch_count(void);
/* Static strings; never NULL. */
WBMM_API const char *wbmm_status_string(int status);
WBMM_API const char *wbmm_path_string(int path);
/* Text of the last CUDA error seen by the calling host thread ("" if none). */
WBMM_API const char *wbmm_last_error_string(void);
WBMM_API int wbmm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WBMM_H_ */
