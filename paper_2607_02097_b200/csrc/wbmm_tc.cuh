// Tensor-core (tcgen05 / TMEM / bulk-copy) WBMM kernels for bf16 / fp16 -- host-side interface.
#pragma once

#include "wbmm_common.cuh"

namespace wbmm {

// How the windows of one channel are cut into MMA tiles of at most 128 windows (= 128 TMEM lanes).
// A tile is NP images x NSY window-rows x all nww windows across; its activation data sits in
// shared memory as a "frame": [image][NSY*w rows][Wp columns] in the padded + shifted coordinate
// system, image stride S bytes.  Window (wl, pl) (wl = wyl*nww + wx inside the frame, pl = image
// inside the tile) is MMA row m = wl*NP + pl.
struct TcTiles {
    int NP, NSY;
    int nstrips;       // strips per image = ceil(nwh / NSY); > 1 only when NP == 1
    int ngb;           // image groups = ceil(B / NP)
    int tiles_per_c;   // ngb * nstrips
    int frame_rows;    // NSY * w
    int S;             // frame image stride in bytes: 16 * odd
    long long ntiles;  // C * tiles_per_c
};

bool tc_tiles(const Geom& g, TcTiles* t);

// True when a tcgen05 forward kernel can serve this problem.
bool tc_forward_supported(const Geom& g, int dtype, const void* x, const void* y);
// Tl != nullptr: the hierarchical operator (global table T, local table Tl; w = 14, bulk kernel only).
// bias [C] (activation dtype, nullable) and ident_bits (16-bit pattern of the identity coefficient, 0 = none;
// w = 14 only) are fused into the pipelined kernel; with either set the call fails where that kernel cannot serve.
cudaError_t tc_forward(const Geom& g, int dtype, const void* x, const void* T, const void* Tl, void* y, bool reverse,
                       cudaStream_t stream, int* launches, int* path, const void* bias = nullptr, uint32_t ident_bits = 0);
bool tc_hier_supported(const Geom& g, int dtype, const void* x, const void* y);
// Cached-M forward through the gather kernel, wherever tc_forward_supported holds:
// M [C][N][N] and bias [C] (nullable) in the activation dtype; transpose applies M_c^T.
cudaError_t tc_forward_matrix(const Geom& g, int dtype, const void* x, const void* M, const void* bias, void* y,
                              bool transpose, cudaStream_t stream, int* launches, int* path);
// True when the pipelined bulk kernel (not the gather fallback) serves this NCHW problem.
bool tc_bulk_supported(const Geom& g, int dtype, const void* x, const void* y);

// FP32 forward / dX on the tensor cores: exact 3-way bf16 splitting, six tcgen05 passes (wbmm_tc_f32.cu).  NCHW, w in {7, 14}.
bool tc_f32_supported(const Geom& g, const void* x, const void* y);
cudaError_t tc_f32_forward(const Geom& g, const void* x, const void* T, void* y, bool reverse, cudaStream_t stream,
                           int* launches);

// FP32 table gradient on the tensor cores: split operands, 3 (w = 14) / 6 (w = 7) passes (wbmm_tc_f32_dt.cu).  Adds into dT.
bool tc_f32_grad_table_supported(const Geom& g, const void* x, const void* dy);
cudaError_t tc_f32_grad_table(const Geom& g, const void* x, const void* dy, float* dT, cudaStream_t stream, int* launches);

// NHWC forward / dX, w = 7, one pass straight from NHWC memory on the pipelined skeleton (wbmm_tc_nhwc7.cu): no shift.
bool tc_nhwc_pipe_supported(const Geom& g, int dtype, const void* x, const void* y);
cudaError_t tc_nhwc_pipe_forward(const Geom& g, int dtype, const void* x, const void* T, void* y, bool reverse,
                                 cudaStream_t stream, int* launches);

// NHWC forward / dX: 8-channel groups gathered with 16-byte cp.async (wbmm_tc_nhwc.cu).
bool tc_nhwc_supported(const Geom& g, int dtype, const void* x, const void* y);
cudaError_t tc_nhwc_forward(const Geom& g, int dtype, const void* x, const void* T, void* y, bool reverse,
                            cudaStream_t stream, int* launches);

bool tc_grad_table_supported(const Geom& g, int dtype, const void* x, const void* dy);
// dTl != nullptr (w = 14 only): also folds S onto the local (w/2) sub-window table of the hierarchical operator.
cudaError_t tc_grad_table(const Geom& g, int dtype, const void* x, const void* dy, float* dT,
                          cudaStream_t stream, int* launches, int* path, float* dTl = nullptr);

// Tensor map (CUtensorMap behind the void*) over an NCHW activation with box = `images` whole frame images of
// one channel (wbmm_tc.cu).
bool image_box_map(const Geom& g, int dtype, const void* base, int images, void* map);
// Plane boxes for planes whose byte size is not a multiple of 16 (wbmm_tc.cu): images per box (0 = not possible) and
// the tensor map over [B][C*H*W] (box = images x (H*W rounded up to 8) elements; inner coordinate c*H*W).
int plane_box_images(const Geom& g, const TcTiles& tl);
bool plane_box_map(const Geom& g, int dtype, const void* base, int images, void* map);

// INT8 forward on the tensor cores (wbmm_tc_i8.cu): kind::i8, exact int32 sums; scale == nullptr: y is int32, else y is
// int8 = sat(rne(fp32(sum) * scale[c])).  w in {7, 14}, any layout / shift / ragged size with at most 128 windows across.
bool tc_i8_supported(const Geom& g);
// fp8: the same kernels with E4M3 operands (kind::f8f6f4, fp32 sums; scale != nullptr: y is E4M3 = rn_satfinite(sum * scale[c])).
cudaError_t tc_i8_forward(const Geom& g, const int8_t* x, const int8_t* T, const float* scale, void* y, cudaStream_t stream,
                          int* launches, int* path, bool fp8 = false);

// wbmm_static_scratch.cu: the NHWC transposition route with its two temporaries in a file-scope device array (no
// allocation).  Returns 0 = served (*err holds the CUDA status), 1 = not a problem of this route, 2 = the activation
// exceeds static_scratch_limit_bytes(); nothing is launched for 1 and 2.
size_t static_scratch_limit_bytes();
int nhwc_forward_static_scratch(const Geom& g, int dtype, const void* x, const void* T, void* y, cudaStream_t stream,
                                int* launches, int* path, cudaError_t* err);

}  // namespace wbmm
