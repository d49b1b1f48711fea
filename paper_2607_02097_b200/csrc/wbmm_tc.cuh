// Tensor-core (tcgen05 / TMEM / TMA) WBMM kernels for bf16 / fp16 -- host-side interface.
#pragma once

#include "wbmm_common.cuh"

namespace wbmm {

// True when the tcgen05 forward kernel can serve this problem (dtype, window, layout, strides
// legal for the TMA tensor map, pointer alignment).
bool tc_forward_supported(const Geom& g, int dtype, const void* x, const void* y);
cudaError_t tc_forward(const Geom& g, int dtype, const void* x, const void* T, void* y, bool reverse,
                       cudaStream_t stream, int* launches, int* path);

bool tc_grad_table_supported(const Geom& g, int dtype, const void* x, const void* dy);
cudaError_t tc_grad_table(const Geom& g, int dtype, const void* x, const void* dy, float* dT,
                          cudaStream_t stream, int* launches, int* path);

void tc_release();

}  // namespace wbmm
