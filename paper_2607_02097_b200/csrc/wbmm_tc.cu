#include "wbmm_tc.cuh"

namespace wbmm {

bool tc_forward_supported(const Geom&, int, const void*, const void*) { return false; }
cudaError_t tc_forward(const Geom&, int, const void*, const void*, void*, bool, cudaStream_t, int*, int*)
{
    return cudaErrorNotSupported;
}
bool tc_grad_table_supported(const Geom&, int, const void*, const void*) { return false; }
cudaError_t tc_grad_table(const Geom&, int, const void*, const void*, float*, cudaStream_t, int*, int*)
{
    return cudaErrorNotSupported;
}
void tc_release() {}

}  // namespace wbmm
