// Batched 2-D transposition of 16-bit elements: in[b][R][Cc] -> out[b][Cc][R].
//
// Used by the NHWC entry path (wbmm_api.cu): NHWC = [B][H*W][C], NCHW = [B][C][H*W].  Reading NHWC at
// anything finer than whole pixels (all C channels, 192+ bytes) wastes the memory system -- a tile that
// feeds the per-channel tensor-core GEMM can hold only 8 channels of its pixels, i.e. 16-byte pieces
// (measured: LSU gather 38-44 us, 16-byte-box TMA 11-28 us per 200 KB tile).  Two
// full-bandwidth transposition passes around the NCHW kernels are faster by 2.5x (forward) to 20x (dT).
//
// 64 x 64 tiles: 16-byte global loads along Cc, eight conflict-free 2-byte shared stores per load into
// the transposed tile (row pitch 66 elements = 33 words), four 32-bit shared loads, 16-byte global
// stores along R.  R and Cc multiples of 8, 16-byte aligned pointers.
#include "wbmm_common.cuh"

namespace wbmm {

namespace {

constexpr int kTile = 64, kPitch = kTile + 2;

__global__ void __launch_bounds__(256) transpose16_kernel(const uint16_t* __restrict__ in, uint16_t* __restrict__ out, int R, int Cc)
{
    __shared__ __align__(16) uint16_t tileT[kTile * kPitch];      // [c][r]
    const long long base = (long long)blockIdx.z * R * Cc;
    const int r0 = blockIdx.y * kTile, c0 = blockIdx.x * kTile;
    const int t = threadIdx.x;
#pragma unroll
    for (int pass = 0; pass < 2; ++pass) {
        const int r = pass * 32 + (t >> 3), ch = (t & 7) * 8;
        if (r0 + r < R && c0 + ch < Cc) {
            const uint4 v = __ldg(reinterpret_cast<const uint4*>(in + base + (long long)(r0 + r) * Cc + c0 + ch));
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int j = 0; j < 8; ++j) tileT[(ch + j) * kPitch + r] = (uint16_t)(w[j >> 1] >> ((j & 1) * 16));
        }
    }
    __syncthreads();
#pragma unroll
    for (int pass = 0; pass < 2; ++pass) {
        const int c = pass * 32 + (t >> 3), r8 = (t & 7) * 8;
        if (c0 + c < Cc && r0 + r8 < R) {
            const uint32_t* src = reinterpret_cast<const uint32_t*>(tileT + c * kPitch + r8);
            const uint4 v = make_uint4(src[0], src[1], src[2], src[3]);
            *reinterpret_cast<uint4*>(out + base + (long long)(c0 + c) * R + r0 + r8) = v;
        }
    }
}

// The same for 32-bit elements (fp32 activations): 32 x 32 tiles, 16-byte global accesses both ways.
__global__ void __launch_bounds__(256) transpose32_kernel(const uint32_t* __restrict__ in, uint32_t* __restrict__ out, int R, int Cc)
{
    __shared__ uint32_t tileT[32 * 33];      // [c][r]
    const long long base = (long long)blockIdx.z * R * Cc;
    const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
    const int t = threadIdx.x;
    {
        const int r = t >> 3, ch = (t & 7) * 4;
        if (r0 + r < R && c0 + ch < Cc) {
            const uint4 v = __ldg(reinterpret_cast<const uint4*>(in + base + (long long)(r0 + r) * Cc + c0 + ch));
            tileT[(ch + 0) * 33 + r] = v.x;
            tileT[(ch + 1) * 33 + r] = v.y;
            tileT[(ch + 2) * 33 + r] = v.z;
            tileT[(ch + 3) * 33 + r] = v.w;
        }
    }
    __syncthreads();
    {
        const int c = t >> 3, r4 = (t & 7) * 4;
        if (c0 + c < Cc && r0 + r4 < R) {
            const uint32_t* src = tileT + c * 33 + r4;
            *reinterpret_cast<uint4*>(out + base + (long long)(c0 + c) * R + r0 + r4) = make_uint4(src[0], src[1], src[2], src[3]);
        }
    }
}

// The same for 8-bit elements (INT8 activations): 64 x 64 tiles, 16-byte global accesses both ways.
__global__ void __launch_bounds__(256) transpose8_kernel(const uint8_t* __restrict__ in, uint8_t* __restrict__ out, int R, int Cc)
{
    constexpr int kP = 68;                       // tile row pitch in bytes (17 words)
    __shared__ __align__(16) uint8_t tileT[64 * kP];   // [c][r]
    const long long base = (long long)blockIdx.z * R * Cc;
    const int r0 = blockIdx.y * 64, c0 = blockIdx.x * 64;
    const int t = threadIdx.x;
    {
        const int r = t >> 2, ch = (t & 3) * 16;
        if (r0 + r < R && c0 + ch < Cc) {
            const uint4 v = __ldg(reinterpret_cast<const uint4*>(in + base + (long long)(r0 + r) * Cc + c0 + ch));
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 16; ++k) tileT[(ch + k) * kP + r] = (uint8_t)(w[k >> 2] >> ((k & 3) * 8));
        }
    }
    __syncthreads();
    {
        const int c = t >> 2, r16 = (t & 3) * 16;
        if (c0 + c < Cc && r0 + r16 < R) {
            const uint32_t* src = reinterpret_cast<const uint32_t*>(tileT + c * kP + r16);
            *reinterpret_cast<uint4*>(out + base + (long long)(c0 + c) * R + r0 + r16) = make_uint4(src[0], src[1], src[2], src[3]);
        }
    }
}

}  // namespace

bool transpose8_supported(long long R, long long Cc, const void* in, const void* out)
{
    return R % 16 == 0 && Cc % 16 == 0 && R <= 0x7fffffff && Cc <= 0x7fffffff &&
           reinterpret_cast<uintptr_t>(in) % 16 == 0 && reinterpret_cast<uintptr_t>(out) % 16 == 0;
}

cudaError_t transpose8(const void* in, void* out, int batch, int R, int Cc, cudaStream_t stream, int* launches)
{
    if (batch == 0 || R == 0 || Cc == 0) return cudaSuccess;
    for (int b0 = 0; b0 < batch; b0 += 65535) {          // gridDim.z limit
        const int nb = batch - b0 < 65535 ? batch - b0 : 65535;
        dim3 grid((Cc + 63) / 64, (R + 63) / 64, nb);
        const long long off = (long long)b0 * R * Cc;
        transpose8_kernel<<<grid, 256, 0, stream>>>((const uint8_t*)in + off, (uint8_t*)out + off, R, Cc);
        *launches += 1;
    }
    return cudaGetLastError();
}

bool transpose32_supported(long long R, long long Cc, const void* in, const void* out)
{
    return R % 4 == 0 && Cc % 4 == 0 && R <= 0x7fffffff && Cc <= 0x7fffffff &&
           reinterpret_cast<uintptr_t>(in) % 16 == 0 && reinterpret_cast<uintptr_t>(out) % 16 == 0;
}

cudaError_t transpose32(const void* in, void* out, int batch, int R, int Cc, cudaStream_t stream, int* launches)
{
    if (batch == 0 || R == 0 || Cc == 0) return cudaSuccess;
    for (int b0 = 0; b0 < batch; b0 += 65535) {          // gridDim.z limit
        const int nb = batch - b0 < 65535 ? batch - b0 : 65535;
        dim3 grid((Cc + 31) / 32, (R + 31) / 32, nb);
        const long long off = (long long)b0 * R * Cc;
        transpose32_kernel<<<grid, 256, 0, stream>>>((const uint32_t*)in + off, (uint32_t*)out + off, R, Cc);
        *launches += 1;
    }
    return cudaGetLastError();
}

bool transpose16_supported(long long R, long long Cc, const void* in, const void* out)
{
    return R % 8 == 0 && Cc % 8 == 0 && R <= 0x7fffffff && Cc <= 0x7fffffff &&
           reinterpret_cast<uintptr_t>(in) % 16 == 0 && reinterpret_cast<uintptr_t>(out) % 16 == 0;
}

cudaError_t transpose16(const void* in, void* out, int batch, int R, int Cc, cudaStream_t stream, int* launches)
{
    if (batch == 0 || R == 0 || Cc == 0) return cudaSuccess;
    for (int b0 = 0; b0 < batch; b0 += 65535) {          // gridDim.z limit
        const int nb = batch - b0 < 65535 ? batch - b0 : 65535;
        dim3 grid((Cc + kTile - 1) / kTile, (R + kTile - 1) / kTile, nb);
        const long long off = (long long)b0 * R * Cc;
        transpose16_kernel<<<grid, 256, 0, stream>>>((const uint16_t*)in + off, (uint16_t*)out + off, R, Cc);
        *launches += 1;
    }
    return cudaGetLastError();
}

}  // namespace wbmm
