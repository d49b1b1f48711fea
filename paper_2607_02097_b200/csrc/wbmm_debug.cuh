// Debug scaffolding, compiled only with -DWBMM_WATCHDOG
//     WBMM_NVCC_EXTRA="-DWBMM_WATCHDOG" python -m paper_2607_02097_b200.build --force
// Every mbarrier wait of the pipelined kernels then gives up after 20 ms and records (block, thread, barrier
// address, parity) instead of hanging the GPU.  Included from inside namespace wbmm::ptx (wbmm_ptx.cuh); the records
// of a translation unit are read back with cudaMemcpyFromSymbol(wbmm::ptx::g_watchdog).  Not in the product build,
// not part of the C ABI.
#pragma once

__device__ unsigned long long g_watchdog[64];
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    if (mbar_try_wait(bar, parity)) return;
    long long t0, t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    for (;;) {
        if (mbar_try_wait(bar, parity)) return;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
        if (t1 - t0 > 20000000ll) break;
    }
    unsigned slot = atomicAdd((unsigned*)&g_watchdog[0], 1u);
    if (slot < 60)
        g_watchdog[2 + slot] = ((unsigned long long)blockIdx.x << 48) | ((unsigned long long)threadIdx.x << 36) |
                               ((unsigned long long)(bar & 0xfffff) << 8) | parity;
}
