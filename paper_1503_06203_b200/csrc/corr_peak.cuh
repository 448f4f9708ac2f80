// corr_peak.cuh -- measurement aid: the int8 tensor-core ceiling of the
// device this library runs on, measured with the SAME instruction the hot path uses
// (tcgen05.mma.cta_group::2.kind::i8, M = 256, N = 128, K = 32, A operand in TMEM, B operand in shared memory)
// in a bare issue loop with no data movement.  Not part of the correlation path; bench.py reports its result
// beside the nominal 4500 TOPS and the measured-bf16-implied figure.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "corr_ptx.cuh"

namespace corr {

constexpr int PK_THREADS = 64;
constexpr int PK_SMEM_BYTES = 1024 + 2 * 4096 + 64;

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PK_THREADS, 1)
corr_peak_kernel(int iters)
{
    extern __shared__ uint8_t pk_raw[];
    const uint32_t base = (ptx::smem_u32(pk_raw) + 1023u) & ~1023u;
    uint8_t *gbase = pk_raw + (base - ptx::smem_u32(pk_raw));
    const uint32_t bar = base + 2 * 4096, slot = bar + 16;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();
    for (int i = threadIdx.x; i < 2 * 4096 / 4; i += PK_THREADS) reinterpret_cast<uint32_t *>(gbase)[i] = 0x01010101u;
    if (threadIdx.x == 0) {
        ptx::mbar_init(bar, 1);
        ptx::fence_mbar_init();
    }
    ptx::fence_proxy_async_smem();
    if (warp == 1) {
        ptx::tmem_alloc<2>(slot, 512);
        ptx::tmem_relinquish<2>();
    }
    ptx::tc_fence_before_sync();
    ptx::cluster_sync();
    ptx::tc_fence_after_sync();
    const uint32_t tmem = *reinterpret_cast<volatile uint32_t *>(gbase + (slot - base));
    if (warp == 0 && rank == 0) {
        constexpr uint32_t idesc = make_idesc_i8(256, 128, true, true, false, true);
        const uint64_t dB0 = make_smem_desc(base, 4096, 512, 4), dB1 = make_smem_desc(base + 4096, 4096, 512, 4);
        if (ptx::elect_one()) {
            for (int i = 0; i < iters; ++i) {
                // the hot path's four products per K-step: three accumulators, A planes at columns 384.. (garbage
                // values: only the issue rate matters)
                ptx::mma_i8_ts<2>(tmem + 0, tmem + 384, dB0, idesc, 1);
                ptx::mma_i8_ts<2>(tmem + 128, tmem + 392, dB1, idesc, 1);
                ptx::mma_i8_ts<2>(tmem + 256, tmem + 400, dB1, idesc, 1);
                ptx::mma_i8_ts<2>(tmem + 128, tmem + 408, dB0, idesc, 1);
            }
            ptx::mma_commit_mcast2(bar, 0x3);
        }
        __syncwarp();
    }
    if (lane == 0 && warp == 0) ptx::mbar_wait_cluster(bar, 0);   // both CTAs: every MMA has completed
    __syncwarp();
    ptx::tc_fence_before_sync();
    ptx::cluster_sync();
    if (warp == 1) ptx::tmem_dealloc<2>(tmem, 512);
}

}  // namespace corr
