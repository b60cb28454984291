// Primitives shared by the TMA-pipelined stage-1 kernels (integrate_pipe.cu, integrate_stream.cu): mbarriers, bulk
// copies, tensor-map boxes (PTX, sm_90+ / sm_100a), and the ring position helper.
#pragma once
#include <cuda.h>
#include <stdint.h>

#include "ctx.h"

// host: tensor map of the frames for the TMA image path (integrate_pipe.cu)
int ai_make_frame_map(ai_ctx *ctx, const FrameArgs &a, int tile_h, CUtensorMap *map, int box_frames = 1);

// ---- mbarrier / bulk-copy primitives (PTX, sm_90+) ---------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
// non-blocking probe (try_wait may suspend the thread for a system-dependent time before it reports failure)
__device__ __forceinline__ bool mbar_test_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\t"
                 "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
// Bounded wait: a protocol bug traps (the launch fails with an error) instead of hanging the device.  The bound is wall
// time (20 s on %globaltimer, looked at every 4096 polls), not a poll count: a block that is kept off its data for a
// while by another tenant of the GPU, a profiler or a sanitizer must not be mistaken for a lost one.
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    unsigned long long t0 = 0;
    for (uint32_t spin = 1; !mbar_try_wait(bar, parity); ++spin) {
        if ((spin & 0xfffu) == 0) {
            const unsigned long long now = globaltimer_ns();
            if (t0 == 0) t0 = now;
            else if (now - t0 > 20000000000ULL) __trap();
        }
    }
}
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// one box of the (x, y, frame) tensor of frames: 32 pixels x tile_h rows, 128-byte swizzle
__device__ __forceinline__ void tma_box(void *dst_smem, const CUtensorMap *map, int x, int y, int f, uint64_t *bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(dst_smem)), "l"(map), "r"(x), "r"(y), "r"(f), "r"(smem_u32(bar)) : "memory");
}
// waits until *counter >= target (acquire); bounded like mbar_wait
__device__ __forceinline__ void wait_count_at_least(const unsigned long long *counter, unsigned long long target)
{
    unsigned long long t0 = 0;
    for (unsigned spin = 1;; ++spin) {
        unsigned long long seen;
        asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(seen) : "l"(counter) : "memory");
        if (seen >= target) return;
        if ((spin & 0x3ffu) == 0) {
            const unsigned long long now = globaltimer_ns();
            if (t0 == 0) t0 = now;
            else if (now - t0 > 20000000000ULL) __trap();
        }
    }
}
// acquire-release fences (lighter than __threadfence / __threadfence_block, which are sequentially consistent fences)
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ void fence_acq_rel_cta() { asm volatile("fence.acq_rel.cta;" ::: "memory"); }
// orders this thread's shared-memory accesses through the generic proxy before later accesses of the async proxy (TMA)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// position in a ring of buffers: stage and parity of the phase the current use completes
struct Ring {
    int stage = 0;
    uint32_t parity = 0;
    __device__ __forceinline__ void next(int stages)
    {
        if (++stage == stages) { stage = 0; parity ^= 1u; }
    }
};

