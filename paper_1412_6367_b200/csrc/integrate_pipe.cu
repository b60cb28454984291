// TILED stage 1 as a persistent, warp-specialised, bulk-copy pipelined kernel -- the B200 design
// of the CSR SpMV of PAPER.md:174-188.
//
// One block per SM stays resident and walks a static list of work items (tile, range of frames), longest tiles first.
// Three roles run concurrently and hand buffers to each other through shared-memory mbarriers:
//
//   producer  (1 elected thread)   issues cp.async.bulk (TMA) copies of the tile's slice of the matrix -- coefficients,
//                                  16-bit pixel positions, segment records, three contiguous ranges -- into a ring of
//                                  shared-memory stages: whole slices in flight per SM with no registers held.
//   stagers   (one warp per image  each warp owns one tile buffer and stages every img_stages-th image tile on its own:
//              stage)              128-bit loads of the image (and the correction arrays) land in registers, are cast,
//                                  corrected and masked there and parked in the warp's buffer once the
//                                  consumers have released it.  The register files of the stager warps are the landing
//                                  zone for the image stream, so that about as many image bytes as matrix bytes are in
//                                  flight and neither stream starves the other.  (One owner per buffer also keeps every
//                                  waiter at most one phase behind its mbarrier, which parity waits require.)
//   consumers (kConsWarps warps)   groups of kLanes lanes each own one (tile, bin) segment at a time: coefficients and
//                                  positions come from the matrix stage, values are gathered from the tile buffer,
//                                  accumulated per lane with compensation, merged by shuffles and
//                                  written as one partial per segment.
//
// With more than one frame per item the matrix stage is loaded once and reused for every frame of the item: that is
// the batched variant that amortises the matrix read across frames.
#include "tiled_common.cuh"

namespace {

constexpr int kStageWarps = kPipeMaxImgStages;    // 1 + 7 + 8 = 16 warps: four per scheduler, 128 registers each
constexpr int kConsWarps = 8;
constexpr int kConsumers = kConsWarps * 32;
constexpr int kPipeThreads = 32 + kStageWarps * 32 + kConsumers;
constexpr int kGroupsPerWarp = 32 / kLanes;
constexpr int kConsGroups = kConsumers / kLanes;
constexpr int kMaxMatStages = 4;
constexpr int kMaxImgStages = 8;
static_assert(kPipeMaxImgStages <= kMaxImgStages, "image ring deeper than the barrier array");
static_assert((2 * kMaxMatStages + 2 * kMaxImgStages) * 8 + kMaxImgStages * 4 <= kPipeHeaderBytes, "header too small");

struct PipeParams {
    const int4 *tile_desc;       // LPT order: {first entry, number of entries, first segment, number of segments}
    const int *tile_order;       // LPT order: tile id
    const int4 *seg_meta;
    const float *tcoef;
    const uint16_t *tidx;
    int tiles_x, tile_h, ntiles, nslot;
    int mat_stages, img_stages, coef_bytes, idx_bytes, meta_bytes, img_stage_bytes;
    const void *frames;
    int64_t frame_stride;
    int nframes, frames_per_item, nitems;
    Corrections cor;
    int height, width, vec_ok;
    void *partials;
};

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
// bounded wait: a protocol bug traps (the launch fails with an error) instead of hanging the device
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    for (uint32_t spin = 0; !mbar_try_wait(bar, parity); ++spin)
        if (spin > (1u << 20)) __trap();
}
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ---- development aid: per-block event trace (compiled in only with -DAI_PIPE_TRACE) -------
#ifdef AI_PIPE_TRACE
__device__ long long *g_trace = nullptr;          // [grid][kTraceItems][8] clock64 stamps
constexpr int kTraceItems = 16;
#define AI_TRACE(item, slot)                                                                             \
    do {                                                                                                 \
        if (g_trace && (item) < kTraceItems) g_trace[((size_t)blockIdx.x * kTraceItems + (item)) * 8 + (slot)] = clock64(); \
    } while (0)
#else
#define AI_TRACE(item, slot) do { } while (0)
#endif

// n-th use of a ring of `stages` buffers -> (stage, parity of the phase that use completes)
struct Slot {
    int stage;
    uint32_t parity;
    __device__ Slot(int n, int stages) : stage(n % stages), parity((uint32_t)(n / stages) & 1u) {}
};

// The segments of one staged tile.  Segment records are sorted by descending length; consecutive records go to the
// lane groups of one warp, warps take runs of records in snake order, so the lanes of a warp finish together and the
// warps carry similar loads.  Per lane the loop is software-pipelined: coefficient / position loads run two steps ahead
// of the accumulate, the gathers one step ahead.
template <int ACC, bool TRACK>
__device__ __forceinline__ void consume_tile(const float *tile, const float *coef, const uint16_t *idx,
                                             const int4 *meta, const int4 &desc, void *part_f, int cwarp, int lane)
{
    const int g = lane / kLanes, gl = lane % kLanes;
    const float4 zero4 = make_float4(0, 0, 0, 0);
    const ushort4 zeroi = make_ushort4(0, 0, 0, 0);
    for (int round = 0; round * kConsGroups < desc.w; ++round) {
        const int wslot = (round & 1) ? kConsWarps - 1 - cwarp : cwarp;
        const int sl = round * kConsGroups + wslot * kGroupsPerWarp + g;
        const bool has = sl < desc.w;
        const int4 m = has ? meta[sl] : make_int4(0, 0, 0, 0);
        const int end = has ? m.y - desc.x : 0;
        int k = has ? m.x - desc.x + gl * 4 : 0;
        Accum2<ACC> S2, C2;
        float4 c0 = zero4, c1 = zero4;
        ushort4 x0 = zeroi, x1 = zeroi;
        if (k < end) {
            c0 = *reinterpret_cast<const float4 *>(coef + k);
            x0 = *reinterpret_cast<const ushort4 *>(idx + k);
        }
        if (k + kStep < end) {
            c1 = *reinterpret_cast<const float4 *>(coef + k + kStep);
            x1 = *reinterpret_cast<const ushort4 *>(idx + k + kStep);
        }
        float4 v0 = gather4(tile, x0);
        while (k < end) {
            float4 c2 = zero4;
            ushort4 x2 = zeroi;
            if (k + 2 * kStep < end) {
                c2 = *reinterpret_cast<const float4 *>(coef + k + 2 * kStep);
                x2 = *reinterpret_cast<const ushort4 *>(idx + k + 2 * kStep);
            }
            const float4 v1 = gather4(tile, x1);
            accumulate4<ACC, TRACK>(c0, v0, S2, C2);
            c0 = c1; v0 = v1; c1 = c2; x1 = x2;
            k += kStep;
        }
        Accum<ACC> S = S2.total(), C = C2.total();
        group_reduce<ACC>(S);
        if constexpr (TRACK) group_reduce<ACC>(C);
        if (gl == 0 && has) store_partial<ACC>(part_f, m.z, S, C, TRACK, (double)__int_as_float(m.w));
    }
}

template <int DT, int ACC>
__global__ void __launch_bounds__(kPipeThreads, 1) tiled_pipe_kernel(const PipeParams p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *mat_full = reinterpret_cast<uint64_t *>(smem);
    uint64_t *mat_empty = mat_full + kMaxMatStages;
    uint64_t *img_full = mat_empty + kMaxMatStages;
    uint64_t *img_empty = img_full + kMaxImgStages;
    volatile int *img_flag = reinterpret_cast<volatile int *>(img_empty + kMaxImgStages);
    const int mat_stage_bytes = p.coef_bytes + p.idx_bytes + p.meta_bytes;
    unsigned char *mat_base = smem + kPipeHeaderBytes;
    unsigned char *img_base = mat_base + (size_t)p.mat_stages * mat_stage_bytes;
    using T = typename RawType<DT>::T;

    if (threadIdx.x == 0) AI_TRACE(0, 7);
    if (threadIdx.x == 0) {
        for (int s = 0; s < kMaxMatStages; ++s) {
            mbar_init(mat_full + s, 1);
            mbar_init(mat_empty + s, kConsWarps);
        }
        for (int s = 0; s < kMaxImgStages; ++s) {
            mbar_init(img_full + s, 32);
            mbar_init(img_empty + s, kConsWarps);
            img_flag[s] = 0;
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp == 0) {
        // ===== producer: matrix slices by bulk copy ======================================================================
        if (lane == 0) {
            int n = 0;
            int4 d = blockIdx.x < p.nitems ? __ldg(p.tile_desc + (blockIdx.x % p.ntiles)) : make_int4(0, 0, 0, 0);
            for (int w = blockIdx.x; w < p.nitems; w += gridDim.x, ++n) {
                const int wn = w + gridDim.x;
                const int4 dn = wn < p.nitems ? __ldg(p.tile_desc + (wn % p.ntiles)) : make_int4(0, 0, 0, 0);
                const Slot ms(n, p.mat_stages);
                mbar_wait(mat_empty + ms.stage, ms.parity ^ 1u);
                AI_TRACE(n, 0);
                unsigned char *dst = mat_base + (size_t)ms.stage * mat_stage_bytes;
                const uint32_t cb = (uint32_t)d.y * 4u, ib = (uint32_t)d.y * 2u, mb = (uint32_t)d.w * 16u;
                if (cb + ib + mb > 0) {
                    mbar_arrive_expect_tx(mat_full + ms.stage, cb + ib + mb);
                    if (mb) bulk_g2s(dst + p.coef_bytes + p.idx_bytes, p.seg_meta + d.z, mb, mat_full + ms.stage);
                    if (ib) bulk_g2s(dst + p.coef_bytes, p.tidx + d.x, ib, mat_full + ms.stage);
                    if (cb) bulk_g2s(dst, p.tcoef + d.x, cb, mat_full + ms.stage);
                } else {
                    mbar_arrive(mat_full + ms.stage);
                }
                d = dn;
            }
        }
    } else if (warp <= kStageWarps) {
        // ===== stagers: image tile -> cast -> corrections -> shared memory; warp sw owns image stage sw ==================
        const int sw = warp - 1;
        if (sw >= p.img_stages) return;
        float *tile = reinterpret_cast<float *>(img_base + (size_t)sw * p.img_stage_bytes);
        int ii = 0;                                   // image items of this block, in consumption order
        for (int w = blockIdx.x; w < p.nitems; w += gridDim.x) {
            const int f0 = (w / p.ntiles) * p.frames_per_item;
            const int f1 = min(p.nframes, f0 + p.frames_per_item);
            const int first = ii + ((sw - ii) % p.img_stages + p.img_stages) % p.img_stages;   // first item of this warp
            if (first >= ii + (f1 - f0)) { ii += f1 - f0; continue; }
            const int t = __ldg(p.tile_order + (w % p.ntiles));
            const int ty = t / p.tiles_x, tx = t - ty * p.tiles_x;
            for (int it = first; it < ii + (f1 - f0); it += p.img_stages) {
                const int f = f0 + (it - ii);
                const uint32_t parity = (uint32_t)(it / p.img_stages) & 1u;
                const void *img = reinterpret_cast<const T *>(p.frames) + (int64_t)f * p.frame_stride;
                if (lane == 0) AI_TRACE(it, 1);
                const bool bad = stage_tile<DT, 32, 16, 3>(tile, img, p.cor, ty, tx, p.tile_h, p.height, p.width, p.vec_ok,
                                                           lane, [&] { mbar_wait(img_empty + sw, parity ^ 1u); });
                if (bad) img_flag[sw] = it + 1;              // value-equal writers; read after the barrier
                if (lane == 0) AI_TRACE(it, 2);
                mbar_arrive(img_full + sw);
            }
            ii += f1 - f0;
        }
    } else {
        // ===== consumers: gather-reduce per (tile, bin) segment ============================================================
        const int cwarp = warp - 1 - kStageWarps;
        int n = 0, ii = 0;
        int4 d = blockIdx.x < p.nitems ? __ldg(p.tile_desc + (blockIdx.x % p.ntiles)) : make_int4(0, 0, 0, 0);
        for (int w = blockIdx.x; w < p.nitems; w += gridDim.x, ++n) {
            const int wn = w + gridDim.x;
            const int4 dn = wn < p.nitems ? __ldg(p.tile_desc + (wn % p.ntiles)) : make_int4(0, 0, 0, 0);
            const int f0 = (w / p.ntiles) * p.frames_per_item;
            const int f1 = min(p.nframes, f0 + p.frames_per_item);
            const Slot ms(n, p.mat_stages);
            if (cwarp == 0 && lane == 0) AI_TRACE(n, 3);
            mbar_wait(mat_full + ms.stage, ms.parity);
            if (cwarp == 0 && lane == 0) AI_TRACE(n, 4);
            const unsigned char *mst = mat_base + (size_t)ms.stage * mat_stage_bytes;
            const float *coef = reinterpret_cast<const float *>(mst);
            const uint16_t *idx = reinterpret_cast<const uint16_t *>(mst + p.coef_bytes);
            const int4 *meta = reinterpret_cast<const int4 *>(mst + p.coef_bytes + p.idx_bytes);
            for (int f = f0; f < f1; ++f, ++ii) {
                const Slot is(ii, p.img_stages);
                mbar_wait(img_full + is.stage, is.parity);
                if (cwarp == 0 && lane == 0) AI_TRACE(ii, 5);
                const float *tile = reinterpret_cast<const float *>(img_base + (size_t)is.stage * p.img_stage_bytes);
                const bool track = img_flag[is.stage] == ii + 1;
                void *part_f = reinterpret_cast<char *>(p.partials) + (int64_t)f * p.nslot * 16;
                if (track) consume_tile<ACC, true>(tile, coef, idx, meta, d, part_f, cwarp, lane);
                else consume_tile<ACC, false>(tile, coef, idx, meta, d, part_f, cwarp, lane);
                __syncwarp();
                if (cwarp == 0 && lane == 0) AI_TRACE(ii, 6);
                if (lane == 0) mbar_arrive(img_empty + is.stage);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(mat_empty + ms.stage);
            d = dn;
        }
    }
}

template <int DT, int ACC>
int launch_pipe(ai_ctx *ctx, const PipeParams &p, size_t smem, int grid, cudaStream_t st)
{
    static int configured_device = -1;            // per instantiation: opt in to the large dynamic shared memory once
    if (configured_device != ctx->device) {
        AI_CUDA(ctx, cudaFuncSetAttribute(tiled_pipe_kernel<DT, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          kPipeSmemBudget));
        configured_device = ctx->device;
    }
    ai_prof_begin(ctx, st);
    tiled_pipe_kernel<DT, ACC><<<grid, kPipeThreads, smem, st>>>(p);
    ai_prof_end(ctx, st);
    AI_CUDA(ctx, cudaGetLastError());
    return AI_OK;
}

template <int DT>
int launch_pipe_dt(ai_ctx *ctx, const PipeParams &p, size_t smem, int grid, cudaStream_t st)
{
    switch (ctx->accum) {
    case AI_ACC_F32_KAHAN: return launch_pipe<DT, AI_ACC_F32_KAHAN>(ctx, p, smem, grid, st);
    case AI_ACC_F32_PLAIN: return launch_pipe<DT, AI_ACC_F32_PLAIN>(ctx, p, smem, grid, st);
    default: return launch_pipe<DT, AI_ACC_F64>(ctx, p, smem, grid, st);
    }
}

}  // namespace

#ifdef AI_PIPE_TRACE
extern "C" int ai_debug_set_trace(void *dev_buffer)
{
    return (int)cudaMemcpyToSymbol(g_trace, &dev_buffer, sizeof(void *));
}
#endif

// Launches the pipelined stage 1 if a tile's slice fits the shared-memory ring (*handled = true); otherwise leaves
// *handled false and the caller falls back to the one-block-per-tile kernel.
int ai_launch_pipe_stage1(ai_ctx *ctx, const FrameArgs &a, int vec_ok, cudaStream_t st, bool *handled)
{
    const TiledLayout &tl = ctx->tl;
    *handled = false;
    if (tl.ntiles < 1) return AI_OK;
    const PipePlan plan = ai_pipe_plan(tl.max_tile_entries, tl.max_tile_segs, tl.tile_h, a.nframes >= 16);
    if (!plan.fits) return AI_OK;                    // slice too large for a double buffer: direct kernel
    PipeParams p{};
    p.coef_bytes = plan.coef_bytes;
    p.idx_bytes = plan.idx_bytes;
    p.meta_bytes = plan.meta_bytes;
    p.mat_stages = plan.mat_stages;
    p.img_stages = plan.img_stages;
    p.img_stage_bytes = plan.img_stage_bytes;

    const int sms = ctx->sm_count > 0 ? ctx->sm_count : 148;
    // items: every tile once per chunk of frames; enough chunks that each block gets several items
    int nchunks = 1;
    if (a.nframes > 1) {
        nchunks = (8 * sms + tl.ntiles - 1) / tl.ntiles;
        if (nchunks > a.nframes) nchunks = a.nframes;
        if (nchunks < 1) nchunks = 1;
    }
    p.frames_per_item = (a.nframes + nchunks - 1) / nchunks;
    nchunks = (a.nframes + p.frames_per_item - 1) / p.frames_per_item;
    const int64_t nitems = (int64_t)tl.ntiles * nchunks;
    if (nitems > 0x7fffffffLL || nitems * p.frames_per_item > 0x3fffffffLL) return AI_OK;
    p.nitems = (int)nitems;
    p.tile_desc = tl.tile_desc;
    p.tile_order = tl.tile_order;
    p.seg_meta = tl.seg_meta;
    p.tcoef = tl.tcoef;
    p.tidx = tl.tidx;
    p.tiles_x = tl.tiles_x;
    p.tile_h = tl.tile_h;
    p.ntiles = tl.ntiles;
    p.nslot = tl.nslot;
    p.frames = a.image;
    p.frame_stride = a.frame_stride;
    p.nframes = a.nframes;
    p.cor = Corrections{a.dark, a.flat, a.solidangle, a.polarization, a.mask};
    p.height = ctx->height;
    p.width = ctx->width;
    p.vec_ok = vec_ok;
    p.partials = ctx->partials;
    const int grid = p.nitems < sms ? p.nitems : sms;
    int rc = AI_EINVAL;
    switch (a.dtype) {
    case AI_F32: rc = launch_pipe_dt<AI_F32>(ctx, p, plan.smem, grid, st); break;
    case AI_I32: rc = launch_pipe_dt<AI_I32>(ctx, p, plan.smem, grid, st); break;
    case AI_U16: rc = launch_pipe_dt<AI_U16>(ctx, p, plan.smem, grid, st); break;
    case AI_I16: rc = launch_pipe_dt<AI_I16>(ctx, p, plan.smem, grid, st); break;
    case AI_U32: rc = launch_pipe_dt<AI_U32>(ctx, p, plan.smem, grid, st); break;
    }
    if (rc == AI_OK) *handled = true;
    return rc;
}
