// TILED stage 1 as a persistent, warp-specialised, bulk-copy pipelined kernel -- the B200 design
// of the CSR SpMV of PAPER.md:174-188.
//
// One block per SM stays resident and walks a static list of work items (tile, range of frames), longest tiles first.
// Three roles run concurrently and hand buffers to each other through shared-memory mbarriers:
//
//   producer  (1 elected thread)   issues cp.async.bulk (TMA) copies of the tile's slice of the matrix -- coefficients,
//                                  16-bit pixel offsets, segment records, three contiguous ranges -- into a ring of
//                                  shared-memory stages, so whole tiles' worth of bytes are in flight per SM with no
//                                  registers held: this is what keeps HBM busy (the kernel is a pure stream).
//   stagers   (kStageWarps warps)  read the image tile (and the correction arrays) with 128-bit loads, cast, correct and
//                                  mask in registers and park the result in a ring of tile buffers.
//   consumers (kConsWarps warps)   groups of kLanes lanes each own one (tile, bin) segment at a time: coefficients and
//                                  offsets come from the matrix stage, values are gathered from the tile buffer,
//                                  accumulated per lane with compensation, merged by shuffles and
//                                  written as one partial per segment.
//
// With more than one frame per item the matrix stage is loaded once and reused for every frame of the item: that is
// the batched variant that amortises the matrix read across frames.
#include "tiled_common.cuh"

namespace {

constexpr int kStageWarps = 4;
constexpr int kConsWarps = 8;
constexpr int kStagers = kStageWarps * 32;
constexpr int kConsumers = kConsWarps * 32;
constexpr int kPipeThreads = 32 + kStagers + kConsumers;
constexpr int kConsGroups = kConsumers / kLanes;
constexpr int kMaxStages = 4;
constexpr int kHeaderBytes = 256;                 // mbarriers + per-image-stage flags
constexpr int kImgStageBytes = kTilePix * 4;
constexpr int kSmemBudget = 227 * 1024;

struct PipeParams {
    const int4 *tile_desc;       // LPT order: {first entry, number of entries, first segment, number of segments}
    const int *tile_order;       // LPT order: tile id
    const int4 *seg_meta;
    const float *tcoef;
    const uint16_t *tidx;
    int tiles_x, ntiles, nslot;
    int mat_stages, img_stages, coef_bytes, idx_bytes, meta_bytes;
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
        if (spin > (1u << 26)) __trap();
}
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

struct Ring {              // use counter -> (stage, parity)
    int n, it = 0;
    __device__ explicit Ring(int stages) : n(stages) {}
    __device__ int stage() const { return it % n; }
    __device__ uint32_t parity() const { return (uint32_t)(it / n) & 1u; }
    __device__ int generation() const { return it / n + 1; }
    __device__ void next() { ++it; }
};

template <int ACC, bool TRACK>
__device__ __forceinline__ void consume_tile(const float *tile, const float *coef, const uint16_t *idx,
                                             const int4 *meta, const int4 &desc, void *part_f, int ctid)
{
    const int group = ctid / kLanes, gl = ctid % kLanes;
    for (int sl = group;; sl += kConsGroups) {
        const bool has = sl < desc.w;
        if (!__any_sync(AI_FULL_MASK, has)) break;
        const int4 m = has ? meta[sl] : make_int4(0, 0, 0, 0);
        const int end = has ? m.y - desc.x : 0;
        Accum<ACC> S, C;
#pragma unroll 2
        for (int k = has ? m.x - desc.x + gl * 4 : 0; k < end; k += kStep) {
            const float4 c4 = *reinterpret_cast<const float4 *>(coef + k);
            const ushort4 i4 = *reinterpret_cast<const ushort4 *>(idx + k);
            consume4<ACC, TRACK>(tile, c4, i4, S, C);
        }
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
    uint64_t *mat_empty = mat_full + kMaxStages;
    uint64_t *img_full = mat_empty + kMaxStages;
    uint64_t *img_empty = img_full + kMaxStages;
    volatile int *img_flag = reinterpret_cast<volatile int *>(smem + 4 * kMaxStages * 8);
    const int mat_stage_bytes = p.coef_bytes + p.idx_bytes + p.meta_bytes;
    unsigned char *mat_base = smem + kHeaderBytes;
    unsigned char *img_base = mat_base + (size_t)p.mat_stages * mat_stage_bytes;
    using T = typename RawType<DT>::T;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kMaxStages; ++s) {
            mbar_init(mat_full + s, 1);
            mbar_init(mat_empty + s, kConsWarps);
            mbar_init(img_full + s, kStagers);
            mbar_init(img_empty + s, kConsWarps);
            img_flag[s] = 0;
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int warp = threadIdx.x >> 5;
    if (warp == 0) {
        // ===== producer: matrix slices by bulk copy ======================================================================
        if (threadIdx.x == 0) {
            Ring mr(p.mat_stages);
            for (int w = blockIdx.x; w < p.nitems; w += gridDim.x) {
                const int4 d = __ldg(p.tile_desc + (w % p.ntiles));
                const int m = mr.stage();
                mbar_wait(mat_empty + m, mr.parity() ^ 1u);
                unsigned char *dst = mat_base + (size_t)m * mat_stage_bytes;
                const uint32_t cb = (uint32_t)d.y * 4u, ib = (uint32_t)d.y * 2u, mb = (uint32_t)d.w * 16u;
                if (cb + ib + mb > 0) {
                    mbar_arrive_expect_tx(mat_full + m, cb + ib + mb);
                    if (cb) bulk_g2s(dst, p.tcoef + d.x, cb, mat_full + m);
                    if (ib) bulk_g2s(dst + p.coef_bytes, p.tidx + d.x, ib, mat_full + m);
                    if (mb) bulk_g2s(dst + p.coef_bytes + p.idx_bytes, p.seg_meta + d.z, mb, mat_full + m);
                } else {
                    mbar_arrive(mat_full + m);
                }
                mr.next();
            }
        }
    } else if (warp <= kStageWarps) {
        // ===== stagers: image tile -> cast -> corrections -> shared memory ==============================================
        const int stid = threadIdx.x - 32;
        Ring ir(p.img_stages);
        for (int w = blockIdx.x; w < p.nitems; w += gridDim.x) {
            const int t = __ldg(p.tile_order + (w % p.ntiles));
            const int ty = t / p.tiles_x, tx = t - ty * p.tiles_x;
            const int f0 = (w / p.ntiles) * p.frames_per_item;
            const int f1 = min(p.nframes, f0 + p.frames_per_item);
            for (int f = f0; f < f1; ++f) {
                const int i = ir.stage();
                mbar_wait(img_empty + i, ir.parity() ^ 1u);
                float *tile = reinterpret_cast<float *>(img_base + (size_t)i * kImgStageBytes);
                const void *img = reinterpret_cast<const T *>(p.frames) + (int64_t)f * p.frame_stride;
                const bool bad = stage_tile<DT, kStagers>(tile, img, p.cor, ty, tx, p.height, p.width, p.vec_ok, stid);
                if (bad) img_flag[i] = ir.generation();      // any value-equal writers; read after the barrier
                mbar_arrive(img_full + i);
                ir.next();
            }
        }
    } else {
        // ===== consumers: gather-reduce per (tile, bin) segment ============================================================
        const int ctid = threadIdx.x - 32 - kStagers;
        const int lane = threadIdx.x & 31;
        Ring mr(p.mat_stages), ir(p.img_stages);
        for (int w = blockIdx.x; w < p.nitems; w += gridDim.x) {
            const int4 d = __ldg(p.tile_desc + (w % p.ntiles));
            const int f0 = (w / p.ntiles) * p.frames_per_item;
            const int f1 = min(p.nframes, f0 + p.frames_per_item);
            const int m = mr.stage();
            mbar_wait(mat_full + m, mr.parity());
            const unsigned char *ms = mat_base + (size_t)m * mat_stage_bytes;
            const float *coef = reinterpret_cast<const float *>(ms);
            const uint16_t *idx = reinterpret_cast<const uint16_t *>(ms + p.coef_bytes);
            const int4 *meta = reinterpret_cast<const int4 *>(ms + p.coef_bytes + p.idx_bytes);
            for (int f = f0; f < f1; ++f) {
                const int i = ir.stage();
                mbar_wait(img_full + i, ir.parity());
                const float *tile = reinterpret_cast<const float *>(img_base + (size_t)i * kImgStageBytes);
                const bool track = img_flag[i] == ir.generation();
                void *part_f = reinterpret_cast<char *>(p.partials) + (int64_t)f * p.nslot * 16;
                if (track) consume_tile<ACC, true>(tile, coef, idx, meta, d, part_f, ctid);
                else consume_tile<ACC, false>(tile, coef, idx, meta, d, part_f, ctid);
                __syncwarp();
                if (lane == 0) mbar_arrive(img_empty + i);
                ir.next();
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(mat_empty + m);
            mr.next();
        }
    }
}

inline int align128(int x) { return (x + 127) & ~127; }

template <int DT, int ACC>
int launch_pipe(ai_ctx *ctx, const PipeParams &p, size_t smem, int grid, cudaStream_t st)
{
    static int configured_device = -1;            // per instantiation: opt in to the large dynamic shared memory once
    if (configured_device != ctx->device) {
        AI_CUDA(ctx, cudaFuncSetAttribute(tiled_pipe_kernel<DT, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          kSmemBudget));
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

// Launches the pipelined stage 1 if a tile's slice fits the shared-memory ring (*handled = true); otherwise leaves
// *handled false and the caller falls back to the one-block-per-tile kernel.
int ai_launch_pipe_stage1(ai_ctx *ctx, const FrameArgs &a, int vec_ok, cudaStream_t st, bool *handled)
{
    const TiledLayout &tl = ctx->tl;
    *handled = false;
    if (tl.ntiles < 1) return AI_OK;
    PipeParams p{};
    p.coef_bytes = align128(tl.max_tile_entries * 4);
    p.idx_bytes = align128(tl.max_tile_entries * 2);
    p.meta_bytes = align128(tl.max_tile_segs * 16);
    const int mat_stage = p.coef_bytes + p.idx_bytes + p.meta_bytes;
    // ring depths: 3 image stages if two matrix stages still fit, else 2; as many matrix stages as fit (2..3)
    int img_stages = 3, mat_stages = 0;
    for (; img_stages >= 2; --img_stages) {
        const int room = kSmemBudget - kHeaderBytes - img_stages * kImgStageBytes;
        mat_stages = mat_stage > 0 ? room / mat_stage : 3;
        if (mat_stages >= 2) break;
    }
    if (mat_stages < 2) return AI_OK;                // slice too large for a double buffer: direct kernel
    if (mat_stages > 3) mat_stages = 3;
    p.mat_stages = mat_stages;
    p.img_stages = img_stages;
    const size_t smem = (size_t)kHeaderBytes + (size_t)mat_stages * mat_stage + (size_t)img_stages * kImgStageBytes;

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
    if (nitems > 0x7fffffffLL) return AI_OK;
    p.nitems = (int)nitems;
    p.tile_desc = tl.tile_desc;
    p.tile_order = tl.tile_order;
    p.seg_meta = tl.seg_meta;
    p.tcoef = tl.tcoef;
    p.tidx = tl.tidx;
    p.tiles_x = tl.tiles_x;
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
    case AI_F32: rc = launch_pipe_dt<AI_F32>(ctx, p, smem, grid, st); break;
    case AI_I32: rc = launch_pipe_dt<AI_I32>(ctx, p, smem, grid, st); break;
    case AI_U16: rc = launch_pipe_dt<AI_U16>(ctx, p, smem, grid, st); break;
    case AI_I16: rc = launch_pipe_dt<AI_I16>(ctx, p, smem, grid, st); break;
    case AI_U32: rc = launch_pipe_dt<AI_U32>(ctx, p, smem, grid, st); break;
    }
    if (rc == AI_OK) *handled = true;
    return rc;
}
