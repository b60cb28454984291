// TILED stage 1 as a persistent, warp-specialised, TMA-pipelined kernel over the sliced layout
// -- the B200 design of the CSR SpMV of PAPER.md:174-188.
//
// One block per SM stays resident and walks a static list of work items (tile, range of frames), longest tiles first,
// dealt to the blocks in snake order.  Three roles run concurrently and hand buffers to each other through mbarriers:
//
//   producer  (1 elected thread)  in consumption order: the image tile of the item as two swizzled TMA boxes
//                                 (cp.async.bulk.tensor, SASS UTMALDG) into a ring of tile buffers, then the tile's
//                                 blob of the matrix as one bulk copy (cp.async.bulk, SASS UBLKCP) into a ring of
//                                 matrix stages.  No registers are held by data in flight.
//   stagers   (kStageWarps warps) TMA mode (32-bit pixels, no correction arrays, aligned rows): turn the raw tile into
//                                 float32 in place and look for non-finite pixels.  Otherwise: load the tile and the
//                                 correction arrays with 128-bit loads, cast, correct and mask in registers
//                                  and park the result in the tile buffer.
//   consumers (kConsWarps warps)  one lane per slice of a (tile, bin) segment: coefficients and pixel positions come
//                                 from the matrix stage with conflict-free 128 / 64-bit shared loads, pixel values are
//                                 gathered from the tile buffer, accumulated per lane with compensation
//                                 (PAPER.md:186-188), merged over the lanes of a run by shuffles with an error-free
//                                 two-sum, and written as one partial per run.
//
// With more than one frame per item the matrix stage is loaded once and reused for every frame of the item: that is
// the batched variant that amortises the matrix read across frames.
#include <cuda.h>

#include "tiled_common.cuh"

namespace {

constexpr int kStageWarps = 3;
constexpr int kConsWarps = 16;
constexpr int kPipeThreads = 32 * (1 + kStageWarps + kConsWarps);
static_assert((2 * kPipeMaxMatStages + 3 * kPipeMaxImgStages) * 8 + kPipeMaxImgStages * 4 <= kPipeHeaderBytes,
              "header too small");

struct PipeParams {
    const int4 *blob_desc;       // longest first: {blob offset / 16, blob bytes, tile id, number of blocks}
    const unsigned char *blob;
    int tiles_x, tile_h, ntiles, nslot;
    int mat_stages, img_stages, mat_stage_bytes, img_stage_bytes;
    const void *frames;
    int64_t frame_stride;
    int nframes, frames_per_item, nitems;
    Corrections cor;
    int height, width, vec_ok, use_tma;
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
        if (spin > (1u << 22)) __trap();
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
// orders this thread's shared-memory accesses through the generic proxy before later accesses of the async proxy (TMA)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// n-th use of a ring of `stages` buffers -> (stage, parity of the phase that use completes)
struct Slot {
    int stage;
    uint32_t parity;
    __device__ Slot(int n, int stages) : stage(n % stages), parity((uint32_t)(n / stages) & 1u) {}
};

// n-th item of this block: tiles (longest first) are dealt to the blocks in snake order
__device__ __forceinline__ int item_at(int n)
{
    return n * gridDim.x + ((n & 1) ? gridDim.x - 1 - blockIdx.x : blockIdx.x);
}

// One block of 32 slices against one staged tile: lane = slice.  All loads of the block are conflict-free 128 / 64-bit
// shared loads at consecutive addresses; the gathers hit the tile buffer at the stored byte offsets.
template <int ACC, bool TRACK>
__device__ __forceinline__ void consume_block(const float *tile, const unsigned char *blob, unsigned h, void *part_f,
                                              int lane)
{
    const int nsteps = h & 15, rounds = (h >> 4) & 7;
    const unsigned char *blk = blob + (size_t)(h >> 8) * 16;
    const float4 *cp = reinterpret_cast<const float4 *>(blk) + lane;
    const ushort4 *xp = reinterpret_cast<const ushort4 *>(blk + nsteps * 512) + lane;
    const int2 m = reinterpret_cast<const int2 *>(blk + nsteps * kBlkStepBytes)[lane];
    Accum2<ACC> S2, C2;
    if (nsteps == kSliceSteps) {
#pragma unroll
        for (int j = 0; j < kSliceSteps; ++j) consume4<ACC, TRACK>(tile, cp[j * 32], xp[j * 32], S2, C2);
    } else {
#pragma unroll
        for (int j = 0; j < kSliceSteps - 1; ++j)
            if (j < nsteps) consume4<ACC, TRACK>(tile, cp[j * 32], xp[j * 32], S2, C2);
    }
    Accum<ACC> S = S2.total(), C = C2.total();
    // lanes of a run are adjacent: suffix sums by doubling, the head of the run ends with the run's total
    const int rem = (m.x >> 24) & 31;
    for (int r = 0; r < rounds; ++r) {
        const int d = 1 << r;
        Accum<ACC> S_o = S, C_o = C;
        S_o.shfl_down(d);
        if constexpr (TRACK) C_o.shfl_down(d);
        if (rem >= d) {
            S.absorb(S_o);
            if constexpr (TRACK) C.absorb(C_o);
        }
    }
    if (m.x < 0) store_partial<ACC>(part_f, m.x & kMetaSlotMask, S, C, TRACK, (double)__int_as_float(m.y));
}

// TMA mode: the raw 32-bit tile becomes float32 in place; non-finite float pixels become NaN.  Returns true if this
// thread met an invalid pixel.
template <int DT>
__device__ __forceinline__ bool convert_tile_in_place(float *tile, int nchunk, int tid, int nthreads)
{
    bool bad = false;
    for (int q = tid; q < nchunk; q += nthreads) {
        float4 *p = reinterpret_cast<float4 *>(tile) + q;
        if constexpr (DT == AI_F32) {
            float4 v = *p;
            if (!finite_f(v.x) || !finite_f(v.y) || !finite_f(v.z) || !finite_f(v.w)) {
                v.x = finite_f(v.x) ? v.x : quiet_nan();
                v.y = finite_f(v.y) ? v.y : quiet_nan();
                v.z = finite_f(v.z) ? v.z : quiet_nan();
                v.w = finite_f(v.w) ? v.w : quiet_nan();
                *p = v;
                bad = true;
            }
        } else if constexpr (DT == AI_I32) {
            const int4 v = *reinterpret_cast<const int4 *>(p);
            *p = make_float4((float)v.x, (float)v.y, (float)v.z, (float)v.w);
        } else if constexpr (DT == AI_U32) {
            const uint4 v = *reinterpret_cast<const uint4 *>(p);
            *p = make_float4((float)v.x, (float)v.y, (float)v.z, (float)v.w);
        }
    }
    return bad;
}

template <int DT, int ACC>
__global__ void __launch_bounds__(kPipeThreads, 1) tiled_pipe_kernel(const __grid_constant__ CUtensorMap tmap,
                                                                     const PipeParams p)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    uint64_t *mat_full = reinterpret_cast<uint64_t *>(smem);       // matrix stage loaded (bulk copy complete)
    uint64_t *mat_empty = mat_full + kPipeMaxMatStages;            // every consumer warp is done with it
    uint64_t *raw_full = mat_empty + kPipeMaxMatStages;            // TMA mode: raw tile landed
    uint64_t *img_ready = raw_full + kPipeMaxImgStages;            // tile converted / staged: consumers may gather
    uint64_t *img_empty = img_ready + kPipeMaxImgStages;           // every consumer warp is done with it
    volatile int *img_flag = reinterpret_cast<volatile int *>(img_empty + kPipeMaxImgStages);
    unsigned char *mat_base = smem + kPipeHeaderBytes;
    unsigned char *img_base = mat_base + (size_t)p.mat_stages * p.mat_stage_bytes;
    using T = typename RawType<DT>::T;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kPipeMaxMatStages; ++s) {
            mbar_init(mat_full + s, 1);
            mbar_init(mat_empty + s, kConsWarps);
        }
        for (int s = 0; s < kPipeMaxImgStages; ++s) {
            mbar_init(raw_full + s, 1);
            mbar_init(img_ready + s, kStageWarps);
            mbar_init(img_empty + s, kConsWarps);
            img_flag[s] = 0;
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp == 0) {
        // ===== producer ================================================================================================
        if (lane != 0) return;
        int ii = 0;
        for (int n = 0;; ++n) {
            const int w = item_at(n);
            if (w >= p.nitems) break;
            const int4 d = __ldg(p.blob_desc + (w % p.ntiles));
            const int f0 = (w / p.ntiles) * p.frames_per_item;
            const int f1 = min(p.nframes, f0 + p.frames_per_item);
            const int ty = d.z / p.tiles_x, tx = d.z - ty * p.tiles_x;
            for (int f = f0; f < f1; ++f, ++ii) {
                if (p.use_tma) {
                    const Slot is(ii, p.img_stages);
                    mbar_wait(img_empty + is.stage, is.parity ^ 1u);
                    unsigned char *dst = img_base + (size_t)is.stage * p.img_stage_bytes;
                    mbar_arrive_expect_tx(raw_full + is.stage, (uint32_t)p.img_stage_bytes);
                    tma_box(dst, &tmap, tx * kTileW, ty * p.tile_h, f, raw_full + is.stage);
                    tma_box(dst + p.img_stage_bytes / 2, &tmap, tx * kTileW + 32, ty * p.tile_h, f, raw_full + is.stage);
                }
                if (f == f0) {
                    const Slot ms(n, p.mat_stages);
                    mbar_wait(mat_empty + ms.stage, ms.parity ^ 1u);
                    mbar_arrive_expect_tx(mat_full + ms.stage, (uint32_t)d.y);
                    bulk_g2s(mat_base + (size_t)ms.stage * p.mat_stage_bytes, p.blob + (size_t)d.x * 16, (uint32_t)d.y,
                             mat_full + ms.stage);
                }
            }
        }
    } else if (warp <= kStageWarps) {
        // ===== stagers: raw tile -> float32, corrected, invalid pixels as NaN ==========================================
        const int sw = warp - 1, tid = sw * 32 + lane;
        int ii = 0;
        for (int n = 0;; ++n) {
            const int w = item_at(n);
            if (w >= p.nitems) break;
            const int f0 = (w / p.ntiles) * p.frames_per_item;
            const int f1 = min(p.nframes, f0 + p.frames_per_item);
            const int t = __ldg(p.blob_desc + (w % p.ntiles)).z;
            const int ty = t / p.tiles_x, tx = t - ty * p.tiles_x;
            for (int f = f0; f < f1; ++f, ++ii) {
                const Slot is(ii, p.img_stages);
                float *tile = reinterpret_cast<float *>(img_base + (size_t)is.stage * p.img_stage_bytes);
                bool bad;
                if (p.use_tma) {
                    mbar_wait(raw_full + is.stage, is.parity);
                    bad = convert_tile_in_place<DT>(tile, p.tile_h * (kTileW / 4), tid, kStageWarps * 32);
                    if (DT != AI_F32 || bad) fence_proxy_async();      // generic-proxy writes before the next TMA write
                } else {
                    const void *img = reinterpret_cast<const T *>(p.frames) + (int64_t)f * p.frame_stride;
                    bad = stage_tile<DT, kStageWarps * 32, 8, 3>(tile, img, p.cor, ty, tx, p.tile_h, p.height, p.width,
                                                                  p.vec_ok, tid,
                                                                  [&] { mbar_wait(img_empty + is.stage, is.parity ^ 1u); });
                }
                if (bad) img_flag[is.stage] = ii + 1;           // value-equal writers; read after the barrier
                __syncwarp();
                if (lane == 0) mbar_arrive(img_ready + is.stage);
            }
        }
    } else {
        // ===== consumers: gather-reduce, one lane per slice ============================================================
        const int cw = warp - 1 - kStageWarps;
        int ii = 0, dealt = 0;                       // blocks are dealt round-robin to the warps across tiles
        for (int n = 0;; ++n) {
            const int w = item_at(n);
            if (w >= p.nitems) break;
            const int4 d = __ldg(p.blob_desc + (w % p.ntiles));
            const int f0 = (w / p.ntiles) * p.frames_per_item;
            const int f1 = min(p.nframes, f0 + p.frames_per_item);
            const Slot ms(n, p.mat_stages);
            mbar_wait(mat_full + ms.stage, ms.parity);
            const unsigned char *blob = mat_base + (size_t)ms.stage * p.mat_stage_bytes;
            const unsigned *hdr = reinterpret_cast<const unsigned *>(blob) + 1;
            const int first = (cw - dealt % kConsWarps + kConsWarps) % kConsWarps;
            for (int f = f0; f < f1; ++f, ++ii) {
                const Slot is(ii, p.img_stages);
                mbar_wait(img_ready + is.stage, is.parity);
                const float *tile = reinterpret_cast<const float *>(img_base + (size_t)is.stage * p.img_stage_bytes);
                const bool track = img_flag[is.stage] == ii + 1;
                void *part_f = reinterpret_cast<char *>(p.partials) + (int64_t)f * p.nslot * 16;
                if (track) {
                    for (int b = first; b < d.w; b += kConsWarps) consume_block<ACC, true>(tile, blob, hdr[b], part_f, lane);
                } else {
                    for (int b = first; b < d.w; b += kConsWarps) consume_block<ACC, false>(tile, blob, hdr[b], part_f, lane);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(img_empty + is.stage);
            }
            dealt += d.w;
            __syncwarp();
            if (lane == 0) mbar_arrive(mat_empty + ms.stage);
        }
    }
}

// ---- host side -------------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// cuTensorMapEncodeTiled through the runtime's driver entry point lookup: no link-time dependency on libcuda
EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
        if (cudaGetDriverEntryPointByVersion("cuTensorMapEncodeTiled", &p, 12000, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            p = nullptr;
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    return fn;
}

// (x, y, frame) view of the frames, boxes of 32 pixels x tile_h rows x 1 frame, 128-byte swizzle, zeros outside
int make_frame_map(ai_ctx *ctx, const FrameArgs &a, int tile_h, CUtensorMap *map)
{
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return ai_fail(ctx, AI_ECUDA, "cuTensorMapEncodeTiled is not available from this driver");
    const CUtensorMapDataType dt = a.dtype == AI_F32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32
                                 : a.dtype == AI_I32 ? CU_TENSOR_MAP_DATA_TYPE_INT32 : CU_TENSOR_MAP_DATA_TYPE_UINT32;
    const cuuint64_t dims[3] = {(cuuint64_t)ctx->width, (cuuint64_t)ctx->height, (cuuint64_t)a.nframes};
    const cuuint64_t strides[2] = {(cuuint64_t)ctx->width * 4, (cuuint64_t)a.frame_stride * 4};
    const cuuint32_t box[3] = {32, (cuuint32_t)tile_h, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = enc(map, dt, 3, const_cast<void *>(a.image), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return ai_fail(ctx, AI_ECUDA, "cuTensorMapEncodeTiled failed with %d", (int)r);
    return AI_OK;
}

template <int DT, int ACC>
int launch_pipe(ai_ctx *ctx, const CUtensorMap &map, const PipeParams &p, size_t smem, int grid, cudaStream_t st)
{
    static int configured_device = -1;            // per instantiation: opt in to the large dynamic shared memory once
    if (configured_device != ctx->device) {
        AI_CUDA(ctx, cudaFuncSetAttribute(tiled_pipe_kernel<DT, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          kPipeSmemBudget));
        configured_device = ctx->device;
    }
    ai_prof_begin(ctx, st);
    tiled_pipe_kernel<DT, ACC><<<grid, kPipeThreads, smem, st>>>(map, p);
    ai_prof_end(ctx, st);
    AI_CUDA(ctx, cudaGetLastError());
    return AI_OK;
}

template <int DT>
int launch_pipe_dt(ai_ctx *ctx, const CUtensorMap &map, const PipeParams &p, size_t smem, int grid, cudaStream_t st)
{
    switch (ctx->accum) {
    case AI_ACC_F32_KAHAN: return launch_pipe<DT, AI_ACC_F32_KAHAN>(ctx, map, p, smem, grid, st);
    case AI_ACC_F32_PLAIN: return launch_pipe<DT, AI_ACC_F32_PLAIN>(ctx, map, p, smem, grid, st);
    default: return launch_pipe<DT, AI_ACC_F64>(ctx, map, p, smem, grid, st);
    }
}

}  // namespace

// Launches the pipelined stage 1 if a tile's blob fits the shared-memory ring (*handled = true); otherwise leaves
// *handled false and the caller falls back to the one-block-per-tile kernel.
int ai_launch_pipe_stage1(ai_ctx *ctx, const FrameArgs &a, int vec_ok, cudaStream_t st, bool *handled)
{
    const TiledLayout &tl = ctx->tl;
    *handled = false;
    if (tl.ntiles < 1 || !tl.blob) return AI_OK;
    const PipePlan plan = ai_pipe_plan(tl.max_blob_bytes, tl.tile_h, a.nframes >= 16);
    if (!plan.fits) return AI_OK;                    // blob too large for the ring: direct kernel
    PipeParams p{};
    p.mat_stages = plan.mat_stages;
    p.img_stages = plan.img_stages;
    p.mat_stage_bytes = plan.mat_stage_bytes;
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
    if (nitems > 0x3fffffffLL || nitems * p.frames_per_item > 0x3fffffffLL) return AI_OK;
    p.nitems = (int)nitems;
    p.blob_desc = tl.blob_desc;
    p.blob = tl.blob;
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
    // TMA for the image: 32-bit pixels, nothing to correct, rows and frames on 16-byte boundaries
    const bool plain = !a.dark && !a.flat && !a.solidangle && !a.polarization && !a.mask;
    const bool is32 = a.dtype == AI_F32 || a.dtype == AI_I32 || a.dtype == AI_U32;
    p.use_tma = plain && is32 && vec_ok && (reinterpret_cast<uintptr_t>(a.image) % 16) == 0 && !ctx->no_tma;
    CUtensorMap map{};
    if (p.use_tma) {
        int rc = make_frame_map(ctx, a, tl.tile_h, &map);
        if (rc != AI_OK) return rc;
    }
    const int grid = p.nitems < sms ? p.nitems : sms;
    int rc = AI_EINVAL;
    switch (a.dtype) {
    case AI_F32: rc = launch_pipe_dt<AI_F32>(ctx, map, p, plan.smem, grid, st); break;
    case AI_I32: rc = launch_pipe_dt<AI_I32>(ctx, map, p, plan.smem, grid, st); break;
    case AI_U16: rc = launch_pipe_dt<AI_U16>(ctx, map, p, plan.smem, grid, st); break;
    case AI_I16: rc = launch_pipe_dt<AI_I16>(ctx, map, p, plan.smem, grid, st); break;
    case AI_U32: rc = launch_pipe_dt<AI_U32>(ctx, map, p, plan.smem, grid, st); break;
    }
    if (rc == AI_OK) *handled = true;
    return rc;
}
