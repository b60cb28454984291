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
//   stagers   (kStageGroups groups of kStageGroupWarps warps, alternate tiles) TMA mode (32-bit pixels, no correction arrays, aligned rows): turn the raw tile into
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
#include <string.h>

#include "pipe_common.cuh"
#include "tiled_common.cuh"

namespace {

constexpr int kStageGroups = 1;                      // stager groups work on alternate tile images (two groups keep the
constexpr int kStageGroupWarps = 3;                  // loads of two tiles in flight, but 23 warps cap the kernel at 80
                                                     // registers and slow the consumers down: measured, one group kept)
constexpr int kStageWarps = kStageGroups * kStageGroupWarps;
constexpr int kConsWarps = 16;
constexpr int kPipeThreads = 32 * (1 + kStageWarps + kConsWarps);
static_assert((kConsWarps & (kConsWarps - 1)) == 0, "block dealing assumes a power of two");
static_assert((2 * kPipeMaxMatStages + 3 * kPipeMaxImgStages) * 8 + kPipeMaxImgStages * 4 <= kPipeHeaderBytes,
              "header too small");

struct PipeParams {
    const int4 *blob_desc;       // longest first: {blob offset / 16, blob bytes, tile row << 16 | column, blocks}
    const unsigned char *blob;
    int tiles_x, tile_h, ntiles, nslot;
    int mat_stages, img_stages, mat_stage_bytes, img_stage_bytes;
    const void *frames;
    int64_t frame_stride;
    int nframes, frames_per_item, nitems;
    Corrections cor;
    int height, width, vec_ok, use_tma, inflight;
    void *partials;
};


// n-th item of this block: tiles (longest first) are dealt to the blocks in snake order
__device__ __forceinline__ int item_at(int n)
{
    return n * gridDim.x + ((n & 1) ? gridDim.x - 1 - blockIdx.x : blockIdx.x);
}

// (tile rank, chunk of frames) of successive items of this block, without integer division
struct ItemWalk {
    int rank = 0, chunk = 0, prev = 0;
    __device__ __forceinline__ void to(int w, int ntiles)
    {
        rank += w - prev;
        prev = w;
        while (rank >= ntiles) { rank -= ntiles; ++chunk; }
    }
};

// Descriptors of this block's items, fetched 32 at a time (lane l holds item n0 + l) one window ahead of their use, so
// that no role ever waits on a dependent global load between two items.  All lanes of the warp call get() together.
struct DescWindow {
    int4 cur, nxt;
    __device__ __forceinline__ static int4 load(const PipeParams &p, int k)
    {
        const int w = item_at(k);
        return w < p.nitems ? __ldg(p.blob_desc + (p.nitems == p.ntiles ? w : w % p.ntiles)) : make_int4(0, 0, 0, 0);
    }
    __device__ __forceinline__ void init(const PipeParams &p, int lane)
    {
        cur = load(p, lane);
        nxt = load(p, 32 + lane);
    }
    __device__ __forceinline__ int4 get(const PipeParams &p, int n, int lane)
    {
        if ((n & 31) == 0 && n > 0) {
            cur = nxt;
            nxt = load(p, n + 32 + lane);
        }
        int4 d;
        d.x = __shfl_sync(AI_FULL_MASK, cur.x, n & 31);
        d.y = __shfl_sync(AI_FULL_MASK, cur.y, n & 31);
        d.z = __shfl_sync(AI_FULL_MASK, cur.z, n & 31);
        d.w = __shfl_sync(AI_FULL_MASK, cur.w, n & 31);
        return d;
    }
};

// One block of 32 slices against one staged tile: lane = slice.  All loads of the block are conflict-free 128 / 64-bit
// shared loads at consecutive addresses; the gathers hit the tile buffer at the stored byte offsets.
// `lazy` (used with TRACK false): the tile was not screened for non-finite pixels; a non-finite lane sum anywhere in
// the warp means one may have been gathered, nothing is stored and true is returned -- the caller repeats the block
// with TRACK, which skips such pixels and accumulates count.  The step loop is kept rolled (two steps per trip, loads
// one trip ahead): the hot code of all consumer warps must stay inside the instruction cache.
template <int ACC, bool TRACK>
__device__ __noinline__ bool consume_block(const float *tile, const unsigned char *blob, unsigned h, void *part_f,
                                           int lane, bool lazy)
{
    const int nsteps = h & 15, rounds = (h >> 4) & 7;
    const unsigned char *blk = blob + (size_t)(h >> 8) * 16;
    const float4 *cp = reinterpret_cast<const float4 *>(blk) + lane;
    const ushort4 *xp = reinterpret_cast<const ushort4 *>(blk + nsteps * 512) + lane;
    const int2 m = reinterpret_cast<const int2 *>(blk + nsteps * kBlkStepBytes)[lane];
    const float4 zero4 = make_float4(0, 0, 0, 0);
    const ushort4 zeroi = make_ushort4(0, 0, 0, 0);
    AccumQ<ACC> S2, C2;
    float4 c0 = cp[0], c1 = nsteps > 1 ? cp[32] : zero4;
    ushort4 x0 = xp[0], x1 = nsteps > 1 ? xp[32] : zeroi;
#pragma unroll 1
    for (int j = 2; j < nsteps + 2; j += 2) {
        float4 n0 = zero4, n1 = zero4;
        ushort4 y0 = zeroi, y1 = zeroi;
        if (j < nsteps) { n0 = cp[j * 32]; y0 = xp[j * 32]; }
        if (j + 1 < nsteps) { n1 = cp[j * 32 + 32]; y1 = xp[j * 32 + 32]; }
        const float4 v0 = gather4(tile, x0), v1 = gather4(tile, x1);
        accumulate4<ACC, TRACK>(c0, v0, S2, C2);
        accumulate4<ACC, TRACK>(c1, v1, S2, C2);
        c0 = n0; c1 = n1; x0 = y0; x1 = y1;
    }
    Accum<ACC> S = S2.total(), C = C2.total();
    if constexpr (!TRACK) {
        if (lazy && __any_sync(AI_FULL_MASK, !finite_f((float)S.s))) return true;
    }
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
    return false;
}

// TMA mode: the raw 32-bit tile becomes float32 in place; non-finite float pixels become NaN.  Returns true if this
// thread met an invalid pixel.
template <int DT>
__device__ __forceinline__ bool convert_tile_in_place(float *tile, int nchunk, int tid, int nthreads)
{
    bool bad = false;
    if constexpr (DT == AI_F32) {
        // all loads first (independent), then one test per 128 bits: exponent field all ones <=> Inf or NaN
        constexpr int U = 6;
        for (int q0 = tid; q0 < nchunk; q0 += nthreads * U) {
            uint4 v[U];
#pragma unroll
            for (int i = 0; i < U; ++i) {
                const int q = q0 + i * nthreads;
                v[i] = q < nchunk ? reinterpret_cast<const uint4 *>(tile)[q] : make_uint4(0, 0, 0, 0);
            }
#pragma unroll
            for (int i = 0; i < U; ++i) {
                const unsigned e = 0x7f800000u;
                if ((v[i].x & e) == e || (v[i].y & e) == e || (v[i].z & e) == e || (v[i].w & e) == e) {
                    float4 *p = reinterpret_cast<float4 *>(tile) + (q0 + i * nthreads);
                    float4 f = *p;
                    f.x = finite_f(f.x) ? f.x : quiet_nan();
                    f.y = finite_f(f.y) ? f.y : quiet_nan();
                    f.z = finite_f(f.z) ? f.z : quiet_nan();
                    f.w = finite_f(f.w) ? f.w : quiet_nan();
                    *p = f;
                    bad = true;
                }
            }
        }
        return bad;
    }
    for (int q = tid; q < nchunk; q += nthreads) {
        float4 *p = reinterpret_cast<float4 *>(tile) + q;
        if constexpr (DT == AI_I32) {
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
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // float32 frames that arrive by TMA need no staging pass: consumers gather from the raw tile and detect
    // non-finite pixels lazily (consume_block)
    const bool direct = DT == AI_F32 && p.use_tma;
    DescWindow win;
    win.init(p, lane);

    if (threadIdx.x == 0) {
        for (int s = 0; s < kPipeMaxMatStages; ++s) {
            mbar_init(mat_full + s, 1);
            mbar_init(mat_empty + s, kConsWarps);
        }
        for (int s = 0; s < kPipeMaxImgStages; ++s) {
            mbar_init(raw_full + s, 1);
            mbar_init(img_ready + s, kStageGroupWarps);
            mbar_init(img_empty + s, kConsWarps);
            img_flag[s] = 0;
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // stage 2 is launched with programmatic stream serialisation: let its blocks be scheduled as SMs free up (they
    // wait in griddepcontrol.wait until this whole grid has completed)
    asm volatile("griddepcontrol.launch_dependents;");

    ItemWalk walk;
    Ring mr, ir;                                     // matrix ring position of item n, image ring position of image ii
    if (warp == 0) {
        // ===== producer: the warp stays converged (waits are warp-uniform), lane 0 issues the copies ===================
        for (int n = 0;; ++n) {
            const int w = item_at(n);
            if (w >= p.nitems) break;
            const int4 d = win.get(p, n, lane);
            if (d.w == 0) continue;                       // tile without entries: skipped by every role
            walk.to(w, p.ntiles);
            const int f0 = walk.chunk * p.frames_per_item;
            const int f1 = min(p.nframes, f0 + p.frames_per_item);
            const int ty = d.z >> 16, tx = d.z & 0xffff;
            if (p.inflight && n >= p.inflight) {         // pace: at most `inflight` blobs outstanding
                const int k = n - p.inflight;
                mbar_wait(mat_full + k % p.mat_stages, (uint32_t)(k / p.mat_stages) & 1u);
            }
            for (int f = f0; f < f1; ++f) {
                if (p.use_tma) {
                    mbar_wait(img_empty + ir.stage, ir.parity ^ 1u);
                    if (lane == 0) {
                        unsigned char *dst = img_base + (size_t)ir.stage * p.img_stage_bytes;
                        mbar_arrive_expect_tx(raw_full + ir.stage, (uint32_t)p.img_stage_bytes);
                        tma_box(dst, &tmap, tx * kTileW, ty * p.tile_h, f, raw_full + ir.stage);
                        tma_box(dst + p.img_stage_bytes / 2, &tmap, tx * kTileW + 32, ty * p.tile_h, f, raw_full + ir.stage);
                    }
                    ir.next(p.img_stages);
                }
                if (f == f0) {
                    mbar_wait(mat_empty + mr.stage, mr.parity ^ 1u);
                    if (lane == 0) {
                        mbar_arrive_expect_tx(mat_full + mr.stage, (uint32_t)d.y);
                        bulk_g2s(mat_base + (size_t)mr.stage * p.mat_stage_bytes, p.blob + (size_t)d.x * 16,
                                 (uint32_t)d.y, mat_full + mr.stage);
                    }
                    mr.next(p.mat_stages);
                }
            }
        }
    } else if (warp <= kStageWarps) {
        // ===== stagers: raw tile -> float32, corrected, invalid pixels as NaN ==========================================

        if (direct) return;
        const int sw = warp - 1, group = sw / kStageGroupWarps, tid = (sw % kStageGroupWarps) * 32 + lane;
        constexpr int kGroupThreads = kStageGroupWarps * 32;
        int ii = 0;
        for (int n = 0;; ++n) {
            const int w = item_at(n);
            if (w >= p.nitems) break;
            const int4 d = win.get(p, n, lane);
            if (d.w == 0) continue;
            walk.to(w, p.ntiles);
            const int f0 = walk.chunk * p.frames_per_item;
            const int f1 = min(p.nframes, f0 + p.frames_per_item);
            const int ty = d.z >> 16, tx = d.z & 0xffff;
            for (int f = f0; f < f1; ++f, ++ii) {
                if (ii % kStageGroups != group) {        // the other group's image
                    ir.next(p.img_stages);
                    continue;
                }
                float *tile = reinterpret_cast<float *>(img_base + (size_t)ir.stage * p.img_stage_bytes);
                bool bad;
                if (p.use_tma) {
                    mbar_wait(raw_full + ir.stage, ir.parity);
                    bad = convert_tile_in_place<DT>(tile, p.tile_h * (kTileW / 4), tid, kGroupThreads);
                    fence_proxy_async();               // generic-proxy writes before the next TMA write to the stage
                } else {
                    const void *img = reinterpret_cast<const T *>(p.frames) + (int64_t)f * p.frame_stride;
                    bad = stage_tile<DT, kGroupThreads, 8, 3>(tile, img, p.cor, ty, tx, p.tile_h, p.height, p.width,
                                                                  p.vec_ok, tid,
                                                                  [&] { mbar_wait(img_empty + ir.stage, ir.parity ^ 1u); });
                }
                if (bad) img_flag[ir.stage] = ii + 1;           // value-equal writers; read after the barrier
                __syncwarp();
                if (lane == 0) mbar_arrive(img_ready + ir.stage);
                ir.next(p.img_stages);
            }
        }
    } else {
        // ===== consumers: gather-reduce, one lane per slice ============================================================
        // A tile's blocks are dealt round-robin to the warps, continuing across tiles.
        const int cw = warp - 1 - kStageWarps;
        uint64_t *img_bar = direct ? raw_full : img_ready;
        int ii = 0, first = cw;
        for (int n = 0;; ++n) {
            const int w = item_at(n);
            if (w >= p.nitems) break;
            const int4 d = win.get(p, n, lane);
            if (d.w == 0) continue;
            walk.to(w, p.ntiles);
            const int f0 = walk.chunk * p.frames_per_item;
            const int f1 = min(p.nframes, f0 + p.frames_per_item);
            // Every warp waits on and arrives at every barrier, also for items of which it holds no block: no warp
            // is ever a whole phase away from a barrier (parity waits would alias).
            const bool mine = first < d.w;
            mbar_wait(mat_full + mr.stage, mr.parity);
            const unsigned char *blob = mat_base + (size_t)mr.stage * p.mat_stage_bytes;
            const unsigned *hdr = reinterpret_cast<const unsigned *>(blob) + 1;
            for (int f = f0; f < f1; ++f, ++ii) {
                mbar_wait(img_bar + ir.stage, ir.parity);
                if (mine) {
                    const float *tile = reinterpret_cast<const float *>(img_base + (size_t)ir.stage * p.img_stage_bytes);
                    void *part_f = reinterpret_cast<char *>(p.partials) + (int64_t)f * p.nslot * 16;
                    const bool track = !direct && img_flag[ir.stage] == ii + 1;
                    for (int b = first; b < d.w; b += kConsWarps) {
                        const unsigned h = hdr[b];
                        if (track || consume_block<ACC, false>(tile, blob, h, part_f, lane, direct))
                            consume_block<ACC, true>(tile, blob, h, part_f, lane, false);
                    }
                    __syncwarp();
                }
                if (lane == 0) mbar_arrive(img_empty + ir.stage);
                ir.next(p.img_stages);
            }
            if (lane == 0) mbar_arrive(mat_empty + mr.stage);
            // the warp after the one that took this tile's last block takes the next tile's first
            first -= d.w & (kConsWarps - 1);
            if (first < 0) first += kConsWarps;
            mr.next(p.mat_stages);
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

}  // namespace

// (x, y, frame) view of the frames, boxes of 32 pixels x tile_h rows x 1 frame, 128-byte swizzle, zeros outside.
// The maps of the last eight buffers are kept in the context: a stream of calls on a ring of buffers pays for
// cuTensorMapEncodeTiled once per buffer, not per call.
int ai_make_frame_map(ai_ctx *ctx, const FrameArgs &a, int tile_h, CUtensorMap *map, int box_frames)
{
    static_assert(sizeof(CUtensorMap) <= sizeof(ctx->map_cache[0].map), "tensor map cache too small");
    const int64_t pitch_el = a.row_pitch ? a.row_pitch : (int64_t)ctx->width;
    for (auto &e : ctx->map_cache)
        if (e.image == a.image && e.dtype == (int)a.dtype && e.tile_h == tile_h + 1024 * box_frames && e.nframes == a.nframes &&
            e.pitch == pitch_el && e.stride == a.frame_stride) {
            memcpy(map, e.map, sizeof(CUtensorMap));
            return AI_OK;
        }
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return ai_fail(ctx, AI_ECUDA, "cuTensorMapEncodeTiled is not available from this driver");
    const CUtensorMapDataType dt = a.dtype == AI_F32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32
                                 : a.dtype == AI_I32 ? CU_TENSOR_MAP_DATA_TYPE_INT32 : CU_TENSOR_MAP_DATA_TYPE_UINT32;
    const cuuint64_t dims[3] = {(cuuint64_t)ctx->width, (cuuint64_t)ctx->height, (cuuint64_t)a.nframes};
    const cuuint64_t strides[2] = {(cuuint64_t)pitch_el * 4, (cuuint64_t)a.frame_stride * 4};
    const cuuint32_t box[3] = {32, (cuuint32_t)tile_h, (cuuint32_t)box_frames};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = enc(map, dt, 3, const_cast<void *>(a.image), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return ai_fail(ctx, AI_ECUDA, "cuTensorMapEncodeTiled failed with %d", (int)r);
    auto &e = ctx->map_cache[ctx->map_next++ % (sizeof(ctx->map_cache) / sizeof(ctx->map_cache[0]))];
    memcpy(e.map, map, sizeof(CUtensorMap));
    e.image = a.image;
    e.dtype = (int)a.dtype;
    e.tile_h = tile_h + 1024 * box_frames;
    e.nframes = a.nframes;
    e.pitch = pitch_el;
    e.stride = a.frame_stride;
    return AI_OK;
}

namespace {

template <int DT, int ACC>
int launch_pipe(ai_ctx *ctx, const CUtensorMap &map, const PipeParams &p, size_t smem, int grid, cudaStream_t st)
{
    const uint64_t bit = 1ULL << (30 + DT * 3 + ACC);      // per context and instantiation: opt in to the large
    if (!(ctx->smem_opt_in & bit)) {                       // dynamic shared memory once
        AI_CUDA(ctx, cudaFuncSetAttribute(tiled_pipe_kernel<DT, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          kPipeSmemBudget));
        ctx->smem_opt_in |= bit;
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
    const PipePlan plan = ai_pipe_plan(tl.max_blob_bytes, tl.tile_h, a.nframes >= 16, ctx->tune);
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
    p.inflight = ctx->tune.inflight > 0 && ctx->tune.inflight < plan.mat_stages ? ctx->tune.inflight : 0;
    // TMA for the image: 32-bit pixels, nothing to correct, rows and frames on 16-byte boundaries
    const bool plain = !a.dark && !a.flat && !a.solidangle && !a.polarization && !a.mask;
    const bool is32 = a.dtype == AI_F32 || a.dtype == AI_I32 || a.dtype == AI_U32;
    p.use_tma = plain && is32 && vec_ok && (reinterpret_cast<uintptr_t>(a.image) % 16) == 0 && !ctx->no_tma;
    CUtensorMap map{};
    if (p.use_tma) {
        int rc = ai_make_frame_map(ctx, a, tl.tile_h, &map);
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
