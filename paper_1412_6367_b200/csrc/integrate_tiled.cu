// Per-frame hot path, TILED layout.  Two launches per call:
//
//   stage 1  the SpMV proper.  Two kernels compute the same partials:
//              - integrate_pipe.cu: persistent, warp-specialised, bulk-copy pipelined (used whenever a tile's slice of
//                the matrix fits the shared-memory ring);
//              - the one here: one thread block per (image tile, frame), matrix streamed with plain 128-bit loads.
//            In both, the tile is read once, fully coalesced, cast and corrected in registers (cast, dark,
//            flat, solid angle, polarisation "in a single pass over each pixel"; mask folded in as NaN) and parked in
//            shared memory; a group of kLanes lanes owns one (tile, bin) segment: per-lane compensated accumulation
//            (PAPER.md:186-188), shuffle merge inside the group, one partial (sum_signal, count) per segment written to
//            a bin-major buffer.
//   stage 2  one warp per (bin, frame): adds the bin's partials in a fixed order and writes the three outputs
//            (ratio, unweighted histogram, weighted histogram).  No atomics anywhere, so results are
//            bit-reproducible; every bin is written exactly once, so the paper's memset disappears.
#include "pipe_common.cuh"
#include "tiled_common.cuh"

int ai_launch_pipe_stage1(ai_ctx *ctx, const FrameArgs &a, int vec_ok, cudaStream_t st, bool *handled);
int ai_launch_stream_stage1(ai_ctx *ctx, const FrameArgs &a, int vec_ok, int track_all, int image_dep, cudaStream_t st,
                            bool *handled, const void **partials_used);
int ai_launch_bstream_stage1(ai_ctx *ctx, const FrameArgs &a, int vec_ok, cudaStream_t st, bool *handled);

namespace {

struct TiledView {
    const int *tile_seg_ptr;
    const int4 *seg_meta;
    const float *tcoef;
    const uint16_t *tidx;
    int tiles_x, tile_h, nslot;
};

constexpr int kS1Threads = 128;                       // 12 blocks per SM: one wave holds 1776 tiles
constexpr int kS1MinBlocks = 12;
constexpr int kGroups = kS1Threads / kLanes;          // segments in flight per block

// the segments of one tile: groups of kLanes lanes take segments round-robin; two loads kept in flight per lane
template <int ACC, bool TRACK>
__device__ __forceinline__ void process_segments(const TiledView &tv, const float *tile, int s_begin, int s_end,
                                                 void *part_f)
{
    const int group = threadIdx.x / kLanes, gl = threadIdx.x % kLanes;
    int s = s_begin + group;
    int4 m = s < s_end ? __ldg(tv.seg_meta + s) : make_int4(0, 0, 0, 0);
    // whole warps iterate together (shuffles inside): loop while any group of the warp still has a segment
    while (__any_sync(AI_FULL_MASK, s < s_end)) {
        const int s_next = s + kGroups;
        const int4 m_next = s_next < s_end ? __ldg(tv.seg_meta + s_next) : make_int4(0, 0, 0, 0);
        AccumQ<ACC> S2, C2;
        const int end = m.y;
        int k = m.x + gl * 4;
        // software pipeline: loads for step i+1 are issued before step i is consumed
        float4 ca = make_float4(0, 0, 0, 0), cb = ca;
        ushort4 ia = make_ushort4(0, 0, 0, 0), ib = ia;
        if (k < end) {
            ca = __ldg(reinterpret_cast<const float4 *>(tv.tcoef + k));
            ia = __ldg(reinterpret_cast<const ushort4 *>(tv.tidx + k));
        }
        while (k < end) {
            const int k2 = k + kStep;
            if (k2 < end) {
                cb = __ldg(reinterpret_cast<const float4 *>(tv.tcoef + k2));
                ib = __ldg(reinterpret_cast<const ushort4 *>(tv.tidx + k2));
            }
            consume4<ACC, TRACK>(tile, ca, ia, S2, C2);
            ca = cb;
            ia = ib;
            k = k2;
        }
        Accum<ACC> S = S2.total(), C = C2.total();
        group_reduce<ACC>(S);
        if constexpr (TRACK) group_reduce<ACC>(C);
        if (gl == 0 && s < s_end && m.y > m.x) store_partial<ACC>(part_f, m.z, S, C, TRACK, (double)__int_as_float(m.w));
        s = s_next;
        m = m_next;
    }
}

template <int DT, int ACC>
__global__ void __launch_bounds__(kS1Threads, kS1MinBlocks) tiled_stage1_kernel(TiledView tv, const void *frames,
                                                                                int64_t frame_stride, Corrections cor,
                                                                                int height, int width, int vec_ok,
                                                                                void *partials)
{
    __shared__ __align__(16) float tile[kTilePixMax];     // ai_tile_pos needs no particular alignment beyond 16 bytes here
    using T = typename RawType<DT>::T;
    const int t = blockIdx.x, f = blockIdx.y;
    const int ty = t / tv.tiles_x, tx = t - ty * tv.tiles_x;
    const void *img = reinterpret_cast<const T *>(frames) + (int64_t)f * frame_stride;
    const bool bad = stage_tile<DT, kS1Threads, 8, 2>(tile, img, cor, ty, tx, tv.tile_h, height, width, vec_ok, threadIdx.x,
                                                [] {});
    // some pixel of the tile is invalid -> count must be accumulated too; else it is the static coefficient sum
    const bool track = __syncthreads_or(bad) != 0;
    void *part_f = reinterpret_cast<char *>(partials) + (int64_t)f * tv.nslot * 16;
    const int s_begin = __ldg(tv.tile_seg_ptr + t), s_end = __ldg(tv.tile_seg_ptr + t + 1);
    if (track) process_segments<ACC, true>(tv, tile, s_begin, s_end, part_f);
    else process_segments<ACC, false>(tv, tile, s_begin, s_end, part_f);
}

// ---- H5: fixed-order sum of each bin's partials, ratio, three outputs --------------------------------------------------
// Launched with programmatic stream serialisation (launch_stage2): the blocks may become resident while stage 1 is
// still running; everything that does not depend on stage 1 (the slot range of the bin, the radial axis) is done
// before griddepcontrol.wait, which returns once stage 1 has completed and its partials are visible.
template <int ACC>
__global__ void __launch_bounds__(256) tiled_stage2_kernel(const int *__restrict__ bin_slot_ptr, int nslot, int npt,
                                                           const void *partials,
                                                           const double *__restrict__ range, float empty,
                                                           float *__restrict__ radial, float *__restrict__ intensity,
                                                           float *__restrict__ sum_signal, float *__restrict__ count)
{
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int f = blockIdx.y, lane = threadIdx.x & 31;
    int beg = 0, end = 0;
    if (b < npt) {
        beg = __ldg(bin_slot_ptr + b);
        end = __ldg(bin_slot_ptr + b + 1);
        if (lane == 0 && radial && f == 0) {
            double u0 = range[0], delta = (range[1] - range[0]) / (double)npt;
            radial[b] = (float)(u0 + ((double)b + 0.5) * delta);
        }
    }
    // the next stage 1 of the stream (integrate_stream.cu) may start its prologue now; it touches the partials only
    // after its own griddepcontrol.wait, i.e. after this grid has completed
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (b >= npt) return;
    const int64_t o = (int64_t)f * npt + b;
    finish_bin<ACC>(reinterpret_cast<const char *>(partials) + (int64_t)f * nslot * 16, beg, end, lane, empty,
                    intensity + o, sum_signal + o, count + o);
}

// H5 of the single-frame kernel (integrate_stream.cu): the same sums in the same order, shaped for the launch chain --
// at most one small block per SM (4 warps, registers capped so that it fits beside a block of the stream kernel), every
// warp taking bins in a grid-wide stride.  All its blocks become resident and let their dependents go while the stream
// kernel before them is still running; they wait for it, add up, and leave.
constexpr int kFinishThreads = 128;
template <int ACC>
__global__ void __launch_bounds__(kFinishThreads, 10) tiled_finish_kernel(const int *__restrict__ bin_slot_ptr, int npt,
                                                                           int serial, const void *partials,
                                                                           const double *__restrict__ range, float empty,
                                                                           float *__restrict__ radial,
                                                                           float *__restrict__ intensity,
                                                                           float *__restrict__ sum_signal,
                                                                           float *__restrict__ count,
                                                                           unsigned long long *chain_done)
{
    // every block counts itself out (release) when it has read its partials: what the kernels that reuse them check
    struct Done {
        unsigned long long *c;
        __device__ ~Done()
        {
            __syncthreads();
            if (threadIdx.x == 0) asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(c), "l"(1ULL) : "memory");
        }
    } done{chain_done};
    const int lane = threadIdx.x & 31, nw = gridDim.x * (kFinishThreads / 32);
    int b = blockIdx.x * (kFinishThreads / 32) + (threadIdx.x >> 5);
    int beg = 0, end = 0;
    if (b < npt) {
        beg = __ldg(bin_slot_ptr + b);
        end = __ldg(bin_slot_ptr + b + 1);
    }
    const double u0 = radial ? range[0] : 0.0, delta = radial ? (range[1] - range[0]) / (double)npt : 0.0;
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (serial) {
        // many bins of a few partials each (bidimensional integration): one thread per bin
        for (int t = blockIdx.x * kFinishThreads + threadIdx.x; t < npt; t += gridDim.x * kFinishThreads) {
            finish_bin_serial<ACC>(partials, __ldg(bin_slot_ptr + t), __ldg(bin_slot_ptr + t + 1), empty, intensity + t,
                                   sum_signal + t, count + t);
            if (radial) radial[t] = (float)(u0 + ((double)t + 0.5) * delta);
        }
        return;
    }
    while (b < npt) {
        const int bn = b + nw;
        int nbeg = 0, nend = 0;
        if (bn < npt) {
            nbeg = __ldg(bin_slot_ptr + bn);
            nend = __ldg(bin_slot_ptr + bn + 1);
        }
        finish_bin<ACC>(partials, beg, end, lane, empty, intensity + b, sum_signal + b, count + b);
        if (lane == 0 && radial) radial[b] = (float)(u0 + ((double)b + 0.5) * delta);
        b = bn; beg = nbeg; end = nend;
    }
}

template <int DT, int ACC>
int launch_simple(ai_ctx *ctx, const FrameArgs &a, int vec_ok, cudaStream_t st)
{
    const TiledLayout &tl = ctx->tl;
    TiledView tv{tl.tile_seg_ptr, tl.seg_meta, tl.tcoef, tl.tidx, tl.tiles_x, tl.tile_h, tl.nslot};
    Corrections cor{a.dark, a.flat, a.solidangle, a.polarization, a.mask};
    dim3 g1(tl.ntiles, a.nframes);
    ai_prof_begin(ctx, st);
    tiled_stage1_kernel<DT, ACC><<<g1, kS1Threads, 0, st>>>(tv, a.image, a.frame_stride, cor, ctx->height, ctx->width,
                                                           vec_ok, ctx->partials);
    ai_prof_end(ctx, st);
    return AI_OK;
}

template <int DT>
int launch_simple_dt(ai_ctx *ctx, const FrameArgs &a, int vec_ok, cudaStream_t st)
{
    switch (ctx->accum) {
    case AI_ACC_F32_KAHAN: return launch_simple<DT, AI_ACC_F32_KAHAN>(ctx, a, vec_ok, st);
    case AI_ACC_F32_PLAIN: return launch_simple<DT, AI_ACC_F32_PLAIN>(ctx, a, vec_ok, st);
    default: return launch_simple<DT, AI_ACC_F64>(ctx, a, vec_ok, st);
    }
}

int launch_simple_any(ai_ctx *ctx, const FrameArgs &a, int vec_ok, cudaStream_t st)
{
    switch (a.dtype) {
    case AI_F32: return launch_simple_dt<AI_F32>(ctx, a, vec_ok, st);
    case AI_I32: return launch_simple_dt<AI_I32>(ctx, a, vec_ok, st);
    case AI_U16: return launch_simple_dt<AI_U16>(ctx, a, vec_ok, st);
    case AI_I16: return launch_simple_dt<AI_I16>(ctx, a, vec_ok, st);
    case AI_U32: return launch_simple_dt<AI_U32>(ctx, a, vec_ok, st);
    }
    return ai_fail(ctx, AI_EINVAL, "unknown dtype %d", (int)a.dtype);
}

int launch_stage2(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    const TiledLayout &tl = ctx->tl;
    // programmatic dependent launch: the launch latency of stage 2 overlaps the tail of stage 1
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((ctx->npt + 7) / 8, a.nframes);
    cfg.blockDim = dim3(256);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
#define AI_S2(ACC)                                                                                                  \
    AI_CUDA(ctx, cudaLaunchKernelEx(&cfg, tiled_stage2_kernel<ACC>, (const int *)tl.bin_slot_ptr, tl.nslot, ctx->npt, \
                                    (const void *)ctx->partials, (const double *)ctx->d_range, ctx->empty_value,    \
                                    a.radial, a.intensity, a.sum_signal, a.count))
    switch (ctx->accum) {
    case AI_ACC_F32_KAHAN: AI_S2(AI_ACC_F32_KAHAN); break;
    case AI_ACC_F32_PLAIN: AI_S2(AI_ACC_F32_PLAIN); break;
    default: AI_S2(AI_ACC_F64); break;
    }
#undef AI_S2
    return AI_OK;
}

int launch_finish(ai_ctx *ctx, const FrameArgs &a, const void *partials, cudaStream_t st)
{
    const TiledLayout &tl = ctx->tl;
    const int sms = ctx->sm_count > 0 ? ctx->sm_count : 148;
    const int wpb = kFinishThreads / 32;
    const int serial = (long long)tl.nslot < 8LL * ctx->npt;      // few partials per bin: one thread per bin
    // up to fin_blocks_per_sm small blocks per SM (they fit beside a block of the stream kernel): the kernel is a chain of
    // memory latencies per bin, so fewer bins per warp end it sooner -- and the stream kernel of the NEXT call cannot
    // leave before this one has ended
    const int per_sm = ctx->tune.fin_blocks_per_sm > 0 ? ctx->tune.fin_blocks_per_sm : 3;
    int grid = serial ? (ctx->npt + kFinishThreads - 1) / kFinishThreads : (ctx->npt + wpb - 1) / wpb;
    if (grid > per_sm * sms) grid = per_sm * sms;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kFinishThreads);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
#define AI_FIN(ACC)                                                                                                   \
    AI_CUDA(ctx, cudaLaunchKernelEx(&cfg, tiled_finish_kernel<ACC>, (const int *)tl.bin_slot_ptr, ctx->npt, serial, partials,  \
                                    (const double *)ctx->d_range, ctx->empty_value, a.radial, a.intensity,           \
                                    a.sum_signal, a.count, ctx->chain_done))
    switch (ctx->accum) {
    case AI_ACC_F32_KAHAN: AI_FIN(AI_ACC_F32_KAHAN); break;
    case AI_ACC_F32_PLAIN: AI_FIN(AI_ACC_F32_PLAIN); break;
    default: AI_FIN(AI_ACC_F64); break;
    }
#undef AI_FIN
    ctx->fin_cum_prev = ctx->fin_cum;
    ctx->fin_cum += (unsigned long long)grid;
    return AI_OK;
}

bool aligned(const void *p, size_t a) { return p == nullptr || (reinterpret_cast<uintptr_t>(p) % a) == 0; }

}  // namespace

// pre-pass (cast + corrections, mode as correct_value) -> stream kernel -> finish kernel, for one frame
static int launch_prepass_stream(ai_ctx *ctx, const FrameArgs &a, int vec_ok, int mode, cudaStream_t st, bool *handled)
{
    float *corrected = nullptr;
    int rc = ai_launch_correct(ctx, a, vec_ok, ai_stream_full_grid(ctx) && !ctx->tune.no_overlap, mode, st, &corrected);
    if (rc != AI_OK) return rc;
    FrameArgs b = a;
    b.image = corrected;
    b.dtype = AI_F32;
    b.row_pitch = (ctx->width + 3) / 4 * 4;
    b.frame_stride = (int64_t)ctx->height * b.row_pitch;
    b.dark = b.flat = b.solidangle = b.polarization = nullptr;
    b.mask = nullptr;
    b.held = false;              // (a held set reached this pass as a dark current and a denominator)
    const int may_be_invalid = a.dark || a.flat || a.solidangle || a.polarization || a.mask || a.dtype == AI_F32;
    const void *used = nullptr;
    rc = ai_launch_stream_stage1(ctx, b, 1, may_be_invalid, 1, st, handled, &used);
    if (rc != AI_OK || !*handled) return rc;
    ctx->last_launches = 2;
    if (ctx->stage1_only) return AI_OK;
    ctx->last_launches = 3;
    return launch_finish(ctx, a, used, st);
}

__global__ void __launch_bounds__(256) ratio_kernel(int npt, float empty, const float *__restrict__ num,
                                                    const float *__restrict__ den, float *__restrict__ out)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < npt) out[b] = den[b] != 0.0f ? __fdiv_rn(num[b], den[b]) : empty;
}

// AI_NORM_SPLIT (ai_set_normalization): sum c (I - dark) and sum c (flat * solidangle * polarization) as two passes of
// the same engine over the numerator and the denominator frame, then their ratio.  One frame, TILED layout.
int ai_launch_tiled_split(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    if (a.nframes != 1 || ctx->npt_azim > 0) return ai_fail(ctx, AI_EUNSUPPORTED, "split normalisation: one 1D frame per call");
    if (ctx->no_prepass || ctx->no_stream || ctx->no_tma || ai_stream_stages(ctx) < 2)
        return ai_fail(ctx, AI_EUNSUPPORTED, "split normalisation needs the pre-pass + single-frame kernel path");
    if (!ctx->norm_scratch) AI_CUDA(ctx, cudaMalloc(&ctx->norm_scratch, 2 * (size_t)ctx->npt * sizeof(float)));
    const size_t esz = (a.dtype == AI_U16 || a.dtype == AI_I16) ? 2 : 4;
    const int vec_ok = ctx->width % 4 == 0 && a.frame_stride % 4 == 0 && aligned(a.image, 4 * esz) &&
                       aligned(a.dark, 16) && aligned(a.flat, 16) && aligned(a.solidangle, 16) &&
                       aligned(a.polarization, 16) && aligned(a.mask, 4);
    bool handled = false;
    FrameArgs n = a;                                   // numerator: sum_signal <- sum c (I - dark)
    n.intensity = ctx->norm_scratch;
    n.count = ctx->norm_scratch + ctx->npt;
    int rc = launch_prepass_stream(ctx, n, vec_ok, 1, st, &handled);
    if (rc != AI_OK) return rc;
    if (!handled) return ai_fail(ctx, AI_EUNSUPPORTED, "split normalisation: the single-frame kernel does not apply");
    FrameArgs d = a;                                   // denominator: count <- sum c (flat * solidangle * polarization)
    d.radial = nullptr;
    d.intensity = ctx->norm_scratch;
    d.sum_signal = a.count;
    d.count = ctx->norm_scratch + ctx->npt;
    rc = launch_prepass_stream(ctx, d, vec_ok, 2, st, &handled);
    if (rc != AI_OK) return rc;
    ratio_kernel<<<(ctx->npt + 255) / 256, 256, 0, st>>>(ctx->npt, ctx->empty_value, a.sum_signal, a.count, a.intensity);
    AI_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = 7;
    return AI_OK;
}

int ai_launch_tiled(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    const TiledLayout &tl = ctx->tl;
    const size_t need = (size_t)(tl.nslot > 0 ? tl.nslot : 1) * 16 * a.nframes;
    // partial records of the two-launch paths (the single-frame kernel has its own, sized at build time): grown on
    // demand; cudaFree synchronises the device, so work in flight on the old buffer has finished.  A first call with
    // the largest batch sizes it for good.
    auto ensure_partials = [&]() -> int {
        if (ctx->partials_bytes >= need) return AI_OK;
        if (ctx->partials) AI_CUDA(ctx, cudaFree(ctx->partials));
        ctx->partials = nullptr;
        ctx->partials_bytes = 0;
        AI_CUDA(ctx, cudaMalloc(&ctx->partials, need));
        ctx->partials_bytes = need;
        return AI_OK;
    };
    const size_t esz = (a.dtype == AI_U16 || a.dtype == AI_I16) ? 2 : 4;
    // 128-bit path: rows of 4 pixels never straddle the image edge and every array is aligned for 4-pixel vectors
    const int vec_ok = ctx->width % 4 == 0 && a.frame_stride % 4 == 0 && aligned(a.image, 4 * esz) &&
                       aligned(a.dark, 16) && aligned(a.flat, 16) && aligned(a.solidangle, 16) &&
                       aligned(a.polarization, 16) && aligned(a.mask, 4);
    bool handled = false;
    int rc = AI_OK;
    if (ctx->layout != AI_LAYOUT_TILED_DIRECT) {
        const void *used = nullptr;
        rc = ai_launch_stream_stage1(ctx, a, vec_ok, 0, 0, st, &handled, &used);     // one plain 32-bit frame
        if (rc != AI_OK) return rc;
        if (handled) {
            ctx->last_launches = 1;
            if (ctx->stage1_only) return AI_OK;
            ctx->last_launches = 2;
            return launch_finish(ctx, a, used, st);
        }
        // one frame with correction arrays, a mask, 16-bit pixels, unaligned buffers or rows that do not start on
        // 16-byte boundaries (width not a multiple of 4): H1 + H2 as a streaming pre-pass into a float32 frame with
        // padded rows (invalid pixels as NaN), then the same single-frame kernel
        if (a.nframes == 1 && !ctx->no_prepass && !ctx->no_stream && !ctx->no_tma && ai_stream_stages(ctx) >= 2) {
            rc = launch_prepass_stream(ctx, a, vec_ok, 0, st, &handled);
            if (rc != AI_OK || handled) return rc;
        }
        // batches of 32-bit frames: the frame-lane kernel (integrate_fl.cu) takes the groups of 64 frames it is faster on,
        // the frames behind them continue below
        int taken = 0;
        rc = ai_launch_fl(ctx, a, vec_ok, st, &taken);
        if (rc != AI_OK || taken == a.nframes) return rc;
        if (taken > 0) {
            const int launches = ctx->last_launches;
            FrameArgs rest = a;
            rest.nframes = a.nframes - taken;
            rest.image = static_cast<const char *>(a.image) + (size_t)taken * (size_t)a.frame_stride * esz;
            rest.intensity = a.intensity + (size_t)taken * ctx->npt;
            rest.sum_signal = a.sum_signal + (size_t)taken * ctx->npt;
            rest.count = a.count + (size_t)taken * ctx->npt;
            rc = ai_launch_tiled(ctx, rest, st);
            ctx->last_launches += launches;
            return rc;
        }
        rc = ensure_partials();
        if (rc != AI_OK) return rc;
        rc = ai_launch_bstream_stage1(ctx, a, vec_ok, st, &handled);          // batch of plain 32-bit frames
        // what is left of a batch -- frames with correction arrays, a mask or held corrections, 16-bit frames, buffers off
        // the 16-byte boundaries: frame by frame through the single-frame paths above.  Measured 1.5 to 4 times faster
        // than staging the corrections inside the general batched kernel (us per frame, 8 to 64 frames per call: cfg3 43
        // against 62-69, held 25 against 100; cfg2's matrix with cfg3's arrays 34 against 54-60, held 12.5 against 90;
        // plain uint16 frames 20 against 30-32)
        if (rc == AI_OK && !handled && a.nframes > 1 && !ctx->no_prepass && !ctx->no_stream && !ctx->no_tma &&
            ai_stream_stages(ctx) >= 2) {
            int launches = 0;
            for (int f = 0; f < a.nframes; ++f) {
                FrameArgs one = a;
                one.nframes = 1;
                one.image = static_cast<const char *>(a.image) + (size_t)f * (size_t)a.frame_stride * esz;
                one.radial = nullptr;
                one.intensity = a.intensity + (size_t)f * ctx->npt;
                one.sum_signal = a.sum_signal + (size_t)f * ctx->npt;
                one.count = a.count + (size_t)f * ctx->npt;
                rc = ai_launch_tiled(ctx, one, st);
                if (rc != AI_OK) return rc;
                launches += ctx->last_launches;
            }
            ctx->last_launches = launches;
            return AI_OK;
        }
        if (rc == AI_OK && !handled) rc = ai_launch_pipe_stage1(ctx, a, vec_ok, st, &handled);
    }
    if (rc != AI_OK) return rc;
    if (!handled) {
        rc = ensure_partials();
        if (rc != AI_OK) return rc;
        // this kernel writes one partial per segment, into the first of the segment's slots (one per run of the
        // sliced layout): the others must read as zero
        AI_CUDA(ctx, cudaMemsetAsync(ctx->partials, 0, need, st));
        rc = launch_simple_any(ctx, a, vec_ok, st);
        if (rc != AI_OK) return rc;
    }
    if (ctx->stage1_only) {
        ctx->last_launches = 1;
        return AI_OK;
    }
    rc = launch_stage2(ctx, a, st);
    ctx->last_launches = 2;
    return rc;
}
