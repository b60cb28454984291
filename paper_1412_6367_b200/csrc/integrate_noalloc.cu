// ai_integrate1d_noalloc: one frame through the tiled matrix without a single device allocation.
//
// Who needs this.  Every other integrate entry of the library may grow a library-owned buffer on the call that first
// needs it (partial sums sized by the batch, the corrected copy of a frame, the padded table, the frame-lane layout),
// i.e. it may call cudaMalloc -- and cudaFree, which waits for the whole device -- in the middle of the acquisition.
// Some programs cannot live with that:
//   - a process in which another component has taken all of the device memory for its own pool (a deep-learning
//     framework's caching allocator, a fixed per-tenant budget on a shared GPU): the library's cudaMalloc simply fails
//     there, although the caller could have handed out memory of its own;
//   - a real-time loop behind a detector that must never stall: an allocation takes the driver's lock and a free
//     synchronises every stream of the device, also the ones that belong to somebody else;
//   - code that has promised its own caller "no allocation after start-up" and is audited for it.
// For them the partial sums -- the only scratch memory the two-kernel tiled path needs beyond the matrix, which
// ai_build_csr made at start-up -- live in a fixed array that is part of the library image itself: 8 MiB
// (AI_NOALLOC_SCRATCH_BYTES) of global memory that every GPU holds from the moment it loads the library until the
// process exits, whether the entry is used or not.  The caller passes the frame, the correction arrays and the outputs
// as usual.  A matrix whose partial sums do not fit is refused (AI_EUNSUPPORTED) and nothing is launched.
//
// The kernels are variants of the block-per-tile pair of integrate_tiled.cu (the AI_LAYOUT_TILED_DIRECT path): stage 1
// reads a tile of the frame once, casts and corrects it, multiplies it with the tile's slice of the
// matrix with compensated sums and leaves one 16-byte record per (tile, bin) segment; stage 2 adds a
// bin's records in a fixed order and writes the weighted histogram, the unweighted one and their ratio
// (PAPER.md:252-254).  Same arithmetic in the same order as that path: the profiles are bit-identical to it.
//
// The array's name is only meaningful to device code.  On the host it is a stand-in object of the same name; its host
// address means nothing to a kernel (a fault, or -- where the GPU can reach host memory -- silent use of the wrong
// memory).  The host therefore asks the runtime once per device, with that device current, for the device address
// (cudaGetSymbolAddress) and hands THAT to the memset and the kernels.
#include <mutex>

#include "tiled_common.cuh"

namespace {

constexpr size_t kScratchBytes = AI_NOALLOC_SCRATCH_BYTES;
static_assert(kScratchBytes % 256 == 0, "whole 256-byte lines");

// the partial records of the call in flight: [nslot] x 16 bytes.  One per device that has loaded the library.
static __device__ __align__(256) unsigned char g_noalloc_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_addr_lock;
void *g_scratch_addr[kMaxDevices] = {nullptr};   // device address of g_noalloc_scratch on device d, NULL = not asked yet

// Set-up of a device, done by the first call made with that device current: the runtime loads the library's device code
// onto the device if it has not yet (this is when the array comes into being there) and reports where the array lives.
// Not an allocation the entry point makes call by call, but it is driver work of the kind a stream capture forbids:
// make the first call on a device outside any capture.
int scratch_address(ai_ctx *ctx, int device, void **out)
{
    if (device < 0 || device >= kMaxDevices) return ai_fail(ctx, AI_EUNSUPPORTED, "device ordinal %d beyond %d", device, kMaxDevices - 1);
    std::lock_guard<std::mutex> hold(g_addr_lock);
    if (!g_scratch_addr[device]) {
        void *p = nullptr;
        AI_CUDA(ctx, cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) % 256) != 0)
            return ai_fail(ctx, AI_ECUDA, "cudaGetSymbolAddress returned an unusable address %p", p);
        g_scratch_addr[device] = p;
    }
    *out = g_scratch_addr[device];
    return AI_OK;
}

struct NaView {
    const int *tile_seg_ptr;     // [ntiles + 1] segments of tile t
    const int4 *seg_meta;        // {first entry, padded end, partial slot, float bits of the coefficient sum}
    const float *tcoef;          // coefficient
    const uint16_t *tidx;        // byte offset of the pixel inside the staged tile
    int tiles_x, tile_h;
};

constexpr int kNaThreads = 128;
constexpr int kNaGroups = kNaThreads / kLanes;

// the segments of one tile: a group of kLanes lanes per segment, four entries per lane and step, the loads of the next
// step in flight while this one is consumed; one record per segment
template <int ACC, bool TRACK>
__device__ __forceinline__ void na_segments(const NaView &v, const float *tile, int s_begin, int s_end, void *records)
{
    const int group = threadIdx.x / kLanes, gl = threadIdx.x % kLanes;
    for (int s0 = s_begin; s0 < s_end; s0 += kNaGroups) {      // block-uniform trip count: shuffles inside
        const int s = s0 + group;
        const bool live = s < s_end;
        const int4 m = live ? __ldg(v.seg_meta + s) : make_int4(0, 0, 0, 0);
        AccumQ<ACC> S4, C4;
        const int end = m.y;
        int k = m.x + gl * 4;
        float4 ca = make_float4(0, 0, 0, 0), cb = ca;
        ushort4 ia = make_ushort4(0, 0, 0, 0), ib = ia;
        if (k < end) {
            ca = __ldg(reinterpret_cast<const float4 *>(v.tcoef + k));
            ia = __ldg(reinterpret_cast<const ushort4 *>(v.tidx + k));
        }
        while (k < end) {
            const int k2 = k + kStep;
            if (k2 < end) {
                cb = __ldg(reinterpret_cast<const float4 *>(v.tcoef + k2));
                ib = __ldg(reinterpret_cast<const ushort4 *>(v.tidx + k2));
            }
            consume4<ACC, TRACK>(tile, ca, ia, S4, C4);
            ca = cb;
            ia = ib;
            k = k2;
        }
        Accum<ACC> S = S4.total(), C = C4.total();
        group_reduce<ACC>(S);
        if constexpr (TRACK) group_reduce<ACC>(C);
        if (gl == 0 && live && m.y > m.x) store_partial<ACC>(records, m.z, S, C, TRACK, (double)__int_as_float(m.w));
    }
}

template <int DT, int ACC>
__global__ void __launch_bounds__(kNaThreads, 12) noalloc_stage1_kernel(NaView v, const void *image, Corrections cor,
                                                                         int height, int width, int vec_ok,
                                                                         void *records)
{
    __shared__ __align__(16) float tile[kTilePixMax];
    const int t = blockIdx.x;
    const int ty = t / v.tiles_x, tx = t - ty * v.tiles_x;
    const bool bad = stage_tile<DT, kNaThreads, 8, 2>(tile, image, cor, ty, tx, v.tile_h, height, width, vec_ok,
                                                      threadIdx.x, [] {});
    // an invalid pixel somewhere in the tile: count is summed as well; else it is the stored sum of the coefficients
    const bool track = __syncthreads_or(bad) != 0;
    const int s_begin = __ldg(v.tile_seg_ptr + t), s_end = __ldg(v.tile_seg_ptr + t + 1);
    if (track) na_segments<ACC, true>(v, tile, s_begin, s_end, records);
    else na_segments<ACC, false>(v, tile, s_begin, s_end, records);
}

// one warp per bin: the bin's records in slot order, then the three outputs and the bin centre
template <int ACC>
__global__ void __launch_bounds__(256) noalloc_stage2_kernel(const int *__restrict__ bin_slot_ptr, int npt,
                                                             const void *records, const double *__restrict__ range,
                                                             float empty, float *__restrict__ radial,
                                                             float *__restrict__ intensity,
                                                             float *__restrict__ sum_signal, float *__restrict__ count)
{
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (b >= npt) return;
    if (lane == 0 && radial) {
        const double u0 = range[0], delta = (range[1] - range[0]) / (double)npt;
        radial[b] = (float)(u0 + ((double)b + 0.5) * delta);
    }
    finish_bin<ACC>(records, __ldg(bin_slot_ptr + b), __ldg(bin_slot_ptr + b + 1), lane, empty, intensity + b,
                    sum_signal + b, count + b);
}

template <int DT, int ACC>
int na_launch(ai_ctx *ctx, const NaView &v, const FrameArgs &a, int vec_ok, void *records, cudaStream_t st)
{
    const Corrections cor{a.dark, a.flat, a.solidangle, a.polarization, a.mask};
    noalloc_stage1_kernel<DT, ACC><<<ctx->tl.ntiles, kNaThreads, 0, st>>>(v, a.image, cor, ctx->height, ctx->width,
                                                                        vec_ok, records);
    AI_CUDA(ctx, cudaGetLastError());
    noalloc_stage2_kernel<ACC><<<(ctx->npt + 7) / 8, 256, 0, st>>>(ctx->tl.bin_slot_ptr, ctx->npt, records, ctx->d_range,
                                                                 ctx->empty_value, a.radial, a.intensity, a.sum_signal,
                                                                 a.count);
    AI_CUDA(ctx, cudaGetLastError());
    return AI_OK;
}

template <int DT>
int na_launch_dt(ai_ctx *ctx, const NaView &v, const FrameArgs &a, int vec_ok, void *records, cudaStream_t st)
{
    switch (ctx->accum) {
    case AI_ACC_F32_KAHAN: return na_launch<DT, AI_ACC_F32_KAHAN>(ctx, v, a, vec_ok, records, st);
    case AI_ACC_F32_PLAIN: return na_launch<DT, AI_ACC_F32_PLAIN>(ctx, v, a, vec_ok, records, st);
    default: return na_launch<DT, AI_ACC_F64>(ctx, v, a, vec_ok, records, st);
    }
}

bool on_boundary(const void *p, size_t a) { return p == nullptr || (reinterpret_cast<uintptr_t>(p) % a) == 0; }

}  // namespace

extern "C" int ai_integrate1d_noalloc(ai_ctx *ctx, const void *image, ai_dtype dtype, const float *dark,
                                      const float *flat, const float *solidangle, const float *polarization,
                                      const uint8_t *mask, float *radial, float *intensity, float *sum_signal,
                                      float *count, void *cuda_stream)
{
    if (!ctx) return AI_EINVAL;
    if (!ctx->built) return ai_fail(ctx, AI_ENOTBUILT, "ai_build_csr has not been called");
    if (ctx->npt_azim > 0) return ai_fail(ctx, AI_EUNSUPPORTED, "ai_integrate1d_noalloc: 1D contexts only");
    if (ctx->norm != AI_NORM_PIXEL) return ai_fail(ctx, AI_EUNSUPPORTED, "ai_integrate1d_noalloc: AI_NORM_PIXEL only");
    if (ctx->held.on && !dark && !flat && !solidangle && !polarization && !mask)
        return ai_fail(ctx, AI_EUNSUPPORTED, "ai_integrate1d_noalloc does not apply held corrections: pass the arrays");
    if (!image || !intensity || !sum_signal || !count) return ai_fail(ctx, AI_EINVAL, "NULL image or output");
    if ((int)dtype < AI_F32 || (int)dtype > AI_U32) return ai_fail(ctx, AI_EINVAL, "bad dtype %d", (int)dtype);
    const TiledLayout &tl = ctx->tl;
    if (!tl.tile_seg_ptr || !tl.seg_meta || !tl.tcoef || !tl.tidx || !tl.bin_slot_ptr || tl.ntiles < 1)
        return ai_fail(ctx, AI_EUNSUPPORTED, "ai_integrate1d_noalloc: this context has no tiled matrix");
    // the size check comes first: a matrix that does not fit is refused before anything touches the device
    const size_t need = (size_t)(tl.nslot > 0 ? tl.nslot : 0) * 16;
    if (need > kScratchBytes)
        return ai_fail(ctx, AI_EUNSUPPORTED,
                       "ai_integrate1d_noalloc: this matrix needs %zu bytes of partial sums (%d records of 16 bytes), the "
                       "library's fixed scratch array holds %zu (AI_NOALLOC_SCRATCH_BYTES); use ai_integrate1d",
                       need, tl.nslot, kScratchBytes);
    int dev = -1;
    AI_CUDA(ctx, cudaGetDevice(&dev));
    if (dev != ctx->device)
        return ai_fail(ctx, AI_EINVAL, "the matrix was built on device %d, the current device is %d", ctx->device, dev);
    void *records = nullptr;
    int rc = scratch_address(ctx, dev, &records);
    if (rc != AI_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // The array still holds the records of whatever call used it last (any context, any stream).  Stage 1 writes one
    // record per segment, into the first of the slots its bin reserves for the segment; the others are summed by
    // stage 2 too and must read as zero.
    if (need) AI_CUDA(ctx, cudaMemsetAsync(records, 0, need, st));
    const size_t esz = (dtype == AI_U16 || dtype == AI_I16) ? 2 : 4;
    const int vec_ok = ctx->width % 4 == 0 && on_boundary(image, 4 * esz) && on_boundary(dark, 16) &&
                       on_boundary(flat, 16) && on_boundary(solidangle, 16) && on_boundary(polarization, 16) &&
                       on_boundary(mask, 4);
    const NaView v{tl.tile_seg_ptr, tl.seg_meta, tl.tcoef, tl.tidx, tl.tiles_x, tl.tile_h};
    const FrameArgs a{image, dtype, dark, flat, solidangle, polarization, mask, radial, intensity, sum_signal, count, 1,
                      (int64_t)ctx->height * ctx->width};
    switch (dtype) {
    case AI_F32: rc = na_launch_dt<AI_F32>(ctx, v, a, vec_ok, records, st); break;
    case AI_I32: rc = na_launch_dt<AI_I32>(ctx, v, a, vec_ok, records, st); break;
    case AI_U16: rc = na_launch_dt<AI_U16>(ctx, v, a, vec_ok, records, st); break;
    case AI_I16: rc = na_launch_dt<AI_I16>(ctx, v, a, vec_ok, records, st); break;
    case AI_U32: rc = na_launch_dt<AI_U32>(ctx, v, a, vec_ok, records, st); break;
    }
    if (rc == AI_OK) ctx->last_launches = 2;
    return rc;
}
