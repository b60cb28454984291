// Per-frame hot path, TILED layout.  Two launches per call:
//
//   stage 1  one thread block per (image tile, frame): the tile is read once, fully coalesced, cast and corrected in
//            registers (cast, dark, flat, solid angle, polarisation "in a single pass over each pixel";
//            mask folded in as NaN) and parked in shared memory; the block then streams the tile's slice of the matrix
//            (coefficient fp32 + 16-bit pixel offset, 128-bit / 64-bit coalesced loads) and gathers from shared memory.
//            One warp per (tile, bin) segment, per-lane compensated accumulation, warp-shuffle merge,
//            one partial (sum_signal, count) per segment written to a bin-major buffer.
//   stage 2  one warp per (bin, frame): adds the bin's partials in a fixed order and writes the three outputs
//            (ratio, unweighted histogram, weighted histogram).  No atomics anywhere, so results are
//            bit-reproducible; every bin is written exactly once, so the paper's memset disappears.
#include "common.cuh"

namespace {

struct TiledView {
    const int *tile_seg_ptr, *seg_ptr, *seg_slot, *bin_slot_ptr;
    const double *seg_csum;
    const float *tcoef;
    const uint16_t *tidx;
    int tiles_x, nslot;
};

constexpr int kS1Threads = 256;
constexpr int kS1Warps = kS1Threads / 32;

template <int ACC>
__device__ __forceinline__ void store_partial(void *partials, int64_t slot, const Accum<ACC> &S, const Accum<ACC> &C,
                                              bool tracked, double csum)
{
    if constexpr (ACC == AI_ACC_F64) {
        reinterpret_cast<double2 *>(partials)[slot] = make_double2(S.s, tracked ? C.s : csum);
    } else if constexpr (ACC == AI_ACC_F32_KAHAN) {
        float c_hi = tracked ? C.s : (float)csum;
        float c_lo = tracked ? -C.c : (float)(csum - (double)c_hi);
        reinterpret_cast<float4 *>(partials)[slot] = make_float4(S.s, -S.c, c_hi, c_lo);
    } else {
        reinterpret_cast<float4 *>(partials)[slot] = make_float4(S.s, 0.0f, tracked ? C.s : (float)csum, 0.0f);
    }
}

template <int DT, int ACC>
__global__ void __launch_bounds__(kS1Threads) tiled_stage1_kernel(TiledView tv, const void *frames,
                                                                  int64_t frame_stride, Corrections cor, int height,
                                                                  int width, int vec_ok, void *partials)
{
    __shared__ __align__(16) float tile[kTilePix];
    using T = typename RawType<DT>::T;
    const int t = blockIdx.x, f = blockIdx.y;
    const int ty = t / tv.tiles_x, tx = t - ty * tv.tiles_x;
    const void *img = reinterpret_cast<const T *>(frames) + (int64_t)f * frame_stride;
    const bool has_den = cor.flat || cor.solidangle || cor.polarization;

    // ---- H1 + H2: load, cast, correct, park in shared memory ----------------------------------------------------------
    bool bad = false;
    if (vec_ok) {
        for (int q = threadIdx.x; q < kTilePix / 4; q += kS1Threads) {
            int ly = q / (kTileW / 4), lx = (q % (kTileW / 4)) * 4;
            int y = ty * kTileH + ly, x = tx * kTileW + lx;
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (y < height && x < width) {
                int64_t p = (int64_t)y * width + x;
                float4 raw = load_raw4<DT>(img, p);
                float4 dk = cor.dark ? __ldg(reinterpret_cast<const float4 *>(cor.dark + p)) : make_float4(0, 0, 0, 0);
                float4 fl = cor.flat ? __ldg(reinterpret_cast<const float4 *>(cor.flat + p)) : make_float4(1, 1, 1, 1);
                float4 sa = cor.solidangle ? __ldg(reinterpret_cast<const float4 *>(cor.solidangle + p))
                                           : make_float4(1, 1, 1, 1);
                float4 po = cor.polarization ? __ldg(reinterpret_cast<const float4 *>(cor.polarization + p))
                                             : make_float4(1, 1, 1, 1);
                uchar4 mk = cor.mask ? __ldg(reinterpret_cast<const uchar4 *>(cor.mask + p)) : make_uchar4(0, 0, 0, 0);
                v.x = correct_value(raw.x, dk.x, fl.x, sa.x, po.x, mk.x != 0, has_den);
                v.y = correct_value(raw.y, dk.y, fl.y, sa.y, po.y, mk.y != 0, has_den);
                v.z = correct_value(raw.z, dk.z, fl.z, sa.z, po.z, mk.z != 0, has_den);
                v.w = correct_value(raw.w, dk.w, fl.w, sa.w, po.w, mk.w != 0, has_den);
                bad = bad || v.x != v.x || v.y != v.y || v.z != v.z || v.w != v.w;
            }
            reinterpret_cast<float4 *>(tile)[q] = v;
        }
    } else {
        for (int k = threadIdx.x; k < kTilePix; k += kS1Threads) {
            int y = ty * kTileH + k / kTileW, x = tx * kTileW + k % kTileW;
            float v = 0.f;
            if (y < height && x < width) {
                v = corrected_pixel<DT>(img, (int64_t)y * width + x, cor);
                bad = bad || v != v;
            }
            tile[k] = v;
        }
    }
    // some pixel of the tile is invalid -> count must be accumulated too; else it is the static coefficient sum
    const bool track = __syncthreads_or(bad) != 0;

    // ---- H4: gather-reduce, one warp per (tile, bin) segment -----------------------------------------------------------
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int s_end = tv.tile_seg_ptr[t + 1];
    void *part_f = reinterpret_cast<char *>(partials) + (int64_t)f * tv.nslot * 16;
    for (int s = tv.tile_seg_ptr[t] + warp; s < s_end; s += kS1Warps) {
        const int beg = __ldg(tv.seg_ptr + s), end = __ldg(tv.seg_ptr + s + 1);
        Accum<ACC> S, C;
        if (!track) {
            for (int k = beg + lane * 4; k < end; k += 128) {
                float4 c4 = __ldg(reinterpret_cast<const float4 *>(tv.tcoef + k));
                ushort4 i4 = __ldg(reinterpret_cast<const ushort4 *>(tv.tidx + k));
                S.add(c4.x, tile[i4.x]);
                S.add(c4.y, tile[i4.y]);
                S.add(c4.z, tile[i4.z]);
                S.add(c4.w, tile[i4.w]);
            }
        } else {
            for (int k = beg + lane * 4; k < end; k += 128) {
                float4 c4 = __ldg(reinterpret_cast<const float4 *>(tv.tcoef + k));
                ushort4 i4 = __ldg(reinterpret_cast<const ushort4 *>(tv.tidx + k));
                float c[4] = {c4.x, c4.y, c4.z, c4.w};
                float v[4] = {tile[i4.x], tile[i4.y], tile[i4.z], tile[i4.w]};
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    bool ok = v[e] == v[e];
                    S.add(c[e], ok ? v[e] : 0.0f);
                    C.add1(ok ? c[e] : 0.0f);
                }
            }
            C.warp_reduce();
        }
        S.warp_reduce();
        if (lane == 0) store_partial<ACC>(part_f, __ldg(tv.seg_slot + s), S, C, track, track ? 0.0 : tv.seg_csum[s]);
    }
}

// ---- H5: fixed-order sum of each bin's partials, ratio, three outputs --------------------------------------------------
template <int ACC>
__global__ void __launch_bounds__(256) tiled_stage2_kernel(const int *__restrict__ bin_slot_ptr, int nslot, int npt,
                                                           const void *__restrict__ partials,
                                                           const double *__restrict__ range, float empty,
                                                           float *__restrict__ radial, float *__restrict__ intensity,
                                                           float *__restrict__ sum_signal, float *__restrict__ count)
{
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int f = blockIdx.y, lane = threadIdx.x & 31;
    if (b >= npt) return;
    const int beg = bin_slot_ptr[b], end = bin_slot_ptr[b + 1];
    const int64_t o = (int64_t)f * npt + b;
    if constexpr (ACC == AI_ACC_F32_PLAIN) {
        const float4 *p = reinterpret_cast<const float4 *>(partials) + (int64_t)f * nslot;
        float S = 0.f, C = 0.f;
        for (int k = beg + lane; k < end; k += 32) { float4 v = p[k]; S += v.x; C += v.z; }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            S += __shfl_xor_sync(AI_FULL_MASK, S, d);
            C += __shfl_xor_sync(AI_FULL_MASK, C, d);
        }
        if (lane == 0) write_bin_f32(0, S, C, empty, intensity + o, sum_signal + o, count + o);
    } else {
        double S = 0.0, C = 0.0;
        if constexpr (ACC == AI_ACC_F64) {
            const double2 *p = reinterpret_cast<const double2 *>(partials) + (int64_t)f * nslot;
            for (int k = beg + lane; k < end; k += 32) { double2 v = p[k]; S += v.x; C += v.y; }
        } else {
            const float4 *p = reinterpret_cast<const float4 *>(partials) + (int64_t)f * nslot;
            for (int k = beg + lane; k < end; k += 32) {
                float4 v = p[k];
                S += (double)v.x + (double)v.y;
                C += (double)v.z + (double)v.w;
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            S += __shfl_xor_sync(AI_FULL_MASK, S, d);
            C += __shfl_xor_sync(AI_FULL_MASK, C, d);
        }
        if (lane == 0) write_bin(0, S, C, empty, intensity + o, sum_signal + o, count + o);
    }
    if (lane == 0 && radial && f == 0) {
        double u0 = range[0], delta = (range[1] - range[0]) / (double)npt;
        radial[b] = (float)(u0 + ((double)b + 0.5) * delta);
    }
}

template <int DT, int ACC>
int launch_typed(ai_ctx *ctx, const FrameArgs &a, const TiledView &tv, const Corrections &cor, int vec_ok,
                 cudaStream_t st)
{
    dim3 g1(ctx->tl.ntiles, a.nframes);
    ai_prof_begin(ctx, st);
    tiled_stage1_kernel<DT, ACC><<<g1, kS1Threads, 0, st>>>(tv, a.image, a.frame_stride, cor, ctx->height, ctx->width,
                                                           vec_ok, ctx->partials);
    ai_prof_end(ctx, st);
    dim3 g2((ctx->npt + 7) / 8, a.nframes);
    tiled_stage2_kernel<ACC><<<g2, 256, 0, st>>>(tv.bin_slot_ptr, tv.nslot, ctx->npt, ctx->partials, ctx->d_range,
                                                 ctx->empty_value, a.radial, a.intensity, a.sum_signal, a.count);
    AI_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = 2;
    return AI_OK;
}

template <int DT>
int launch_dt(ai_ctx *ctx, const FrameArgs &a, const TiledView &tv, const Corrections &cor, int vec_ok, cudaStream_t st)
{
    switch (ctx->accum) {
    case AI_ACC_F32_KAHAN: return launch_typed<DT, AI_ACC_F32_KAHAN>(ctx, a, tv, cor, vec_ok, st);
    case AI_ACC_F32_PLAIN: return launch_typed<DT, AI_ACC_F32_PLAIN>(ctx, a, tv, cor, vec_ok, st);
    default: return launch_typed<DT, AI_ACC_F64>(ctx, a, tv, cor, vec_ok, st);
    }
}

bool aligned(const void *p, size_t a) { return p == nullptr || (reinterpret_cast<uintptr_t>(p) % a) == 0; }

}  // namespace

int ai_launch_tiled(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    const TiledLayout &tl = ctx->tl;
    const size_t need = (size_t)(tl.nslot > 0 ? tl.nslot : 1) * 16 * a.nframes;
    if (ctx->partials_bytes < need) {
        if (ctx->partials) AI_CUDA(ctx, cudaFree(ctx->partials));
        ctx->partials = nullptr;
        ctx->partials_bytes = 0;
        AI_CUDA(ctx, cudaMalloc(&ctx->partials, need));
        ctx->partials_bytes = need;
    }
    TiledView tv{tl.tile_seg_ptr, tl.seg_ptr, tl.seg_slot, tl.bin_slot_ptr, tl.seg_csum, tl.tcoef, tl.tidx, tl.tiles_x,
                 tl.nslot};
    Corrections cor{a.dark, a.flat, a.solidangle, a.polarization, a.mask};
    const size_t esz = (a.dtype == AI_U16 || a.dtype == AI_I16) ? 2 : 4;
    // 128-bit path: rows of 4 pixels never straddle the image edge and every array is aligned for 4-pixel vectors
    const int vec_ok = ctx->width % 4 == 0 && a.frame_stride % 4 == 0 && aligned(a.image, 4 * esz) &&
                       aligned(a.dark, 16) && aligned(a.flat, 16) && aligned(a.solidangle, 16) &&
                       aligned(a.polarization, 16) && aligned(a.mask, 4);
    switch (a.dtype) {
    case AI_F32: return launch_dt<AI_F32>(ctx, a, tv, cor, vec_ok, st);
    case AI_I32: return launch_dt<AI_I32>(ctx, a, tv, cor, vec_ok, st);
    case AI_U16: return launch_dt<AI_U16>(ctx, a, tv, cor, vec_ok, st);
    case AI_I16: return launch_dt<AI_I16>(ctx, a, tv, cor, vec_ok, st);
    case AI_U32: return launch_dt<AI_U32>(ctx, a, tv, cor, vec_ok, st);
    }
    return ai_fail(ctx, AI_EINVAL, "unknown dtype %d", (int)a.dtype);
}
