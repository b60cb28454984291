// Per-frame hot path in the paper's own two layouts, kept as selectable baselines for the TILED design and tuned as
// far as the layouts allow (they gather pixels of the whole frame through L2: a row is a thin ring, so a 32-byte sector
// is fetched for every 4-byte pixel -- that, not the kernels' shape, is what the tiled layout removes):
//   AI_LAYOUT_CSR  canonical CSR (PAPER.md:180 data / indices / indptr).  Rows are cut into segments of at most
//                  kCsrSegment entries (rows run from 16 to 17 544 entries: one thread block per bin, the paper's "all
//                  threads within a workgroup are collaborating to calculate the content of a single bin", leaves most
//                  of a B200 idle behind the long rows); one warp per segment, 128-bit coalesced loads of four
//                  coefficients and four indices per lane, per-lane compensated sums, shuffle merge, one partial per
//                  segment; a second small kernel adds each row's partials in order and writes the outputs.
//   AI_LAYOUT_LUT  padded look-up table, rows padded to the longest one, row-major; one warp
//                  per bin, the same 128-bit loads.  (The paper stores the table transposed for one work-item per bin,
//                  PAPER.md:176; with 1000 - 5000 bins that shape cannot fill 148 SMs.)
#include <stdlib.h>

#include <vector>

#include "common.cuh"

namespace {

constexpr int kCsrSegment = 2048;       // entries per warp-sized unit of work
constexpr int kCsrThreads = 256;

template <int ACC>
__device__ __forceinline__ void finish_bin(const Accum<ACC> &S, const Accum<ACC> &C, float empty, float *intensity,
                                           float *sum_signal, float *count)
{
    if constexpr (ACC == AI_ACC_F32_PLAIN) write_bin_f32(0, S.value_f(), C.value_f(), empty, intensity, sum_signal, count);
    else write_bin(0, S.value(), C.value(), empty, intensity, sum_signal, count);
}

template <int DT, int ACC>
__device__ __forceinline__ void gather_add(const void *img, const Corrections &cor, bool plain, int idx, float c,
                                           Accum<ACC> &S, Accum<ACC> &C)
{
    const float v = plain ? load_raw<DT>(img, idx) : corrected_pixel<DT>(img, idx, cor);
    const bool ok = DT == AI_F32 || !plain ? finite_f(v) : true;
    S.add(c, ok ? v : 0.0f);
    C.add1(ok ? c : 0.0f);
}

// entries [beg, end) of one row of (coef, idx) arrays, by one warp: scalar head up to a 16-byte boundary, 128-bit body,
// scalar tail
template <int DT, int ACC>
__device__ __forceinline__ void warp_row_part(const float *__restrict__ coef, const int32_t *__restrict__ idx, int beg,
                                              int end, const void *img, const Corrections &cor, bool plain, int lane,
                                              Accum<ACC> &S, Accum<ACC> &C)
{
    const int body0 = min(end, (beg + 3) & ~3), body1 = body0 + ((end - body0) & ~3);
    if (beg + lane < body0) gather_add<DT, ACC>(img, cor, plain, __ldg(idx + beg + lane), __ldg(coef + beg + lane), S, C);
    for (int k = body0 + 4 * lane; k < body1; k += 128) {
        const float4 c4 = __ldg(reinterpret_cast<const float4 *>(coef + k));
        const int4 x4 = __ldg(reinterpret_cast<const int4 *>(idx + k));
        gather_add<DT, ACC>(img, cor, plain, x4.x, c4.x, S, C);
        gather_add<DT, ACC>(img, cor, plain, x4.y, c4.y, S, C);
        gather_add<DT, ACC>(img, cor, plain, x4.z, c4.z, S, C);
        gather_add<DT, ACC>(img, cor, plain, x4.w, c4.w, S, C);
    }
    if (body1 + lane < end) gather_add<DT, ACC>(img, cor, plain, __ldg(idx + body1 + lane), __ldg(coef + body1 + lane), S, C);
}

// stage 1: one warp per (segment, frame); partial = (S_hi, S_lo, C_hi, C_lo) as four doubles' worth of two
template <int DT, int ACC>
__global__ void __launch_bounds__(kCsrThreads) csr_segment_kernel(const int4 *__restrict__ seg, int nseg,
                                                                  const int32_t *__restrict__ indices,
                                                                  const float *__restrict__ data, const void *frames,
                                                                  int64_t frame_stride, Corrections cor,
                                                                  double2 *__restrict__ partials)
{
    using T = typename RawType<DT>::T;
    const int s = blockIdx.x * (kCsrThreads / 32) + (threadIdx.x >> 5), f = blockIdx.y, lane = threadIdx.x & 31;
    if (s >= nseg) return;
    const void *img = reinterpret_cast<const T *>(frames) + (int64_t)f * frame_stride;
    const bool plain = !cor.dark && !cor.flat && !cor.solidangle && !cor.polarization && !cor.mask;
    const int4 sg = __ldg(seg + s);                  // {row, first entry, end entry, -}
    Accum<ACC> S, C;
    warp_row_part<DT, ACC>(data, indices, sg.y, sg.z, img, cor, plain, lane, S, C);
    S.warp_reduce();
    C.warp_reduce();
    if (lane == 0) partials[(int64_t)f * nseg + s] = make_double2(S.value(), C.value());
}

// stage 2: one thread per (bin, frame) adds the bin's partials in segment order
template <int ACC>
__global__ void __launch_bounds__(256) csr_finish_kernel(const int *__restrict__ row_seg_ptr, int npt, int nseg,
                                                         const double2 *__restrict__ partials,
                                                         const double *__restrict__ range, float empty,
                                                         float *__restrict__ radial, float *__restrict__ intensity,
                                                         float *__restrict__ sum_signal, float *__restrict__ count)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x, f = blockIdx.y;
    if (b >= npt) return;
    double S = 0.0, C = 0.0;
    for (int s = row_seg_ptr[b]; s < row_seg_ptr[b + 1]; ++s) {
        const double2 v = partials[(int64_t)f * nseg + s];
        S += v.x;
        C += v.y;
    }
    const int64_t o = (int64_t)f * npt + b;
    if constexpr (ACC == AI_ACC_F32_PLAIN) write_bin_f32(0, (float)S, (float)C, empty, intensity + o, sum_signal + o, count + o);
    else write_bin(0, S, C, empty, intensity + o, sum_signal + o, count + o);
    if (radial && f == 0) {
        double u0 = range[0], delta = (range[1] - range[0]) / (double)npt;
        radial[b] = (float)(u0 + ((double)b + 0.5) * delta);
    }
}

// one warp per (bin, frame) over the row-major padded table
template <int DT, int ACC>
__global__ void __launch_bounds__(kCsrThreads) lut_kernel(const float *__restrict__ lut_coef,
                                                          const int32_t *__restrict__ lut_idx, int lut_width, int npt,
                                                          const void *frames, int64_t frame_stride, Corrections cor,
                                                          const double *__restrict__ range, float empty,
                                                          float *__restrict__ radial, float *__restrict__ intensity,
                                                          float *__restrict__ sum_signal, float *__restrict__ count)
{
    using T = typename RawType<DT>::T;
    const int b = blockIdx.x * (kCsrThreads / 32) + (threadIdx.x >> 5), f = blockIdx.y, lane = threadIdx.x & 31;
    if (b >= npt) return;
    const void *img = reinterpret_cast<const T *>(frames) + (int64_t)f * frame_stride;
    const bool plain = !cor.dark && !cor.flat && !cor.solidangle && !cor.polarization && !cor.mask;
    Accum<ACC> S, C;
    const int64_t row = (int64_t)b * lut_width;     // lut_width is a multiple of 4: rows start on 16-byte boundaries
    for (int k = 4 * lane; k < lut_width; k += 128) {
        const float4 c4 = __ldg(reinterpret_cast<const float4 *>(lut_coef + row + k));
        const int4 x4 = __ldg(reinterpret_cast<const int4 *>(lut_idx + row + k));
        gather_add<DT, ACC>(img, cor, plain, x4.x, c4.x, S, C);
        gather_add<DT, ACC>(img, cor, plain, x4.y, c4.y, S, C);
        gather_add<DT, ACC>(img, cor, plain, x4.z, c4.z, S, C);
        gather_add<DT, ACC>(img, cor, plain, x4.w, c4.w, S, C);
    }
    S.warp_reduce();
    C.warp_reduce();
    if (lane == 0) {
        const int64_t o = (int64_t)f * npt + b;
        finish_bin<ACC>(S, C, empty, intensity + o, sum_signal + o, count + o);
        if (radial && f == 0) {
            double u0 = range[0], delta = (range[1] - range[0]) / (double)npt;
            radial[b] = (float)(u0 + ((double)b + 0.5) * delta);
        }
    }
}

// the table of row segments, built on first use (one host copy of indptr)
int ensure_segments(ai_ctx *ctx, cudaStream_t st)
{
    if (ctx->csr_seg) return AI_OK;
    std::vector<int32_t> indptr((size_t)ctx->npt + 1);
    AI_CUDA(ctx, cudaMemcpyAsync(indptr.data(), ctx->indptr, indptr.size() * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    std::vector<int4> seg;
    std::vector<int> ptr((size_t)ctx->npt + 1, 0);
    for (int b = 0; b < ctx->npt; ++b) {
        ptr[b] = (int)seg.size();
        const int beg = indptr[b], end = indptr[b + 1], n = end - beg;
        const int parts = n > 0 ? (n + kCsrSegment - 1) / kCsrSegment : 0;
        for (int q = 0; q < parts; ++q) {
            // equal parts, cut on 4-entry boundaries of the arrays so that the 128-bit bodies stay aligned
            int lo = beg + (int)((long long)n * q / parts), hi = beg + (int)((long long)n * (q + 1) / parts);
            if (q > 0) lo = (lo + 3) & ~3;
            if (q + 1 < parts) hi = (hi + 3) & ~3;
            if (hi > lo) seg.push_back(make_int4(b, lo, hi, 0));
        }
    }
    ptr[ctx->npt] = (int)seg.size();
    // built into local pointers and published together once both copies have arrived: a failure half-way leaves the
    // context without a table (the next call tries again), never with half of one
    const size_t n = seg.empty() ? 1 : seg.size();
    void *d_seg = nullptr;
    int *d_ptr = nullptr;
    cudaError_t e = cudaMalloc(&d_seg, n * sizeof(int4));
    if (e == cudaSuccess) e = cudaMalloc(&d_ptr, ptr.size() * sizeof(int));
    if (e == cudaSuccess && !seg.empty())
        e = cudaMemcpyAsync(d_seg, seg.data(), seg.size() * sizeof(int4), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_ptr, ptr.data(), ptr.size() * sizeof(int), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        cudaFree(d_seg);
        cudaFree(d_ptr);
        AI_CUDA(ctx, e);
    }
    ctx->csr_row_seg_ptr = d_ptr;
    ctx->csr_nseg = (int)seg.size();
    ctx->csr_seg = d_seg;
    return AI_OK;
}

template <int DT, int ACC>
int launch_csr_typed(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    int rc = ensure_segments(ctx, st);
    if (rc != AI_OK) return rc;
    const size_t need = (size_t)(ctx->csr_nseg > 0 ? ctx->csr_nseg : 1) * a.nframes * sizeof(double2);
    if (ctx->csr_partials_bytes < need) {
        if (ctx->csr_partials) AI_CUDA(ctx, cudaFree(ctx->csr_partials));
        ctx->csr_partials = nullptr;
        ctx->csr_partials_bytes = 0;
        AI_CUDA(ctx, cudaMalloc(&ctx->csr_partials, need));
        ctx->csr_partials_bytes = need;
    }
    Corrections cor{a.dark, a.flat, a.solidangle, a.polarization, a.mask};
    const int wpb = kCsrThreads / 32;
    ai_prof_begin(ctx, st);
    if (ctx->csr_nseg > 0)
        csr_segment_kernel<DT, ACC><<<dim3((ctx->csr_nseg + wpb - 1) / wpb, a.nframes), kCsrThreads, 0, st>>>(
            static_cast<const int4 *>(ctx->csr_seg), ctx->csr_nseg, ctx->indices, ctx->data, a.image, a.frame_stride, cor,
            static_cast<double2 *>(ctx->csr_partials));
    ai_prof_end(ctx, st);
    csr_finish_kernel<ACC><<<dim3((ctx->npt + 255) / 256, a.nframes), 256, 0, st>>>(
        ctx->csr_row_seg_ptr, ctx->npt, ctx->csr_nseg, static_cast<const double2 *>(ctx->csr_partials), ctx->d_range,
        ctx->empty_value, a.radial, a.intensity, a.sum_signal, a.count);
    AI_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = 2;
    return AI_OK;
}

template <int DT, int ACC>
int launch_lut_typed(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    Corrections cor{a.dark, a.flat, a.solidangle, a.polarization, a.mask};
    const int wpb = kCsrThreads / 32;
    dim3 grid((ctx->npt + wpb - 1) / wpb, a.nframes);
    ai_prof_begin(ctx, st);
    lut_kernel<DT, ACC><<<grid, kCsrThreads, 0, st>>>(ctx->lut_coef, ctx->lut_idx, ctx->lut_width, ctx->npt, a.image,
                                                     a.frame_stride, cor, ctx->d_range, ctx->empty_value, a.radial,
                                                     a.intensity, a.sum_signal, a.count);
    ai_prof_end(ctx, st);
    AI_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = 1;
    return AI_OK;
}

#define AI_DISPATCH(FN, ctx, a, st)                                                                         \
    switch ((a).dtype) {                                                                                    \
    case AI_F32: return dispatch_acc<AI_F32>(FN##_tag{}, ctx, a, st);                                       \
    case AI_I32: return dispatch_acc<AI_I32>(FN##_tag{}, ctx, a, st);                                       \
    case AI_U16: return dispatch_acc<AI_U16>(FN##_tag{}, ctx, a, st);                                       \
    case AI_I16: return dispatch_acc<AI_I16>(FN##_tag{}, ctx, a, st);                                       \
    case AI_U32: return dispatch_acc<AI_U32>(FN##_tag{}, ctx, a, st);                                       \
    }

struct csr_tag {};
struct lut_tag {};
template <int DT, int ACC> int call(csr_tag, ai_ctx *c, const FrameArgs &a, cudaStream_t s) { return launch_csr_typed<DT, ACC>(c, a, s); }
template <int DT, int ACC> int call(lut_tag, ai_ctx *c, const FrameArgs &a, cudaStream_t s) { return launch_lut_typed<DT, ACC>(c, a, s); }

template <int DT, class Tag>
int dispatch_acc(Tag tag, ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    switch (ctx->accum) {
    case AI_ACC_F32_KAHAN: return call<DT, AI_ACC_F32_KAHAN>(tag, ctx, a, st);
    case AI_ACC_F32_PLAIN: return call<DT, AI_ACC_F32_PLAIN>(tag, ctx, a, st);
    default: return call<DT, AI_ACC_F64>(tag, ctx, a, st);
    }
}

}  // namespace

// frames ride on gridDim.y in these comparison layouts
static int frames_fit_grid(ai_ctx *ctx, const FrameArgs &a)
{
    if (a.nframes > 65535) return ai_fail(ctx, AI_EUNSUPPORTED, "this layout takes at most 65535 frames per call (%d given)", a.nframes);
    return AI_OK;
}

int ai_launch_csr(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    if (int rc = frames_fit_grid(ctx, a)) return rc;
    AI_DISPATCH(csr, ctx, a, st)
    return ai_fail(ctx, AI_EINVAL, "unknown dtype %d", (int)a.dtype);
}

int ai_launch_lut(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    int rc = frames_fit_grid(ctx, a);
    if (rc != AI_OK) return rc;
    rc = ai_build_lut(ctx, st);
    if (rc != AI_OK) return rc;
    AI_DISPATCH(lut, ctx, a, st)
    return ai_fail(ctx, AI_EINVAL, "unknown dtype %d", (int)a.dtype);
}
