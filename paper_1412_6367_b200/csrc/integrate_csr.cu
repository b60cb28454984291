// Per-frame hot path in the paper's own two layouts, kept as selectable baselines for the TILED design:
//   AI_LAYOUT_CSR  canonical CSR, "all threads within a workgroup are collaborating to calculate the content of a
//                  single bin": one thread block per (bin, frame), pixel corrections applied at gather
//                  time, block-wide compensated reduction, one launch.
//   AI_LAYOUT_LUT  padded look-up table, one thread per bin walking its padded row, stored
//                  transposed so that neighbouring bins read neighbouring addresses.
#include "common.cuh"

namespace {

constexpr int kRowThreads = 256;

template <int ACC>
__device__ __forceinline__ void finish_bin(const Accum<ACC> &S, const Accum<ACC> &C, float empty, float *intensity,
                                           float *sum_signal, float *count)
{
    if constexpr (ACC == AI_ACC_F32_PLAIN) write_bin_f32(0, S.value_f(), C.value_f(), empty, intensity, sum_signal, count);
    else write_bin(0, S.value(), C.value(), empty, intensity, sum_signal, count);
}

template <int DT, int ACC>
__global__ void __launch_bounds__(kRowThreads) csr_row_kernel(const int32_t *__restrict__ indptr,
                                                              const int32_t *__restrict__ indices,
                                                              const float *__restrict__ data, int npt,
                                                              const void *frames, int64_t frame_stride,
                                                              Corrections cor, const double *__restrict__ range,
                                                              float empty, float *__restrict__ radial,
                                                              float *__restrict__ intensity,
                                                              float *__restrict__ sum_signal, float *__restrict__ count)
{
    using T = typename RawType<DT>::T;
    const int b = blockIdx.x, f = blockIdx.y;
    const void *img = reinterpret_cast<const T *>(frames) + (int64_t)f * frame_stride;
    const int beg = indptr[b], end = indptr[b + 1];
    Accum<ACC> S, C;
    for (int k = beg + threadIdx.x; k < end; k += kRowThreads) {
        float c = __ldg(data + k);
        float v = corrected_pixel<DT>(img, __ldg(indices + k), cor);
        bool ok = v == v;
        S.add(c, ok ? v : 0.0f);
        C.add1(ok ? c : 0.0f);
    }
    S.warp_reduce();
    C.warp_reduce();
    // per-warp results through shared memory as raw words (sum, compensation) x (S, C); thread 0 merges in warp order
    __shared__ double sh[kRowThreads / 32][4];
    if ((threadIdx.x & 31) == 0) {
        double *d = sh[threadIdx.x >> 5];
        d[0] = (double)S.s; d[2] = (double)C.s;
        if constexpr (ACC == AI_ACC_F32_KAHAN) { d[1] = (double)S.c; d[3] = (double)C.c; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < kRowThreads / 32; ++w) {
            const double *d = sh[w];
            if constexpr (ACC == AI_ACC_F32_KAHAN) { S.merge((float)d[0], (float)d[1]); C.merge((float)d[2], (float)d[3]); }
            else if constexpr (ACC == AI_ACC_F32_PLAIN) { S.s += (float)d[0]; C.s += (float)d[2]; }
            else { S.s += d[0]; C.s += d[2]; }
        }
        const int64_t o = (int64_t)f * npt + b;
        finish_bin<ACC>(S, C, empty, intensity + o, sum_signal + o, count + o);
        if (radial && f == 0) {
            double u0 = range[0], delta = (range[1] - range[0]) / (double)npt;
            radial[b] = (float)(u0 + ((double)b + 0.5) * delta);
        }
    }
}

template <int DT, int ACC>
__global__ void __launch_bounds__(128) lut_kernel(const float *__restrict__ lut_coef,
                                                  const int32_t *__restrict__ lut_idx, int lut_width, int npt,
                                                  const void *frames, int64_t frame_stride, Corrections cor,
                                                  const double *__restrict__ range, float empty,
                                                  float *__restrict__ radial, float *__restrict__ intensity,
                                                  float *__restrict__ sum_signal, float *__restrict__ count)
{
    using T = typename RawType<DT>::T;
    const int b = blockIdx.x * blockDim.x + threadIdx.x, f = blockIdx.y;
    if (b >= npt) return;
    const void *img = reinterpret_cast<const T *>(frames) + (int64_t)f * frame_stride;
    Accum<ACC> S, C;
    for (int j = 0; j < lut_width; ++j) {
        float c = __ldg(lut_coef + (int64_t)j * npt + b);
        float v = corrected_pixel<DT>(img, __ldg(lut_idx + (int64_t)j * npt + b), cor);
        bool ok = v == v;
        S.add(c, ok ? v : 0.0f);
        C.add1(ok ? c : 0.0f);
    }
    const int64_t o = (int64_t)f * npt + b;
    finish_bin<ACC>(S, C, empty, intensity + o, sum_signal + o, count + o);
    if (radial && f == 0) {
        double u0 = range[0], delta = (range[1] - range[0]) / (double)npt;
        radial[b] = (float)(u0 + ((double)b + 0.5) * delta);
    }
}

template <int DT, int ACC>
int launch_csr_typed(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    Corrections cor{a.dark, a.flat, a.solidangle, a.polarization, a.mask};
    dim3 grid(ctx->npt, a.nframes);
    ai_prof_begin(ctx, st);
    csr_row_kernel<DT, ACC><<<grid, kRowThreads, 0, st>>>(ctx->indptr, ctx->indices, ctx->data, ctx->npt, a.image,
                                                         a.frame_stride, cor, ctx->d_range, ctx->empty_value, a.radial,
                                                         a.intensity, a.sum_signal, a.count);
    ai_prof_end(ctx, st);
    AI_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = 1;
    return AI_OK;
}

template <int DT, int ACC>
int launch_lut_typed(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    Corrections cor{a.dark, a.flat, a.solidangle, a.polarization, a.mask};
    dim3 grid((ctx->npt + 127) / 128, a.nframes);
    ai_prof_begin(ctx, st);
    lut_kernel<DT, ACC><<<grid, 128, 0, st>>>(ctx->lut_coef, ctx->lut_idx, ctx->lut_width, ctx->npt, a.image,
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

int ai_launch_csr(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    AI_DISPATCH(csr, ctx, a, st)
    return ai_fail(ctx, AI_EINVAL, "unknown dtype %d", (int)a.dtype);
}

int ai_launch_lut(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    int rc = ai_build_lut(ctx, st);
    if (rc != AI_OK) return rc;
    AI_DISPATCH(lut, ctx, a, st)
    return ai_fail(ctx, AI_EINVAL, "unknown dtype %d", (int)a.dtype);
}
