// H1 + H2 as a streaming pre-pass for single frames that carry correction arrays, a mask or 16-bit pixels:
// cast, dark, flat, solid angle, polarisation in one pass over the pixels, invalid pixels
// (masked, zero / non-finite denominator, non-finite value: DESIGN.md reading 8) written as NaN.  The result is a
// float32 image owned by the context that the single-frame kernel (integrate_stream.cu) consumes right away -- 16.8 MB
// for a 2048 x 2048 frame, normally still in L2 when it is read back.  Chosen by measurement over staging the
// corrections inside the gather kernel.
#include "common.cuh"
#include "pipe_common.cuh"

namespace {

constexpr int kPrepThreads = 256;

template <int DT>
__global__ void __launch_bounds__(kPrepThreads) correct_frame_kernel(const void *__restrict__ img, Corrections cor,
                                                                     int64_t npix, int width, int pitch, int vec_ok,
                                                                     int overlap, int mode, float *__restrict__ out,
                                                                     const unsigned long long *chain_done,
                                                                     unsigned long long chain_target)
{
    // Launch chain (integrate_stream.cu): the single-frame kernel that follows may start its prologue (it reads `out`
    // after its griddepcontrol.wait).  overlap: this pass itself runs beside the stream kernel of the PREVIOUS call --
    // it reads the caller's inputs and writes the corrected frame of its own parity, which the call before the
    // previous one has finished reading (its stream kernel has left every SM) -- and waits for the grid dependency
    // only before it leaves, so that completion stays transitive along the stream.
    asm volatile("griddepcontrol.launch_dependents;");
    if (!overlap) asm volatile("griddepcontrol.wait;" ::: "memory");
    if (overlap) {
        // the corrected frame this pass overwrites was read by the stream kernel of the call before the previous one: it
        // has ended if the finish kernel behind it has (checked for the case of another tenant on the GPU, integrate_stream.cu)
        if (threadIdx.x == 0) wait_count_at_least(chain_done, chain_target);
        __syncthreads();
    }

    const bool has_den = cor.flat || cor.solidangle || cor.polarization;
    const int64_t stride = (int64_t)gridDim.x * kPrepThreads;
    if (vec_ok) {
        const float4 one4 = make_float4(1, 1, 1, 1), zero4 = make_float4(0, 0, 0, 0);
        for (int64_t q = (int64_t)blockIdx.x * kPrepThreads + threadIdx.x; q < npix / 4; q += stride) {
            const int64_t p = q * 4;
            const float4 raw = load_raw4<DT>(img, p);
            const float4 dk = cor.dark ? __ldg(reinterpret_cast<const float4 *>(cor.dark + p)) : zero4;
            const float4 fl = cor.flat ? __ldg(reinterpret_cast<const float4 *>(cor.flat + p)) : one4;
            const float4 sa = cor.solidangle ? __ldg(reinterpret_cast<const float4 *>(cor.solidangle + p)) : one4;
            const float4 po = cor.polarization ? __ldg(reinterpret_cast<const float4 *>(cor.polarization + p)) : one4;
            const uchar4 mk = cor.mask ? __ldg(reinterpret_cast<const uchar4 *>(cor.mask + p)) : make_uchar4(0, 0, 0, 0);
            float4 v;
            v.x = correct_value(raw.x, dk.x, fl.x, sa.x, po.x, mk.x != 0, has_den, mode);
            v.y = correct_value(raw.y, dk.y, fl.y, sa.y, po.y, mk.y != 0, has_den, mode);
            v.z = correct_value(raw.z, dk.z, fl.z, sa.z, po.z, mk.z != 0, has_den, mode);
            v.w = correct_value(raw.w, dk.w, fl.w, sa.w, po.w, mk.w != 0, has_den, mode);
            *reinterpret_cast<float4 *>(out + p) = v;
        }
    } else {
        // rows of the output start on 16-byte boundaries (pitch = width rounded up to 4): what the tensor map needs
        for (int64_t p = (int64_t)blockIdx.x * kPrepThreads + threadIdx.x; p < npix; p += stride) {
            const int64_t y = p / width;
            out[y * pitch + (p - y * width)] = corrected_pixel<DT>(img, p, cor, mode);
        }
    }
    if (overlap) asm volatile("griddepcontrol.wait;" ::: "memory");
}

}  // namespace

// Writes the corrected float32 image of frame 0 of `a` into one of the context's two corrected frames (*out; they
// alternate from call to call and are allocated on first use; row pitch = width rounded up to a multiple of 4, so that
// frames of any width reach the single-frame kernel through a tensor map).  mode: 0 corrected value, 1 numerator,
// 2 denominator (correct_value).
int ai_launch_correct(ai_ctx *ctx, const FrameArgs &a, int vec_ok, int overlap, int mode, cudaStream_t st, float **out)
{
    const int64_t npix = (int64_t)ctx->height * ctx->width;
    const int pitch = (ctx->width + 3) / 4 * 4;
    for (int i = 0; i < 2; ++i)
        if (!ctx->corrected[i]) AI_CUDA(ctx, cudaMalloc(&ctx->corrected[i], (size_t)ctx->height * pitch * sizeof(float)));
    float *dst = ctx->corrected[ctx->prep_launches & 1];
    Corrections cor{a.dark, a.flat, a.solidangle, a.polarization, a.mask};
    const int vec = vec_ok && ctx->width % 4 == 0;
    const int sms = ctx->sm_count > 0 ? ctx->sm_count : 148;
    int64_t blocks = ((vec ? npix / 4 : npix) + kPrepThreads - 1) / kPrepThreads;
    if (blocks > (int64_t)sms * 8) blocks = (int64_t)sms * 8;        // grid-stride: 8 resident blocks per SM
    if (blocks < 1) blocks = 1;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)blocks);
    cfg.blockDim = dim3(kPrepThreads);
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
#define AI_PREP(DT) \
    AI_CUDA(ctx, cudaLaunchKernelEx(&cfg, correct_frame_kernel<DT>, a.image, cor, npix, ctx->width, pitch, vec, overlap, mode, dst, \
                                    (const unsigned long long *)ctx->chain_done, ctx->fin_cum_prev))
    switch (a.dtype) {
    case AI_F32: AI_PREP(AI_F32); break;
    case AI_I32: AI_PREP(AI_I32); break;
    case AI_U16: AI_PREP(AI_U16); break;
    case AI_I16: AI_PREP(AI_I16); break;
    case AI_U32: AI_PREP(AI_U32); break;
    }
#undef AI_PREP
    ++ctx->prep_launches;
    *out = dst;
    return AI_OK;
}
