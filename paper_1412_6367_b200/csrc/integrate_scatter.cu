// AI_LAYOUT_SCATTER: the forward ("scatter") form of bounding-box pixel splitting on the GPU -- "linear read / random
// write", the form the paper's CPU code uses and its OpenCL code abandons because "the
// scatter operation ... requires the support of atomic operations".  B200 has fast fp32 atomics, so this
// is kept as a measured comparison against the matrix path: it reads the frame and 12
// bytes of split geometry per pixel (first bin, position inside it, width in bins) instead of 8 bytes per matrix entry.
//
// One thread block per 64 x 64 tile of the detector: a tile touches a short contiguous range of bins, so the block
// scatters into a shared-memory pair of histograms (shared-memory atomics) and adds that range to the global
// histograms with one global atomic per bin (tiles with a longer range scatter to global memory directly).  The paper's
// memset is back: the outputs are the accumulators.  Atomic sums are plain fp32 in whatever order the
// hardware takes them: NOT compensated and NOT bit-reproducible -- which is why this is a comparison, not the product
// path; the parity test holds it to 2e-5 and reports what it finds.
#include "build_common.cuh"
#include "common.cuh"

int ai_build_spans(ai_ctx *ctx, PixelSpans *sp, int npt, cudaStream_t st);

namespace {

constexpr int kScatTile = 64;
constexpr int kScatThreads = 256;
constexpr int kScatHist = 2048;          // bins of a tile kept in shared memory

// 12 bytes per pixel: first bin | number of bins << 24, position of the lower bound inside the first bin, width in bins
__global__ void __launch_bounds__(256) pack_spans_kernel(int64_t n, const double *__restrict__ fmin_a,
                                                         const double *__restrict__ fmax_a, const int *__restrict__ first_a,
                                                         const int *__restrict__ nb_a, int *__restrict__ first_nb,
                                                         float2 *__restrict__ gw, int *__restrict__ too_wide)
{
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
        const int first = first_a[p], nb = nb_a[p];
        if (nb > 255 || first >= (1 << 24)) *too_wide = 1;
        first_nb[p] = first | (min(nb, 255) << 24);
        // lower bound relative to the first bin (negative when the pixel starts below the range: that part is lost, the
        // width stays the pixel's)
        gw[p] = make_float2((float)(fmin_a[p] - (double)first), (float)(fmax_a[p] - fmin_a[p]));
    }
}

struct ScatArgs {
    const int *first_nb;
    const float2 *gw;
    int height, width, npt, tiles_x;
    const void *frames;
    int64_t frame_stride;
    Corrections cor;
    float *sum_signal, *count;        // [nframes][npt], zeroed
};

template <int DT>
__global__ void __launch_bounds__(kScatThreads) scatter_kernel(ScatArgs a)
{
    __shared__ float hs[kScatHist], hc[kScatHist];
    __shared__ int s_lo, s_hi;
    using T = typename RawType<DT>::T;
    const int f = blockIdx.y, ty = blockIdx.x / a.tiles_x, tx = blockIdx.x - ty * a.tiles_x;
    const void *img = reinterpret_cast<const T *>(a.frames) + (int64_t)f * a.frame_stride;
    float *S = a.sum_signal + (int64_t)f * a.npt, *C = a.count + (int64_t)f * a.npt;
    const bool plain = !a.cor.dark && !a.cor.flat && !a.cor.solidangle && !a.cor.polarization && !a.cor.mask;
    if (threadIdx.x == 0) { s_lo = 0x7fffffff; s_hi = -1; }
    __syncthreads();
    // range of bins of the tile
    int lo = 0x7fffffff, hi = -1;
    for (int k = threadIdx.x; k < kScatTile * kScatTile; k += kScatThreads) {
        const int y = ty * kScatTile + k / kScatTile, x = tx * kScatTile + k % kScatTile;
        if (y >= a.height || x >= a.width) continue;
        const int fn = __ldg(a.first_nb + (int64_t)y * a.width + x);
        const int first = fn & 0xffffff, nb = (unsigned)fn >> 24;
        if (nb) { lo = min(lo, first); hi = max(hi, first + nb - 1); }
    }
    atomicMin(&s_lo, lo);
    atomicMax(&s_hi, hi);
    __syncthreads();
    lo = s_lo; hi = s_hi;
    if (hi < 0) return;
    const bool local = hi - lo + 1 <= kScatHist;
    if (local) {
        for (int b = threadIdx.x; b <= hi - lo; b += kScatThreads) { hs[b] = 0.0f; hc[b] = 0.0f; }
        __syncthreads();
    }
    for (int k = threadIdx.x; k < kScatTile * kScatTile; k += kScatThreads) {
        const int y = ty * kScatTile + k / kScatTile, x = tx * kScatTile + k % kScatTile;
        if (y >= a.height || x >= a.width) continue;
        const int64_t p = (int64_t)y * a.width + x;
        const int fn = __ldg(a.first_nb + p);
        const int first = fn & 0xffffff, nb = (unsigned)fn >> 24;
        if (nb == 0) continue;
        const float v = plain ? load_raw<DT>(img, p) : corrected_pixel<DT>(img, p, a.cor);
        if (!finite_f(v)) continue;                       // masked / invalid pixel (O5)
        const float2 g = __ldg(a.gw + p);
        const float inv_w = g.y > 0.0f ? 1.0f / g.y : 0.0f;
        for (int q = 0; q < nb; ++q) {
            // overlap of [g, g + w] with bin q of the pixel's run, over w; the upper end is clipped by
            // the run itself (nb stops at the last bin of the range)
            float c = g.y > 0.0f ? (fminf(g.x + g.y, (float)(q + 1)) - fmaxf(fmaxf(g.x, 0.0f), (float)q)) * inv_w : 1.0f;
            c = fmaxf(c, 0.0f);
            const int b = first + q;
            if (local) {
                atomicAdd(&hs[b - lo], c * v);
                atomicAdd(&hc[b - lo], c);
            } else {
                atomicAdd(S + b, c * v);
                atomicAdd(C + b, c);
            }
        }
    }
    if (local) {
        __syncthreads();
        for (int b = threadIdx.x; b <= hi - lo; b += kScatThreads) {
            if (hc[b] != 0.0f) {
                atomicAdd(S + lo + b, hs[b]);
                atomicAdd(C + lo + b, hc[b]);
            }
        }
    }
}

__global__ void __launch_bounds__(256) scatter_finish_kernel(int npt, const double *__restrict__ range, float empty,
                                                             float *__restrict__ radial, float *__restrict__ intensity,
                                                             const float *__restrict__ sum_signal,
                                                             const float *__restrict__ count)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x, f = blockIdx.y;
    if (b >= npt) return;
    const int64_t o = (int64_t)f * npt + b;
    intensity[o] = count[o] > 0.0f ? __fdiv_rn(sum_signal[o], count[o]) : empty;
    if (radial && f == 0) {
        double u0 = range[0], delta = (range[1] - range[0]) / (double)npt;
        radial[b] = (float)(u0 + ((double)b + 0.5) * delta);
    }
}

}  // namespace

int ai_launch_scatter(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st)
{
    if (ctx->npt_azim > 0) return ai_fail(ctx, AI_EUNSUPPORTED, "the scatter comparison path is 1D only");
    // the per-pixel geometry below is the bounding box's; with full pixel splitting it would disagree with the matrix
    if (ctx->split == AI_SPLIT_FULL)
        return ai_fail(ctx, AI_EUNSUPPORTED, "the scatter comparison path splits by bounding box only (context built with AI_SPLIT_FULL)");
    if (a.nframes > 65535) return ai_fail(ctx, AI_EUNSUPPORTED, "this layout takes at most 65535 frames per call (%d given)", a.nframes);
    const int64_t n = (int64_t)ctx->height * ctx->width;
    if (!ctx->scat_first_nb) {
        // split geometry per pixel, from the same bounds as the matrix (one-time, synchronises)
        PixelSpans sp;
        const bool keep_range = ctx->user_range;
        ctx->user_range = true;                 // the range in use is final: do not recompute it
        double *saved = ctx->d_range;
        ctx->d_range = nullptr;
        int rc = ai_build_spans(ctx, &sp, ctx->npt, st);
        cudaFree(ctx->d_range);
        ctx->d_range = saved;
        ctx->user_range = keep_range;
        if (rc != AI_OK) { ai_free_spans(&sp); return rc; }
        int *too_wide = nullptr, h_wide = 0;
        cudaError_t e = cudaMalloc(&ctx->scat_first_nb, n * sizeof(int));
        if (e == cudaSuccess) e = cudaMalloc(&ctx->scat_gw, n * sizeof(float2));
        if (e == cudaSuccess) e = cudaMalloc(&too_wide, sizeof(int));
        if (e == cudaSuccess) e = cudaMemsetAsync(too_wide, 0, sizeof(int), st);
        if (e == cudaSuccess) {
            pack_spans_kernel<<<148 * 8, 256, 0, st>>>(n, sp.fmin, sp.fmax, sp.first, sp.nb, ctx->scat_first_nb,
                                                       static_cast<float2 *>(ctx->scat_gw), too_wide);
            e = cudaMemcpyAsync(&h_wide, too_wide, sizeof(int), cudaMemcpyDeviceToHost, st);
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        cudaFree(too_wide);
        ai_free_spans(&sp);
        AI_CUDA(ctx, e);
        if (h_wide) {
            cudaFree(ctx->scat_first_nb); cudaFree(ctx->scat_gw);
            ctx->scat_first_nb = nullptr; ctx->scat_gw = nullptr;
            return ai_fail(ctx, AI_EUNSUPPORTED, "scatter path: a pixel spans more than 255 bins or npt >= 2^24");
        }
    }
    const size_t out_bytes = (size_t)a.nframes * ctx->npt * sizeof(float);
    AI_CUDA(ctx, cudaMemsetAsync(a.sum_signal, 0, out_bytes, st));       // the memset is back
    AI_CUDA(ctx, cudaMemsetAsync(a.count, 0, out_bytes, st));
    ScatArgs s{ctx->scat_first_nb, static_cast<const float2 *>(ctx->scat_gw), ctx->height, ctx->width, ctx->npt,
               (ctx->width + kScatTile - 1) / kScatTile, a.image, a.frame_stride,
               Corrections{a.dark, a.flat, a.solidangle, a.polarization, a.mask}, a.sum_signal, a.count};
    const dim3 grid(s.tiles_x * ((ctx->height + kScatTile - 1) / kScatTile), a.nframes);
    ai_prof_begin(ctx, st);
    switch (a.dtype) {
    case AI_F32: scatter_kernel<AI_F32><<<grid, kScatThreads, 0, st>>>(s); break;
    case AI_I32: scatter_kernel<AI_I32><<<grid, kScatThreads, 0, st>>>(s); break;
    case AI_U16: scatter_kernel<AI_U16><<<grid, kScatThreads, 0, st>>>(s); break;
    case AI_I16: scatter_kernel<AI_I16><<<grid, kScatThreads, 0, st>>>(s); break;
    case AI_U32: scatter_kernel<AI_U32><<<grid, kScatThreads, 0, st>>>(s); break;
    }
    ai_prof_end(ctx, st);
    scatter_finish_kernel<<<dim3((ctx->npt + 255) / 256, a.nframes), 256, 0, st>>>(ctx->npt, ctx->d_range, ctx->empty_value,
                                                                                  a.radial, a.intensity, a.sum_signal, a.count);
    AI_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = 2;
    return AI_OK;
}
