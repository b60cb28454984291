// Held corrections (ai_hold_corrections, include/azint.h).  The correction arrays of an experiment -- dark current, flat
// field, solid angle, polarisation, mask -- do not change from frame to frame, and
//     sum_i c_i (I_i - dark_i) / den_i  =  sum_i (c_i / den_i) (I_i - dark_i).
// Holding a set of them folds the division and the mask into the matrix once: a copy of the tiled blobs with every
// coefficient multiplied by its pixel's 1 / den (0 for a pixel that is invalid for every frame: masked, zero or
// non-finite denominator or reciprocal, non-finite dark current) and the runs' coefficient sums (the count of a frame
// without invalid pixels) taken over the other pixels only.  What is left of H2 per frame is I - dark, done by the
// single-frame kernel on the fly (integrate_stream.cu, HELD: the dark tile arrives by TMA behind the frame tile), so a
// corrected frame costs one pass over the frame, the dark current and the matrix instead of a pre-pass over six arrays
// plus the pass over the corrected frame and the matrix.
//
// Derived arrays, per pixel: gone (byte), scale = 1 / den or 0, dark (0 where gone), keep (all ones, 0 where gone: float
// frames are ANDed with it so that a NaN under the mask stays harmless), den (0 where gone).  The last one, with `dark`,
// lets every other kernel of the library serve a held set as an ordinary (dark, flat) pair: a zero denominator is an
// invalid pixel there too.
#include "common.cuh"

namespace {

__global__ void __launch_bounds__(256) hold_prep_kernel(int64_t npix, Corrections cor, uint8_t *__restrict__ gone,
                                                        float *__restrict__ scale, float *__restrict__ dark,
                                                        uint32_t *__restrict__ keep, float *__restrict__ den_out)
{
    const bool has_den = cor.flat || cor.solidangle || cor.polarization;
    for (int64_t px = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; px < npix; px += (int64_t)gridDim.x * blockDim.x) {
        bool g = cor.mask && __ldg(cor.mask + px) != 0;
        float sc = 1.0f, den = 1.0f;
        if (has_den) {
            den = cor.flat ? __ldg(cor.flat + px) : 1.0f;
            den *= cor.solidangle ? __ldg(cor.solidangle + px) : 1.0f;
            den *= cor.polarization ? __ldg(cor.polarization + px) : 1.0f;
            sc = __frcp_rn(den);
            g = g || den == 0.f || !finite_f(den) || !finite_f(sc);
        }
        const float dk = cor.dark ? __ldg(cor.dark + px) : 0.f;
        g = g || !finite_f(dk);
        gone[px] = g ? 1 : 0;
        scale[px] = g ? 0.f : sc;
        dark[px] = g ? 0.f : dk;
        keep[px] = g ? 0u : 0xffffffffu;
        if (den_out) den_out[px] = g ? 0.f : den;
    }
}

// One warp per block of the sliced layout (ctx.h): coefficients times the scale of their pixels, positions and the rest
// copied, and the run heads' coefficient sums recomputed over the pixels that are not gone -- the same suffix sums by
// doubling as the kernel's own (integrate_stream.cu: stream_finish_d), in fp64.
__global__ void __launch_bounds__(256) hold_scale_tiled_kernel(int ntiles, const int4 *__restrict__ blob_desc,
                                                               const unsigned char *__restrict__ blob,
                                                               const float *__restrict__ scale, int width, int height,
                                                               int tile_h, unsigned char *__restrict__ out)
{
    const int t = blockIdx.x, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (t >= ntiles) return;
    const int4 d = __ldg(blob_desc + t);
    const unsigned char *src = blob + (size_t)d.x * 16;
    unsigned char *dst = out + (size_t)d.x * 16;
    const int x0 = (d.z & 0xffff) * kTileW, y0 = (d.z >> 16) * tile_h;
    // the whole blob first (header: number of blocks, then one word per block; positions; padding), then the
    // coefficients and the run sums are overwritten
    for (int i = threadIdx.x; i < d.y / 16; i += blockDim.x)
        reinterpret_cast<uint4 *>(dst)[i] = __ldg(reinterpret_cast<const uint4 *>(src) + i);
    __syncthreads();
    const unsigned *hdr = reinterpret_cast<const unsigned *>(src);
    const int nblk = d.w;
    auto factor = [&](unsigned off) {
        const int pf = (int)(off >> 2), half = pf / (tile_h * 32), o = pf - half * tile_h * 32;
        const int ly = o >> 5, w = o & 31;
        const int lx = half * 32 + ((((w >> 2) ^ (ly & 7)) & 7) << 2) + (w & 3);
        const int y = y0 + ly, x = x0 + lx;
        return (y < height && x < width) ? __ldg(scale + (int64_t)y * width + x) : 0.f;
    };
    for (int b = warp; b < nblk; b += blockDim.x / 32) {
        const unsigned h = hdr[1 + b];
        const int nsteps = h & 15, rounds = (h >> 4) & 7;
        const size_t off = (size_t)(h >> 8) * 16;
        const float4 *cp = reinterpret_cast<const float4 *>(src + off) + lane;
        const uint2 *xp = reinterpret_cast<const uint2 *>(src + off + nsteps * 512) + lane;
        float4 *cq = reinterpret_cast<float4 *>(dst + off) + lane;
        double sum = 0.0;
        for (int j = 0; j < nsteps; ++j) {
            const float4 c = cp[j * 32];
            const uint2 x = xp[j * 32];
            const float f0 = factor(x.x & 0xffffu), f1 = factor(x.x >> 16), f2 = factor(x.y & 0xffffu), f3 = factor(x.y >> 16);
            cq[j * 32] = make_float4(__fmul_rn(c.x, f0), __fmul_rn(c.y, f1), __fmul_rn(c.z, f2), __fmul_rn(c.w, f3));
            sum += (double)(f0 != 0.f ? c.x : 0.f) + (double)(f1 != 0.f ? c.y : 0.f) + (double)(f2 != 0.f ? c.z : 0.f) +
                   (double)(f3 != 0.f ? c.w : 0.f);
        }
        int2 m = reinterpret_cast<const int2 *>(src + off + nsteps * kBlkStepBytes)[lane];
        const int rem = (m.x >> 24) & 31;
        for (int r = 0; r < rounds; ++r) {
            const int dd = 1 << r;
            const double o = __shfl_down_sync(AI_FULL_MASK, sum, dd);
            if (rem >= dd) sum += o;
        }
        if (m.x < 0) m.y = __float_as_int((float)sum);
        reinterpret_cast<int2 *>(dst + off + nsteps * kBlkStepBytes)[lane] = m;
    }
}

}  // namespace

// the derived per-pixel arrays of one set of correction arrays (den_out may be NULL)
int ai_launch_corr_prep(ai_ctx *ctx, const float *dark, const float *flat, const float *solidangle, const float *polarization,
                        const uint8_t *mask, uint8_t *gone, float *scale, float *dark_out, uint32_t *keep, float *den_out,
                        cudaStream_t st)
{
    const int64_t npix = (int64_t)ctx->height * ctx->width;
    const int sms = ctx->sm_count > 0 ? ctx->sm_count : 148;
    const Corrections cor{dark, flat, solidangle, polarization, mask};
    hold_prep_kernel<<<sms * 8, 256, 0, st>>>(npix, cor, gone, scale, dark_out, keep, den_out);
    AI_CUDA(ctx, cudaGetLastError());
    return AI_OK;
}

void ai_release_held(ai_ctx *ctx)
{
    HeldCorrections &h = ctx->held;
    cudaFree(h.gone); cudaFree(h.scale); cudaFree(h.tl_blob); cudaFree(h.fl_blob); cudaFree(h.fl_csum);
    h = HeldCorrections{};
}

// see include/azint.h: ai_hold_corrections
int ai_hold_build(ai_ctx *ctx, const float *dark, const float *flat, const float *solidangle, const float *polarization,
                  const uint8_t *mask, cudaStream_t st)
{
    HeldCorrections &h = ctx->held;
    const int64_t npix = (int64_t)ctx->height * ctx->width;
    h.on = false;
    h.fl_ready = false;
    if (!h.gone) AI_CUDA(ctx, cudaMalloc(&h.gone, (size_t)npix));
    if (!h.scale) {
        AI_CUDA(ctx, cudaMalloc(&h.scale, 4 * (size_t)npix * sizeof(float)));
        h.dark = h.scale + npix;
        h.keep = reinterpret_cast<uint32_t *>(h.scale + 2 * npix);
        h.den = h.scale + 3 * npix;
    }
    int rc = ai_launch_corr_prep(ctx, dark, flat, solidangle, polarization, mask, h.gone, h.scale, h.dark, h.keep, h.den, st);
    if (rc != AI_OK) return rc;
    const TiledLayout &tl = ctx->tl;
    h.tl_ready = false;
    if (tl.blob && tl.ntiles > 0 && tl.blob_bytes > 0) {      // (1D and 2D; whatever ai_set_options says now)
        if (!h.tl_blob) AI_CUDA(ctx, cudaMalloc(&h.tl_blob, (size_t)tl.blob_bytes));
        hold_scale_tiled_kernel<<<tl.ntiles, 256, 0, st>>>(tl.ntiles, tl.blob_desc, tl.blob, h.scale, ctx->width, ctx->height,
                                                          tl.tile_h, h.tl_blob);
        AI_CUDA(ctx, cudaGetLastError());
        h.tl_ready = true;
    }
    h.on = true;
    return AI_OK;
}
