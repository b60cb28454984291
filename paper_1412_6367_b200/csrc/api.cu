// C ABI entry points of libazint (include/azint.h): argument checks, context life cycle, dispatch to the kernels.
#include <math.h>
#include <stdarg.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "ctx.h"

int ai_fail(ai_ctx *ctx, int code, const char *fmt, ...)
{
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

extern "C" {

const char *ai_strerror(int code)
{
    switch (code) {
    case AI_OK: return "ok";
    case AI_EINVAL: return "invalid argument";
    case AI_ENOTBUILT: return "matrix not built (call ai_build_csr first)";
    case AI_ECUDA: return "CUDA error";
    case AI_ENOMEM: return "out of memory";
    case AI_EUNSUPPORTED: return "unsupported size";
    }
    return "unknown status";
}

const char *ai_last_error(const ai_ctx *ctx) { return ctx ? ctx->err : ""; }

int ai_last_launch_count(const ai_ctx *ctx) { return ctx ? ctx->last_launches : 0; }

int ai_get_layout_info(const ai_ctx *ctx, int64_t info[8])
{
    if (!ctx || !info) return AI_EINVAL;
    if (!ctx->built) return AI_ENOTBUILT;
    const TiledLayout &tl = ctx->tl;
    info[0] = tl.tile_h;
    info[1] = tl.ntiles;
    info[2] = tl.nseg;
    info[3] = tl.tnnz;
    info[4] = tl.blob_bytes;
    info[5] = tl.max_blob_bytes;
    info[6] = tl.nslot;
    info[7] = ai_stream_stages(ctx);
    return AI_OK;
}

int ai_get_batch_layout_info(const ai_ctx *ctx, int64_t info[8])
{
    if (!ctx || !info) return AI_EINVAL;
    if (!ctx->built) return AI_ENOTBUILT;
    const FlLayout &fl = ctx->fl;
    for (int k = 0; k < 8; ++k) info[k] = 0;
    if (!fl.ok) return AI_OK;
    info[0] = 1;
    info[1] = kFlTileH;
    info[2] = fl.ntiles;
    info[3] = fl.nchunks;
    info[4] = fl.nslot;
    info[5] = fl.blob_bytes;
    info[6] = fl.max_blob_bytes;
    info[7] = kFlFrames;
    return AI_OK;
}

int ai_profile_enable(ai_ctx *ctx, int on)
{
    if (!ctx) return AI_EINVAL;
    if (on == 1 && !ctx->ev0) {
        AI_CUDA(ctx, cudaEventCreate(&ctx->ev0));
        AI_CUDA(ctx, cudaEventCreate(&ctx->ev1));
    }
    ctx->profile = on == 1;
    ctx->stage1_only = on == 2;
    ctx->profile_valid = false;
    return AI_OK;
}

int ai_profile_last(ai_ctx *ctx, float *kernel_ms)
{
    if (!ctx || !kernel_ms) return AI_EINVAL;
    if (!ctx->profile_valid) return ai_fail(ctx, AI_EINVAL, "no profiled call yet");
    AI_CUDA(ctx, cudaEventSynchronize(ctx->ev1));
    AI_CUDA(ctx, cudaEventElapsedTime(kernel_ms, ctx->ev0, ctx->ev1));
    return AI_OK;
}

static void release_matrix_and_scratch(ai_ctx *ctx);
static int setup_common(ai_ctx **out, const ai_geometry *g, int height, int width, int npt, ai_unit unit,
                        const double *range_or_null);

int ai_setup(ai_ctx **out, const ai_geometry *g, int height, int width, int npt, ai_unit unit,
             const double *range_or_null)
{
    int rc = setup_common(out, g, height, width, npt, unit, range_or_null);
    if (rc == AI_OK) (*out)->npt_rad = npt;
    return rc;
}

int ai_setup2d(ai_ctx **out, const ai_geometry *g, int height, int width, int npt_rad, int npt_azim, ai_unit unit,
               const double *range_or_null, const double *azim_range_or_null)
{
    if (!out) return AI_EINVAL;
    *out = nullptr;
    if (npt_rad < 1 || npt_azim < 1 || (int64_t)npt_rad * npt_azim > 0xfffffffLL) return AI_EINVAL;
    const double two_pi = 2.0 * 3.14159265358979323846;
    if (azim_range_or_null && !(azim_range_or_null[1] > azim_range_or_null[0] && isfinite(azim_range_or_null[0]) &&
                                isfinite(azim_range_or_null[1]) &&
                                azim_range_or_null[1] - azim_range_or_null[0] <= two_pi * (1.0 + 1e-15) &&
                                azim_range_or_null[0] >= -two_pi && azim_range_or_null[1] <= 1.5 * two_pi))
        return AI_EINVAL;       // (a pixel's chi interval starts in [-pi, pi); its images shifted by -2 pi, 0 and +2 pi
                                //  are what the builder looks at: together they cover [-3 pi, 3 pi])
    int rc = setup_common(out, g, height, width, npt_rad * npt_azim, unit, range_or_null);
    if (rc != AI_OK) return rc;
    (*out)->npt_rad = npt_rad;
    (*out)->npt_azim = npt_azim;
    if (azim_range_or_null) {
        (*out)->azim_host[0] = azim_range_or_null[0];
        (*out)->azim_host[1] = azim_range_or_null[1];
    }
    return AI_OK;
}

static int setup_common(ai_ctx **out, const ai_geometry *g, int height, int width, int npt, ai_unit unit,
                        const double *range_or_null)
{
    if (!out) return AI_EINVAL;
    *out = nullptr;
    if (!g || height < 1 || width < 1 || npt < 1) return AI_EINVAL;
    if ((int)unit < AI_R_MM || (int)unit > AI_Q_A) return AI_EINVAL;
    if (!(g->distance_m > 0.0) || !(g->pixel_x_m > 0.0) || !(g->pixel_y_m > 0.0) || !(g->wavelength_m > 0.0)) return AI_EINVAL;
    if (!isfinite(g->distance_m) || !isfinite(g->pixel_x_m) || !isfinite(g->pixel_y_m) || !isfinite(g->wavelength_m) ||
        !isfinite(g->center_x_px) || !isfinite(g->center_y_px))
        return AI_EINVAL;
    if ((int64_t)height * width > 0x7fffffffLL) return AI_EUNSUPPORTED;     // pixel indices are int32
    if (range_or_null && !(range_or_null[1] > range_or_null[0] && isfinite(range_or_null[0]) && isfinite(range_or_null[1])))
        return AI_EINVAL;
    ai_ctx *ctx = new (std::nothrow) ai_ctx();
    if (!ctx) return AI_ENOMEM;
    ctx->geo = *g;
    ctx->height = height;
    ctx->width = width;
    ctx->npt = npt;
    ctx->unit = unit;
    if (range_or_null) {
        ctx->user_range = true;
        ctx->range_host[0] = range_or_null[0];
        ctx->range_host[1] = range_or_null[1];
    }
    *out = ctx;
    return AI_OK;
}

int ai_build_csr(ai_ctx *ctx, void *cuda_stream)
{
    if (!ctx) return AI_EINVAL;
    if (ctx->built) return AI_OK;
    release_matrix_and_scratch(ctx);          // whatever an earlier, failed build left
    cudaStream_t st = (cudaStream_t)cuda_stream;
    AI_CUDA(ctx, cudaGetDevice(&ctx->device));
    AI_CUDA(ctx, cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device));
    int rc;
    if (ctx->npt_azim > 0) {
        rc = ai_build_2d(ctx, st);
        if (rc == AI_OK) {
            // bin centres of the two axes, copied out by ai_integrate2d
            float *h = static_cast<float *>(malloc(((size_t)ctx->npt_rad + ctx->npt_azim) * sizeof(float)));
            if (!h) return ai_fail(ctx, AI_ENOMEM, "axes");
            const double du = (ctx->range_host[1] - ctx->range_host[0]) / ctx->npt_rad;
            const double dc = (ctx->azim_host[1] - ctx->azim_host[0]) / ctx->npt_azim;
            for (int r = 0; r < ctx->npt_rad; ++r) h[r] = (float)(ctx->range_host[0] + (r + 0.5) * du);
            for (int a = 0; a < ctx->npt_azim; ++a) h[ctx->npt_rad + a] = (float)(ctx->azim_host[0] + (a + 0.5) * dc);
            cudaError_t e = cudaMalloc(&ctx->axes2d, ((size_t)ctx->npt_rad + ctx->npt_azim) * sizeof(float));
            if (e == cudaSuccess)
                e = cudaMemcpy(ctx->axes2d, h, ((size_t)ctx->npt_rad + ctx->npt_azim) * sizeof(float), cudaMemcpyHostToDevice);
            free(h);
            AI_CUDA(ctx, e);
        }
    } else if (ctx->split == AI_SPLIT_FULL) {
        rc = ai_build_full(ctx, st);
    } else {
        PixelSpans spans;
        rc = ai_build_canonical(ctx, &spans, st);
        if (rc == AI_OK) rc = ai_build_tiled(ctx, spans, st);
        ai_free_spans(&spans);
    }
    if (rc != AI_OK) return rc;
    AI_CUDA(ctx, cudaMalloc(&ctx->out_dev, 3 * (size_t)ctx->npt * sizeof(float)));
    AI_CUDA(ctx, cudaMalloc(&ctx->grid_sync, 3 * sizeof(unsigned long long)));
    AI_CUDA(ctx, cudaMalloc(&ctx->chain_done, sizeof(unsigned long long)));
    AI_CUDA(ctx, cudaMemsetAsync(ctx->chain_done, 0, sizeof(unsigned long long), st));
    AI_CUDA(ctx, cudaMemsetAsync(ctx->grid_sync, 0, 3 * sizeof(unsigned long long), st));
    AI_CUDA(ctx, cudaMalloc(&ctx->stream_partials, 2 * (size_t)(ctx->tl.nslot > 0 ? ctx->tl.nslot : 1) * 16));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    ctx->built = true;
    return AI_OK;
}

int ai_get_csr(const ai_ctx *ctx, const int32_t **indptr, const int32_t **indices, const float **data, int64_t *nnz,
               double *u0, double *u1)
{
    if (!ctx) return AI_EINVAL;
    if (!ctx->built) return AI_ENOTBUILT;
    if (indptr) *indptr = ctx->indptr;
    if (indices) *indices = ctx->indices;
    if (data) *data = ctx->data;
    if (nnz) *nnz = ctx->nnz;
    if (u0) *u0 = ctx->range_host[0];
    if (u1) *u1 = ctx->range_host[1];
    return AI_OK;
}

int ai_copy_csr_to_host(const ai_ctx *ctx, int32_t *indptr_host, int32_t *indices_host, float *data_host)
{
    if (!ctx) return AI_EINVAL;
    if (!ctx->built) return AI_ENOTBUILT;
    ai_ctx *c = const_cast<ai_ctx *>(ctx);      // only the error text is written
    if (indptr_host)
        AI_CUDA(c, cudaMemcpy(indptr_host, ctx->indptr, ((size_t)ctx->npt + 1) * sizeof(int32_t), cudaMemcpyDeviceToHost));
    if (indices_host && ctx->nnz)
        AI_CUDA(c, cudaMemcpy(indices_host, ctx->indices, (size_t)ctx->nnz * sizeof(int32_t), cudaMemcpyDeviceToHost));
    if (data_host && ctx->nnz)
        AI_CUDA(c, cudaMemcpy(data_host, ctx->data, (size_t)ctx->nnz * sizeof(float), cudaMemcpyDeviceToHost));
    return AI_OK;
}

int ai_set_options(ai_ctx *ctx, ai_layout layout, ai_accum accum, float empty_value)
{
    if (!ctx) return AI_EINVAL;
    if ((int)layout < AI_LAYOUT_TILED || (int)layout > AI_LAYOUT_SCATTER) return ai_fail(ctx, AI_EINVAL, "bad layout %d", (int)layout);
    if ((int)accum < AI_ACC_F32_KAHAN || (int)accum > AI_ACC_F64) return ai_fail(ctx, AI_EINVAL, "bad accum %d", (int)accum);
    ctx->layout = layout;
    ctx->accum = accum;
    ctx->empty_value = empty_value;
    return AI_OK;
}

int ai_set_path_options(ai_ctx *ctx, const ai_path_options *opt)
{
    if (!ctx) return AI_EINVAL;
    if (ctx->built) return ai_fail(ctx, AI_EINVAL, "path options are fixed once the matrix is built");
    const ai_path_options none{};
    const ai_path_options &o = opt ? *opt : none;
    for (int r : o.reserved)
        if (r != 0) return ai_fail(ctx, AI_EINVAL, "ai_path_options.reserved must be zero");
    if (o.fl_chunk < 0 || o.fl_stages < 0 || (o.no_fl && o.force_fl))
        return ai_fail(ctx, AI_EINVAL, "bad path options (negative size, or no_fl together with force_fl)");
    ctx->no_tma = o.no_tma != 0;
    ctx->no_schedule = o.no_schedule != 0;
    ctx->no_prepass = o.no_prepass != 0;
    ctx->no_stream = o.no_stream != 0;
    ctx->no_fl = o.no_fl != 0;
    ctx->force_fl = o.force_fl != 0;
    ctx->tune.no_overlap = o.no_overlap != 0;
    ctx->tune.fl_chunk = o.fl_chunk;
    ctx->tune.fl_stages = o.fl_stages;
    ctx->tune.fl_owner = o.fl_owner != 0;
    return AI_OK;
}

int ai_set_splitting(ai_ctx *ctx, ai_split split)
{
    if (!ctx) return AI_EINVAL;
    if ((int)split < AI_SPLIT_BBOX || (int)split > AI_SPLIT_FULL) return ai_fail(ctx, AI_EINVAL, "bad splitting %d", (int)split);
    if (ctx->built) return ai_fail(ctx, AI_EINVAL, "the matrix is already built");
    if (split == AI_SPLIT_FULL && ctx->npt_azim > 0) return ai_fail(ctx, AI_EUNSUPPORTED, "full pixel splitting is 1D only");
    ctx->split = split;
    return AI_OK;
}

int ai_set_normalization(ai_ctx *ctx, ai_norm norm)
{
    if (!ctx) return AI_EINVAL;
    if ((int)norm < AI_NORM_PIXEL || (int)norm > AI_NORM_SPLIT) return ai_fail(ctx, AI_EINVAL, "bad normalisation %d", (int)norm);
    ctx->norm = norm;
    return AI_OK;
}

static int integrate(ai_ctx *ctx, const FrameArgs &args, cudaStream_t st)
{
    if (!ctx) return AI_EINVAL;
    if (!ctx->built) return ai_fail(ctx, AI_ENOTBUILT, "ai_build_csr has not been called");
    // held corrections (ai_hold_corrections) serve the calls that pass no correction array of their own: to every kernel
    // but the ones that know better (hold.cu) they are a dark current and a denominator, 0 where the pixel is invalid
    FrameArgs a = args;
    if (ctx->held.on && !a.dark && !a.flat && !a.solidangle && !a.polarization && !a.mask) {
        a.held = true;
        a.dark = ctx->held.dark;
        // always with the denominator, also for a set that holds a dark current only: a pixel whose dark current is not
        // finite is invalid for every frame, and the derived pair says so through den == 0 (its dark reads 0 there)
        a.flat = ctx->held.den;
    }
    if (!a.image || !a.intensity || !a.sum_signal || !a.count) return ai_fail(ctx, AI_EINVAL, "NULL image or output");
    if ((int)a.dtype < AI_F32 || (int)a.dtype > AI_U32) return ai_fail(ctx, AI_EINVAL, "bad dtype %d", (int)a.dtype);
    if (a.nframes < 1) return ai_fail(ctx, AI_EINVAL, "nframes < 1");
    int dev = -1;
    AI_CUDA(ctx, cudaGetDevice(&dev));
    if (dev != ctx->device)
        return ai_fail(ctx, AI_EINVAL, "the matrix was built on device %d, the current device is %d", ctx->device, dev);
    if (a.frame_stride < (int64_t)ctx->height * ctx->width) return ai_fail(ctx, AI_EINVAL, "frame stride < height*width");
    if (ctx->norm == AI_NORM_SPLIT) {
        if (ctx->layout != AI_LAYOUT_TILED) return ai_fail(ctx, AI_EUNSUPPORTED, "split normalisation: AI_LAYOUT_TILED only");
        return ai_launch_tiled_split(ctx, a, st);
    }
    switch (ctx->layout) {
    case AI_LAYOUT_TILED:
    case AI_LAYOUT_TILED_DIRECT: return ai_launch_tiled(ctx, a, st);
    case AI_LAYOUT_CSR: return ai_launch_csr(ctx, a, st);
    case AI_LAYOUT_LUT: return ai_launch_lut(ctx, a, st);
    case AI_LAYOUT_SCATTER: return ai_launch_scatter(ctx, a, st);
    }
    return AI_EINVAL;
}

int ai_integrate1d(ai_ctx *ctx, const void *image, ai_dtype dtype, const float *dark, const float *flat,
                   const float *solidangle, const float *polarization, const uint8_t *mask, float *radial,
                   float *intensity, float *sum_signal, float *count, void *cuda_stream)
{
    if (!ctx) return AI_EINVAL;
    if (ctx->npt_azim > 0) return ai_fail(ctx, AI_EINVAL, "bidimensional context: use ai_integrate2d");
    FrameArgs a{image, dtype, dark, flat, solidangle, polarization, mask, radial, intensity, sum_signal, count, 1,
                (int64_t)ctx->height * ctx->width};
    return integrate(ctx, a, (cudaStream_t)cuda_stream);
}

int ai_hold_corrections(ai_ctx *ctx, const float *dark, const float *flat, const float *solidangle,
                        const float *polarization, const uint8_t *mask, void *cuda_stream)
{
    if (!ctx) return AI_EINVAL;
    if (!ctx->built) return ai_fail(ctx, AI_ENOTBUILT, "ai_build_csr has not been called");
    int dev = -1;
    AI_CUDA(ctx, cudaGetDevice(&dev));
    if (dev != ctx->device)
        return ai_fail(ctx, AI_EINVAL, "the matrix was built on device %d, the current device is %d", ctx->device, dev);
    if (!dark && !flat && !solidangle && !polarization && !mask) {
        // scratch of calls in flight on other streams is the caller's to wait for, as with ai_destroy
        ai_release_held(ctx);
        return AI_OK;
    }
    return ai_hold_build(ctx, dark, flat, solidangle, polarization, mask, (cudaStream_t)cuda_stream);
}

int ai_integrate2d(ai_ctx *ctx, const void *image, ai_dtype dtype, const float *dark, const float *flat,
                   const float *solidangle, const float *polarization, const uint8_t *mask, float *radial,
                   float *azimuthal, float *intensity, float *sum_signal, float *count, void *cuda_stream)
{
    if (!ctx) return AI_EINVAL;
    if (ctx->npt_azim < 1) return ai_fail(ctx, AI_EINVAL, "not a bidimensional context (use ai_setup2d)");
    if (ctx->layout == AI_LAYOUT_LUT) return ai_fail(ctx, AI_EUNSUPPORTED, "no padded LUT for the 2D matrix");
    FrameArgs a{image, dtype, dark, flat, solidangle, polarization, mask, nullptr, intensity, sum_signal, count, 1,
                (int64_t)ctx->height * ctx->width};
    int rc = integrate(ctx, a, (cudaStream_t)cuda_stream);
    if (rc != AI_OK) return rc;
    if (radial)
        AI_CUDA(ctx, cudaMemcpyAsync(radial, ctx->axes2d, (size_t)ctx->npt_rad * sizeof(float), cudaMemcpyDeviceToDevice,
                                     (cudaStream_t)cuda_stream));
    if (azimuthal)
        AI_CUDA(ctx, cudaMemcpyAsync(azimuthal, ctx->axes2d + ctx->npt_rad, (size_t)ctx->npt_azim * sizeof(float),
                                     cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
    return AI_OK;
}

int ai_integrate1d_batch(ai_ctx *ctx, const void *frames, ai_dtype dtype, int nframes, int64_t frame_stride_elems,
                         const float *dark, const float *flat, const float *solidangle, const float *polarization,
                         const uint8_t *mask, float *intensity, float *sum_signal, float *count, void *cuda_stream)
{
    if (!ctx) return AI_EINVAL;
    FrameArgs a{frames, dtype, dark, flat, solidangle, polarization, mask, nullptr, intensity, sum_signal, count,
                nframes, frame_stride_elems};
    return integrate(ctx, a, (cudaStream_t)cuda_stream);
}

int ai_prepare_batch(ai_ctx *ctx, int max_frames, void *cuda_stream)
{
    if (!ctx) return AI_EINVAL;
    if (!ctx->built) return ai_fail(ctx, AI_ENOTBUILT, "ai_build_csr has not been called");
    if (max_frames < 1) return ai_fail(ctx, AI_EINVAL, "max_frames < 1");
    int dev = -1;
    AI_CUDA(ctx, cudaGetDevice(&dev));
    if (dev != ctx->device)
        return ai_fail(ctx, AI_EINVAL, "the matrix was built on device %d, the current device is %d", ctx->device, dev);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // partial records of the two-launch kernels (slice-per-lane batches, the general pipelined kernel)
    const size_t need = (size_t)(ctx->tl.nslot > 0 ? ctx->tl.nslot : 1) * 16 * (size_t)max_frames;
    if (ctx->partials_bytes < need) {
        if (ctx->partials) AI_CUDA(ctx, cudaFree(ctx->partials));
        ctx->partials = nullptr;
        ctx->partials_bytes = 0;
        AI_CUDA(ctx, cudaMalloc(&ctx->partials, need));
        ctx->partials_bytes = need;
    }
    // the two corrected frames of the pre-pass (frames of a batch that go one by one)
    const int pitch = (ctx->width + 3) / 4 * 4;
    for (int i = 0; i < 2; ++i)
        if (!ctx->corrected[i]) AI_CUDA(ctx, cudaMalloc(&ctx->corrected[i], (size_t)ctx->height * pitch * sizeof(float)));
    int rc = ai_prepare_fl(ctx, max_frames, st);
    if (rc != AI_OK) return rc;
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    return AI_OK;
}

int ai_integrate1d_host(ai_ctx *ctx, const void *image_host, ai_dtype dtype, const float *dark, const float *flat,
                        const float *solidangle, const float *polarization, const uint8_t *mask,
                        float *intensity_host, float *sum_signal_host, float *count_host, void *cuda_stream)
{
    if (!ctx) return AI_EINVAL;
    if (!ctx->built) return ai_fail(ctx, AI_ENOTBUILT, "ai_build_csr has not been called");
    if (!image_host || !intensity_host || !sum_signal_host || !count_host) return ai_fail(ctx, AI_EINVAL, "NULL image or output");
    if ((int)dtype < AI_F32 || (int)dtype > AI_U32) return ai_fail(ctx, AI_EINVAL, "bad dtype %d", (int)dtype);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t esz = (dtype == AI_U16 || dtype == AI_I16) ? 2 : 4;
    const size_t bytes = (size_t)ctx->height * ctx->width * esz;
    if (ctx->staging_bytes < bytes) {
        if (ctx->staging) AI_CUDA(ctx, cudaFree(ctx->staging));
        ctx->staging = nullptr;
        ctx->staging_bytes = 0;
        AI_CUDA(ctx, cudaMalloc(&ctx->staging, bytes));
        ctx->staging_bytes = bytes;
    }
    const size_t nb = (size_t)ctx->npt * sizeof(float);
    AI_CUDA(ctx, cudaMemcpyAsync(ctx->staging, image_host, bytes, cudaMemcpyHostToDevice, st));
    FrameArgs a{ctx->staging, dtype, dark, flat, solidangle, polarization, mask, nullptr, ctx->out_dev,
                ctx->out_dev + ctx->npt, ctx->out_dev + 2 * ctx->npt, 1, (int64_t)ctx->height * ctx->width};
    int rc = integrate(ctx, a, st);
    if (rc != AI_OK) return rc;
    // the three outputs are adjacent on the device; three copies because the host buffers are the caller's
    AI_CUDA(ctx, cudaMemcpyAsync(intensity_host, ctx->out_dev, nb, cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaMemcpyAsync(sum_signal_host, ctx->out_dev + ctx->npt, nb, cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaMemcpyAsync(count_host, ctx->out_dev + 2 * ctx->npt, nb, cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    return AI_OK;
}

int ai_integrate1d_host_frames(ai_ctx *ctx, const void *frames_host, ai_dtype dtype, int nframes,
                               int64_t frame_stride_elems, const float *dark, const float *flat,
                               const float *solidangle, const float *polarization, const uint8_t *mask,
                               float *intensity_host, float *sum_signal_host, float *count_host, void *cuda_stream)
{
    if (!ctx) return AI_EINVAL;
    if (!ctx->built) return ai_fail(ctx, AI_ENOTBUILT, "ai_build_csr has not been called");
    if (!frames_host || !intensity_host || !sum_signal_host || !count_host) return ai_fail(ctx, AI_EINVAL, "NULL frames or output");
    if ((int)dtype < AI_F32 || (int)dtype > AI_U32) return ai_fail(ctx, AI_EINVAL, "bad dtype %d", (int)dtype);
    if (nframes < 1) return ai_fail(ctx, AI_EINVAL, "nframes < 1");
    const int64_t npix = (int64_t)ctx->height * ctx->width;
    if (frame_stride_elems < npix) return ai_fail(ctx, AI_EINVAL, "frame stride < height*width");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t esz = (dtype == AI_U16 || dtype == AI_I16) ? 2 : 4;
    const size_t bytes = (size_t)npix * esz;
    if (!ctx->host_frames_ready) {           // set only once every resource exists (a failed attempt is retried)
        if (!ctx->copy_stream) AI_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            if (!ctx->h2d_done[i]) AI_CUDA(ctx, cudaEventCreateWithFlags(&ctx->h2d_done[i], cudaEventDisableTiming));
            if (!ctx->slot_free[i]) AI_CUDA(ctx, cudaEventCreateWithFlags(&ctx->slot_free[i], cudaEventDisableTiming));
        }
        ctx->host_frames_ready = true;
    }
    // Frames travel in chunks of up to kHostChunk: one upload per chunk into one of two staging buffers (the upload of
    // chunk k+1 overlaps the kernels of chunk k), ONE batched launch per chunk (ai_integrate1d_batch: the matrix is read
    // once per chunk), three downloads per chunk.
    constexpr int kHostChunk = 8;
    const int chunk = nframes < kHostChunk ? nframes : kHostChunk;
    const size_t chunk_bytes = bytes * chunk, out_floats = (size_t)ctx->npt * chunk;
    if (ctx->stage2_bytes < chunk_bytes || ctx->out2_floats < 3 * out_floats) {
        AI_CUDA(ctx, cudaStreamSynchronize(st));
        AI_CUDA(ctx, cudaStreamSynchronize(ctx->copy_stream));
        for (int i = 0; i < 2; ++i) {
            cudaFree(ctx->stage2[i]); cudaFree(ctx->out2[i]);
            ctx->stage2[i] = nullptr; ctx->out2[i] = nullptr;
        }
        ctx->stage2_bytes = 0;
        ctx->out2_floats = 0;
        for (int i = 0; i < 2; ++i) {
            AI_CUDA(ctx, cudaMalloc(&ctx->stage2[i], chunk_bytes));
            AI_CUDA(ctx, cudaMalloc(&ctx->out2[i], 3 * out_floats * sizeof(float)));
        }
        ctx->stage2_bytes = chunk_bytes;
        ctx->out2_floats = 3 * out_floats;
    }
    // uploads must not overtake work already queued on the caller's stream that may still use the staging buffers
    AI_CUDA(ctx, cudaEventRecord(ctx->slot_free[0], st));
    AI_CUDA(ctx, cudaEventRecord(ctx->slot_free[1], st));
    int rc = AI_OK;
    for (int k0 = 0, c = 0; k0 < nframes && rc == AI_OK; k0 += chunk, ++c) {
        const int slot = c & 1, n = nframes - k0 < chunk ? nframes - k0 : chunk;
        const char *src = static_cast<const char *>(frames_host) + (size_t)k0 * frame_stride_elems * esz;
        AI_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->slot_free[slot], 0));
        if (frame_stride_elems == npix) {
            AI_CUDA(ctx, cudaMemcpyAsync(ctx->stage2[slot], src, bytes * n, cudaMemcpyHostToDevice, ctx->copy_stream));
        } else {
            for (int q = 0; q < n; ++q)
                AI_CUDA(ctx, cudaMemcpyAsync(static_cast<char *>(ctx->stage2[slot]) + bytes * q,
                                             src + (size_t)q * frame_stride_elems * esz, bytes, cudaMemcpyHostToDevice,
                                             ctx->copy_stream));
        }
        AI_CUDA(ctx, cudaEventRecord(ctx->h2d_done[slot], ctx->copy_stream));
        AI_CUDA(ctx, cudaStreamWaitEvent(st, ctx->h2d_done[slot], 0));
        float *o = ctx->out2[slot];
        const size_t on = (size_t)ctx->npt * n;
        FrameArgs a{ctx->stage2[slot], dtype, dark, flat, solidangle, polarization, mask, nullptr, o, o + on, o + 2 * on, n, npix};
        rc = integrate(ctx, a, st);
        if (rc != AI_OK) break;
        AI_CUDA(ctx, cudaEventRecord(ctx->slot_free[slot], st));
        AI_CUDA(ctx, cudaMemcpyAsync(intensity_host + (size_t)k0 * ctx->npt, o, on * sizeof(float), cudaMemcpyDeviceToHost, st));
        AI_CUDA(ctx, cudaMemcpyAsync(sum_signal_host + (size_t)k0 * ctx->npt, o + on, on * sizeof(float), cudaMemcpyDeviceToHost, st));
        AI_CUDA(ctx, cudaMemcpyAsync(count_host + (size_t)k0 * ctx->npt, o + 2 * on, on * sizeof(float), cudaMemcpyDeviceToHost, st));
    }
    // also on failure: nothing of this call may still be writing the staging buffers when it returns
    cudaStreamSynchronize(ctx->copy_stream);
    if (rc != AI_OK) {
        cudaStreamSynchronize(st);
        return rc;
    }
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    return AI_OK;
}

// everything ai_build_csr and the integrate calls allocate on the device (and the host copies that go with it), freed and
// reset: ai_destroy, and ai_build_csr before it builds (a build that failed half-way leaves nothing behind)
static void release_matrix_and_scratch(ai_ctx *ctx)
{
    auto drop = [](auto *&p) { cudaFree(p); p = nullptr; };
    drop(ctx->indptr); drop(ctx->indices); drop(ctx->data); drop(ctx->row_csum); drop(ctx->d_range);
    drop(ctx->lut_coef); drop(ctx->lut_idx); drop(ctx->csr_seg); drop(ctx->csr_row_seg_ptr); drop(ctx->csr_partials);
    drop(ctx->scat_first_nb); drop(ctx->scat_gw); drop(ctx->norm_scratch);
    ctx->csr_partials_bytes = 0;
    ctx->csr_nseg = 0;
    ctx->lut_width = 0;
    TiledLayout &tl = ctx->tl;
    cudaFree(tl.tile_seg_ptr); cudaFree(tl.seg_ptr); cudaFree(tl.seg_slot); cudaFree(tl.seg_meta); cudaFree(tl.seg_csum);
    cudaFree(tl.tile_desc); cudaFree(tl.tile_order); cudaFree(tl.blob); cudaFree(tl.blob_desc);
    cudaFree(tl.tcoef); cudaFree(tl.tidx); cudaFree(tl.bin_slot_ptr);
    free(tl.h_first_desc);
    tl = TiledLayout{};
    free(ctx->stream_first);
    ctx->stream_first = nullptr;
    ctx->stream_first_grid = 0;
    ai_free_fl(ctx->fl);
    ai_release_held(ctx);
    drop(ctx->partials); drop(ctx->staging); drop(ctx->out_dev); drop(ctx->grid_sync); drop(ctx->chain_done);
    drop(ctx->stream_partials); drop(ctx->axes2d); drop(ctx->corrected[0]); drop(ctx->corrected[1]);
    ctx->partials_bytes = ctx->staging_bytes = 0;
    ctx->nnz = 0;
}

void ai_destroy(ai_ctx *ctx)
{
    if (!ctx) return;
    for (int i = 0; i < 2; ++i) {
        cudaFree(ctx->stage2[i]); cudaFree(ctx->out2[i]);
        if (ctx->h2d_done[i]) cudaEventDestroy(ctx->h2d_done[i]);
        if (ctx->slot_free[i]) cudaEventDestroy(ctx->slot_free[i]);
    }
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    release_matrix_and_scratch(ctx);
    if (ctx->ev0) cudaEventDestroy(ctx->ev0);
    if (ctx->ev1) cudaEventDestroy(ctx->ev1);
    delete ctx;
}

}  // extern "C"
