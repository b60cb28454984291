// One-time matrix build on the device: bounds -> range -> count -> scan -> ordered fill.
// The paper builds its look-up table single-threaded on the host; the coefficient definition is
// PAPER.md:120-122 (bounding-box pixel splitting), the CSR format PAPER.md:180, and the decomposition into map /
// reduction / scan kernels follows PAPER.md:142-153.
#include <math.h>

#include "build_common.cuh"
#include "ctx.h"

namespace {

// B1: bounds of every pixel's bounding box along the radial axis (PAPER.md:50 r = sqrt((x-xc)^2 + (y-yc)^2);
// PAPER.md:120 "rectangular box circumscribing the actual pixel") + block partials of the automatic range (B2).
__global__ void __launch_bounds__(256) bounds_kernel(ai_geometry g, int height, int width, int unit,
                                                     double *__restrict__ umin, double *__restrict__ umax,
                                                     double *__restrict__ part_lo, double *__restrict__ part_hi)
{
    const int64_t n = (int64_t)height * width;
    double lo = INFINITY, hi = -INFINITY;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
        int i = (int)(p / width), j = (int)(p - (int64_t)i * width);
        double x_lo = __dmul_rn(__dsub_rn((double)j, g.center_x_px), g.pixel_x_m);
        double x_hi = __dmul_rn(__dsub_rn((double)(j + 1), g.center_x_px), g.pixel_x_m);
        double y_lo = __dmul_rn(__dsub_rn((double)i, g.center_y_px), g.pixel_y_m);
        double y_hi = __dmul_rn(__dsub_rn((double)(i + 1), g.center_y_px), g.pixel_y_m);
        double nx = fmax(fmax(x_lo, -x_hi), 0.0);          // nearest point of the rectangle to the beam centre
        double ny = fmax(fmax(y_lo, -y_hi), 0.0);
        double fx = fmax(fabs(x_lo), fabs(x_hi));          // farthest corner
        double fy = fmax(fabs(y_lo), fabs(y_hi));
        double r_min = __dsqrt_rn(__dadd_rn(__dmul_rn(nx, nx), __dmul_rn(ny, ny)));
        double r_max = __dsqrt_rn(__dadd_rn(__dmul_rn(fx, fx), __dmul_rn(fy, fy)));
        double a = unit_of_r(r_min, g.distance_m, g.wavelength_m, unit);
        double z = unit_of_r(r_max, g.distance_m, g.wavelength_m, unit);
        umin[p] = a;
        umax[p] = z;
        lo = fmin(lo, a);
        hi = fmax(hi, z);
    }
    __shared__ double s_lo[8], s_hi[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if ((threadIdx.x & 31) == 0) { s_lo[threadIdx.x >> 5] = lo; s_hi[threadIdx.x >> 5] = hi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { lo = fmin(lo, s_lo[w]); hi = fmax(hi, s_hi[w]); }
        part_lo[blockIdx.x] = lo;
        part_hi[blockIdx.x] = hi;
    }
}

// B2 (reduction): u0 = min u_min, u1 = max u_max over all pixels.
__global__ void range_kernel(const double *__restrict__ part_lo, const double *__restrict__ part_hi, int nparts,
                             double *__restrict__ range)
{
    double lo = INFINITY, hi = -INFINITY;
    for (int k = threadIdx.x; k < nparts; k += blockDim.x) { lo = fmin(lo, part_lo[k]); hi = fmax(hi, part_hi[k]); }
    __shared__ double s_lo[32], s_hi[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if ((threadIdx.x & 31) == 0) { s_lo[threadIdx.x >> 5] = lo; s_hi[threadIdx.x >> 5] = hi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) { lo = fmin(lo, s_lo[w]); hi = fmax(hi, s_hi[w]); }
        range[0] = lo;
        range[1] = hi;
    }
}

// B3a (map): bounds in bin units f = (u - u0)/delta, first bin and number of bins of each pixel (in place over u).
__global__ void __launch_bounds__(256) span_kernel(int64_t n, int npt, const double *__restrict__ range,
                                                   double *__restrict__ fmin_a, double *__restrict__ fmax_a,
                                                   int *__restrict__ first_a, int *__restrict__ nb_a)
{
    const double u0 = range[0], u1 = range[1];
    const double delta = __ddiv_rn(__dsub_rn(u1, u0), (double)npt);
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
        double f_lo = __ddiv_rn(__dsub_rn(fmin_a[p], u0), delta);
        double f_hi = __ddiv_rn(__dsub_rn(fmax_a[p], u0), delta);
        int first, nb;
        split_span(f_lo, f_hi, npt, &first, &nb);
        fmin_a[p] = f_lo;
        fmax_a[p] = f_hi;
        first_a[p] = first;
        nb_a[p] = nb;
    }
}

// B3b (count): cnt[line][b] = number of pixels of image line `line` with an entry in bin b.  One block per line; the
// line's histogram is kept in shared memory when it fits, else counted with global integer atomics (cnt pre-zeroed).
__global__ void __launch_bounds__(256) count_lines_kernel(int width, int npt, const int *__restrict__ first_a,
                                                          const int *__restrict__ nb_a, int *__restrict__ cnt,
                                                          int use_smem)
{
    extern __shared__ int hist[];
    const int line = blockIdx.x;
    int *dst = cnt + (int64_t)line * npt;
    if (use_smem) {
        for (int b = threadIdx.x; b < npt; b += blockDim.x) hist[b] = 0;
        __syncthreads();
    }
    for (int j = threadIdx.x; j < width; j += blockDim.x) {
        int64_t p = (int64_t)line * width + j;
        int first = first_a[p], nb = nb_a[p];
        for (int b = first; b < first + nb; ++b) atomicAdd(use_smem ? &hist[b] : &dst[b], 1);
    }
    if (use_smem) {
        __syncthreads();
        for (int b = threadIdx.x; b < npt; b += blockDim.x) dst[b] = hist[b];
    }
}

// B4a (scan down the lines): cnt[line][b] <- number of entries of bin b in earlier lines; row_len[b] = total.
__global__ void __launch_bounds__(128) column_scan_kernel(int height, int npt, int *__restrict__ cnt,
                                                          long long *__restrict__ row_len)
{
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= npt) return;
    long long run = 0;
    int line = 0;
    for (; line + 8 <= height; line += 8) {
        int c[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) c[k] = cnt[(int64_t)(line + k) * npt + b];
#pragma unroll
        for (int k = 0; k < 8; ++k) { cnt[(int64_t)(line + k) * npt + b] = (int)run; run += c[k]; }
    }
    for (; line < height; ++line) {
        int c = cnt[(int64_t)line * npt + b];
        cnt[(int64_t)line * npt + b] = (int)run;
        run += c;
    }
    row_len[b] = run;
}

// B4b (scan): exclusive prefix sum of the row lengths -> indptr; total in 64 bits.  One block.
__global__ void __launch_bounds__(1024) indptr_scan_kernel(int npt, const long long *__restrict__ row_len,
                                                           int32_t *__restrict__ indptr, long long *__restrict__ total)
{
    __shared__ long long warp_sum[32];
    __shared__ long long carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int base = 0; base < npt; base += blockDim.x) {
        int b = base + threadIdx.x;
        long long v = b < npt ? row_len[b] : 0;
        long long x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            long long y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_sum[wid] = x;
        __syncthreads();
        if (wid == 0) {
            long long w = warp_sum[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                long long y = __shfl_up_sync(0xffffffffu, w, o);
                if (lane >= o) w += y;
            }
            warp_sum[lane] = w;      // inclusive over warps
        }
        __syncthreads();
        long long before = carry + (wid > 0 ? warp_sum[wid - 1] : 0) + (x - v);
        if (b < npt) indptr[b] = (int32_t)before;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry = before + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        *total = carry;
        indptr[npt] = (int32_t)carry;
    }
}

// B5 (ordered fill): one warp per image line.
struct LineChunk {
    int line, width, npt;
    const int32_t *indptr;
    int *cnt_line;
    int32_t *indices;
    float *data;
    __device__ int npix() const { return width; }
    __device__ bool pixel(int k, int64_t *p) const { *p = (int64_t)line * width + k; return true; }
    __device__ int base(int b) const { return indptr[b]; }
    __device__ volatile int *cursor(int b) const { return cnt_line + b; }
    __device__ int64_t place(int, int64_t pos) const { return pos; }      // canonical CSR: ascending pixel order
    __device__ void emit(int64_t pos, int, int64_t p, float coef) const { indices[pos] = (int32_t)p; data[pos] = coef; }
};

__global__ void __launch_bounds__(128) fill_lines_kernel(int height, int width, int npt,
                                                         const double *__restrict__ fmin_a,
                                                         const double *__restrict__ fmax_a,
                                                         const int *__restrict__ first_a, const int *__restrict__ nb_a,
                                                         const int32_t *__restrict__ indptr, int *cnt,
                                                         int32_t *__restrict__ indices, float *__restrict__ data)
{
    int line = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (line >= height) return;
    LineChunk ch{line, width, npt, indptr, cnt + (int64_t)line * npt, indices, data};
    marching_fill(ch, fmin_a, fmax_a, first_a, nb_a, npt);
}

// sum of each row's coefficients in fp64, fixed order (one warp per row)
__global__ void __launch_bounds__(256) row_sum_kernel(int npt, const int32_t *__restrict__ indptr,
                                                      const float *__restrict__ data, float *__restrict__ row_csum)
{
    int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (b >= npt) return;
    double s = 0.0;
    for (int k = indptr[b] + (threadIdx.x & 31); k < indptr[b + 1]; k += 32) s += (double)data[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) row_csum[b] = (float)s;
}

// B6: padded look-up table, row-major: entry j of bin b at [b * lut_width + j]; padding has
// coefficient 0 and index 0.
__global__ void __launch_bounds__(256) lut_kernel(int npt, int lut_width, const int32_t *__restrict__ indptr,
                                                  const int32_t *__restrict__ indices, const float *__restrict__ data,
                                                  float *__restrict__ lut_coef, int32_t *__restrict__ lut_idx)
{
    int64_t total = (int64_t)npt * lut_width;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        int b = (int)(e / lut_width), j = (int)(e - (int64_t)b * lut_width);
        int k = indptr[b] + j;
        bool in = k < indptr[b + 1];
        lut_coef[e] = in ? data[k] : 0.0f;
        lut_idx[e] = in ? indices[k] : 0;
    }
}

__global__ void max_row_len_kernel(int npt, const int32_t *__restrict__ indptr, int *__restrict__ out)
{
    int m = 0;
    for (int b = threadIdx.x; b < npt; b += blockDim.x) m = max(m, indptr[b + 1] - indptr[b]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(out, m);
}

}  // namespace

void ai_free_spans(PixelSpans *s)
{
    cudaFree(s->fmin); cudaFree(s->fmax); cudaFree(s->first); cudaFree(s->nb);
    *s = PixelSpans{};
}

// B1-B3a: bounds of every pixel on the radial axis, the range, and the pixel's first bin / number of bins for `npt` bins
int ai_build_spans(ai_ctx *ctx, PixelSpans *sp, int npt, cudaStream_t st)
{
    const int H = ctx->height, W = ctx->width;
    const int64_t n = (int64_t)H * W;
    AI_CUDA(ctx, cudaMalloc(&sp->fmin, n * sizeof(double)));
    AI_CUDA(ctx, cudaMalloc(&sp->fmax, n * sizeof(double)));
    AI_CUDA(ctx, cudaMalloc(&sp->first, n * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&sp->nb, n * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&ctx->d_range, 2 * sizeof(double)));

    const int nblk = (int)((n + 255) / 256 < 4 * 148 * 8 ? (n + 255) / 256 : 4 * 148 * 8);
    double *parts = nullptr;
    AI_CUDA(ctx, cudaMalloc(&parts, 2 * (size_t)nblk * sizeof(double)));
    bounds_kernel<<<nblk, 256, 0, st>>>(ctx->geo, H, W, (int)ctx->unit, sp->fmin, sp->fmax, parts, parts + nblk);
    if (ctx->user_range) {
        AI_CUDA(ctx, cudaMemcpyAsync(ctx->d_range, ctx->range_host, 2 * sizeof(double), cudaMemcpyHostToDevice, st));
    } else {
        range_kernel<<<1, 1024, 0, st>>>(parts, parts + nblk, nblk, ctx->d_range);
    }
    span_kernel<<<nblk, 256, 0, st>>>(n, npt, ctx->d_range, sp->fmin, sp->fmax, sp->first, sp->nb);
    AI_CUDA(ctx, cudaGetLastError());
    AI_CUDA(ctx, cudaMemcpyAsync(ctx->range_host, ctx->d_range, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    cudaFree(parts);
    return AI_OK;
}

int ai_build_canonical(ai_ctx *ctx, PixelSpans *sp, cudaStream_t st)
{
    const int H = ctx->height, W = ctx->width, npt = ctx->npt;
    int rc = ai_build_spans(ctx, sp, npt, st);
    if (rc != AI_OK) return rc;

    int *cnt = nullptr;
    long long *row_len = nullptr;      // [npt] lengths, then [1] total
    AI_CUDA(ctx, cudaMalloc(&cnt, (size_t)H * npt * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&row_len, ((size_t)npt + 1) * sizeof(long long)));
    AI_CUDA(ctx, cudaMalloc(&ctx->indptr, ((size_t)npt + 1) * sizeof(int32_t)));
    const size_t hist_bytes = (size_t)npt * sizeof(int);
    const int use_smem = hist_bytes <= 160 * 1024;
    if (use_smem && hist_bytes > 48 * 1024)
        AI_CUDA(ctx, cudaFuncSetAttribute(count_lines_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)hist_bytes));
    if (!use_smem) AI_CUDA(ctx, cudaMemsetAsync(cnt, 0, (size_t)H * npt * sizeof(int), st));
    count_lines_kernel<<<H, 256, use_smem ? hist_bytes : 0, st>>>(W, npt, sp->first, sp->nb, cnt, use_smem);
    column_scan_kernel<<<(npt + 127) / 128, 128, 0, st>>>(H, npt, cnt, row_len);
    indptr_scan_kernel<<<1, 1024, 0, st>>>(npt, row_len, ctx->indptr, row_len + npt);
    AI_CUDA(ctx, cudaGetLastError());

    long long total = 0;
    AI_CUDA(ctx, cudaMemcpyAsync(&total, row_len + npt, sizeof(long long), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));      // nnz sizes the matrix
    if (total > 0x7fffffffLL) {
        cudaFree(cnt); cudaFree(row_len);
        return ai_fail(ctx, AI_EUNSUPPORTED, "matrix has %lld entries, more than int32 row pointers can address", total);
    }
    ctx->nnz = total;
    const size_t alloc = total > 0 ? (size_t)total : 1;
    AI_CUDA(ctx, cudaMalloc(&ctx->indices, alloc * sizeof(int32_t)));
    AI_CUDA(ctx, cudaMalloc(&ctx->data, alloc * sizeof(float)));
    AI_CUDA(ctx, cudaMalloc(&ctx->row_csum, (size_t)npt * sizeof(float)));
    fill_lines_kernel<<<(H + 3) / 4, 128, 0, st>>>(H, W, npt, sp->fmin, sp->fmax, sp->first, sp->nb, ctx->indptr, cnt,
                                                   ctx->indices, ctx->data);
    row_sum_kernel<<<(npt + 7) / 8, 256, 0, st>>>(npt, ctx->indptr, ctx->data, ctx->row_csum);
    AI_CUDA(ctx, cudaGetLastError());
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    cudaFree(cnt); cudaFree(row_len);
    return AI_OK;
}

int ai_build_lut(ai_ctx *ctx, cudaStream_t st)
{
    if (ctx->lut_coef) return AI_OK;
    int *d_max = nullptr, h_max = 0;
    AI_CUDA(ctx, cudaMalloc(&d_max, sizeof(int)));
    AI_CUDA(ctx, cudaMemsetAsync(d_max, 0, sizeof(int), st));
    max_row_len_kernel<<<1, 1024, 0, st>>>(ctx->npt, ctx->indptr, d_max);
    AI_CUDA(ctx, cudaMemcpyAsync(&h_max, d_max, sizeof(int), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    cudaFree(d_max);
    ctx->lut_width = h_max > 0 ? (h_max + 3) / 4 * 4 : 4;      // rows start on 16-byte boundaries
    const size_t total = (size_t)ctx->npt * ctx->lut_width;
    size_t free_b = 0, total_b = 0;
    AI_CUDA(ctx, cudaMemGetInfo(&free_b, &total_b));
    if (total * 8 > free_b / 2)
        return ai_fail(ctx, AI_EUNSUPPORTED, "padded LUT of %zu bytes does not fit in device memory", total * 8);
    AI_CUDA(ctx, cudaMalloc(&ctx->lut_coef, total * sizeof(float)));
    AI_CUDA(ctx, cudaMalloc(&ctx->lut_idx, total * sizeof(int32_t)));
    lut_kernel<<<148 * 8, 256, 0, st>>>(ctx->npt, ctx->lut_width, ctx->indptr, ctx->indices, ctx->data, ctx->lut_coef,
                                        ctx->lut_idx);
    AI_CUDA(ctx, cudaGetLastError());
    return AI_OK;
}
