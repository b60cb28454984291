// One-time build of the BIDIMENSIONAL ("cake") matrix: bins = azimuthal x radial ("mono- and bidimensional
// integration"; PAPER.md:114-116 and Fig. 3: the case where pixel splitting matters most).  Row b = a * npt_rad + r.
//
// The weight of pixel p in bin (a, r) is the bounding box of PAPER.md:120 taken on both axes: the pixel's extent along
// the radial unit (as in 1D, build_csr.cu) times its extent along chi = atan2(y, x), each split over its
// bins by overlap / width.  The azimuthal axis is periodic: a pixel that crosses the negative x axis is split across the
// seam, a pixel that holds the beam centre strictly inside covers the full circle (readings).
//
// A pixel's bins are no longer one contiguous range, so the count -> scan -> ordered-fill scheme of the 1D builder
// (one counter per image line and bin) does not carry over.  Here: count per pixel -> exclusive scan -> emit
// (key, coefficient) pairs -> radix sort by key.  Sorted by (bin, pixel) the pairs ARE the canonical CSR, columns
// ascending; sorted by (tile, bin, position in the tile) they are the tiled layout's segments, which then go through the
// same slicing into blobs as in 1D (build_sliced.cu).  The sort and the scans are CUB's device-wide primitives (this is
// the one-time build; the per-frame kernels are the library's own).  Deterministic: keys are unique.
#include <cub/cub.cuh>

#include <algorithm>
#include <vector>

#include "build_common.cuh"
#include "ctx.h"
#include "tiled_build_common.cuh"

struct SliceScratch;
int ai_build_spans(ai_ctx *ctx, PixelSpans *sp, int npt, cudaStream_t st);
int ai_slice_max_blob(ai_ctx *ctx, int ntiles, const int *tile_seg_ptr, const int *seg_len, cudaStream_t st, int *max_blob);
int ai_build_sliced_plan(ai_ctx *ctx, SliceScratch *sc, int *seg_nruns, cudaStream_t st);
int ai_build_sliced_fill(ai_ctx *ctx, SliceScratch *sc, cudaStream_t st);
SliceScratch *ai_slice_scratch_new();
void ai_slice_scratch_delete(SliceScratch *sc);

namespace {

constexpr double kPi = 3.14159265358979323846;
constexpr double kTwoPi = 2.0 * kPi;

// Azimuthal extent of pixel (i, j): start in [-pi, pi) and width in [0, 2 pi]; the pixel covers [lo, lo + w], which may
// run past +pi.  Corner angles are measured from the direction of the pixel centre (signed angle atan2(cross, dot)), a
// corner on the beam centre has no direction.  Plain fp64, every operation rounded once.
__device__ __forceinline__ void chi_extent(const ai_geometry &g, int i, int j, double *lo, double *w)
{
    const double x_lo = __dmul_rn(__dsub_rn((double)j, g.center_x_px), g.pixel_x_m);
    const double x_hi = __dmul_rn(__dsub_rn((double)(j + 1), g.center_x_px), g.pixel_x_m);
    const double y_lo = __dmul_rn(__dsub_rn((double)i, g.center_y_px), g.pixel_y_m);
    const double y_hi = __dmul_rn(__dsub_rn((double)(i + 1), g.center_y_px), g.pixel_y_m);
    if (x_lo < 0.0 && x_hi > 0.0 && y_lo < 0.0 && y_hi > 0.0) {
        *lo = -kPi;
        *w = kTwoPi;
        return;
    }
    const double xc = __dmul_rn(0.5, __dadd_rn(x_lo, x_hi)), yc = __dmul_rn(0.5, __dadd_rn(y_lo, y_hi));
    const double chi_c = atan2(yc, xc);
    double d_min = 0.0, d_max = 0.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double x = (k & 1) ? x_hi : x_lo, y = (k & 2) ? y_hi : y_lo;
        if (x == 0.0 && y == 0.0) continue;
        const double d = atan2(__dsub_rn(__dmul_rn(xc, y), __dmul_rn(yc, x)), __dadd_rn(__dmul_rn(xc, x), __dmul_rn(yc, y)));
        d_min = fmin(d_min, d);
        d_max = fmax(d_max, d);
    }
    double a = __dadd_rn(chi_c, d_min);
    if (a < -kPi) a = __dadd_rn(a, kTwoPi);
    if (a >= kPi) a = __dsub_rn(a, kTwoPi);
    *lo = a;
    *w = __dsub_rn(d_max, d_min);
}

// The images of [lo, lo + w] shifted by -2 pi, 0, +2 pi that meet the range [c0, c0 + npt * delta], in bin units.
struct AzimPieces {
    double f_lo[3], f_hi[3];
    int first[3], nb[3];
    int n;
};
__device__ __forceinline__ void azim_pieces(double lo, double w, double c0, double delta, int npt, AzimPieces *out)
{
    out->n = 0;
    if (w >= kTwoPi) {       // the pixel holds the beam centre: every bin of the range, weight = bin width / 2 pi
        out->f_lo[0] = 0.0;
        out->f_hi[0] = __ddiv_rn(kTwoPi, delta);      // only the WIDTH is used: overlap of a whole bin is 1
        out->first[0] = 0;
        out->nb[0] = npt;
        out->n = -1;
        return;
    }
    for (int k = -1; k <= 1; ++k) {
        const double s = __dmul_rn(kTwoPi, (double)k);
        const double f_lo = __ddiv_rn(__dsub_rn(__dadd_rn(lo, s), c0), delta);
        const double f_hi = __ddiv_rn(__dsub_rn(__dadd_rn(__dadd_rn(lo, w), s), c0), delta);
        int first, nb;
        split_span(f_lo, f_hi, npt, &first, &nb);
        if (nb > 0) {
            const int q = out->n++;
            out->f_lo[q] = f_lo; out->f_hi[q] = f_hi; out->first[q] = first; out->nb[q] = nb;
        }
    }
    // One azimuthal bin over the full circle: the two images of a pixel across the seam fall into the same bin and would
    // be two entries with one (bin, pixel) key.  They become one piece with the overlap of both: [ov - w, ov] in bin units
    // has overlap ov (<= w) with bin 0 and width w.  With two bins or more the images land in different bins.
    if (npt == 1 && out->n > 1) {
        const double wf = __dsub_rn(out->f_hi[0], out->f_lo[0]);
        double ov = 0.0;
        for (int q = 0; q < out->n; ++q) ov = __dadd_rn(ov, split_overlap(out->f_lo[q], out->f_hi[q], 0, 1));
        out->f_hi[0] = ov;
        out->f_lo[0] = __dsub_rn(ov, wf);
        out->first[0] = 0;
        out->nb[0] = 1;
        out->n = 1;
    }
}

__global__ void __launch_bounds__(256) chi_kernel(ai_geometry g, int height, int width, double *__restrict__ chi_lo,
                                                  double *__restrict__ chi_w)
{
    const int64_t n = (int64_t)height * width;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(p / width), j = (int)(p - (int64_t)i * width);
        chi_extent(g, i, j, chi_lo + p, chi_w + p);
    }
}

// entries of every pixel = (radial bins) x (azimuthal bins)
__global__ void __launch_bounds__(256) count2d_kernel(int64_t n, const int *__restrict__ nb_r,
                                                      const double *__restrict__ chi_lo, const double *__restrict__ chi_w,
                                                      double c0, double delta, int npt_azim, long long *__restrict__ cnt)
{
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
        AzimPieces az;
        azim_pieces(chi_lo[p], chi_w[p], c0, delta, npt_azim, &az);
        int na = 0;
        for (int q = 0; q < (az.n < 0 ? 1 : az.n); ++q) na += az.nb[q];
        cnt[p] = (long long)na * nb_r[p];
    }
}

// key = bin << 32 | pixel (canonical CSR order), coefficient = azimuthal weight x radial weight
__global__ void __launch_bounds__(256) emit2d_kernel(int64_t n, int npt_rad, int npt_azim, const double *__restrict__ fmin_r,
                                                     const double *__restrict__ fmax_r, const int *__restrict__ first_r,
                                                     const int *__restrict__ nb_r, const double *__restrict__ chi_lo,
                                                     const double *__restrict__ chi_w, double c0, double delta,
                                                     const long long *__restrict__ offset,
                                                     unsigned long long *__restrict__ keys, float *__restrict__ vals)
{
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
        const int nr = nb_r[p];
        if (nr == 0) continue;
        AzimPieces az;
        azim_pieces(chi_lo[p], chi_w[p], c0, delta, npt_azim, &az);
        const double f_lo = fmin_r[p], f_hi = fmax_r[p];
        const int r0 = first_r[p];
        long long at = offset[p];
        for (int q = 0; q < (az.n < 0 ? 1 : az.n); ++q) {
            for (int a = az.first[q]; a < az.first[q] + az.nb[q]; ++a) {
                const double ca = az.n < 0 ? __ddiv_rn(1.0, az.f_hi[0]) : split_coefficient(az.f_lo[q], az.f_hi[q], a, npt_azim);
                for (int r = r0; r < r0 + nr; ++r) {
                    const double cr = split_coefficient(f_lo, f_hi, r, npt_rad);
                    keys[at] = ((unsigned long long)((long long)a * npt_rad + r) << 32) | (unsigned long long)p;
                    vals[at] = (float)__dmul_rn(ca, cr);
                    ++at;
                }
            }
        }
    }
}

// first index whose (key >> shift) is >= b, for b = 0 .. nb
__global__ void __launch_bounds__(256) lower_bound_kernel(const unsigned long long *__restrict__ keys, long long n, int shift,
                                                          int nb, int *__restrict__ out)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b > nb) return;
    long long lo = 0, hi = n;
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if ((long long)(keys[mid] >> shift) < (long long)b) lo = mid + 1;
        else hi = mid;
    }
    out[b] = (int)lo;
}

__global__ void __launch_bounds__(256) csr_unpack_kernel(long long n, const unsigned long long *__restrict__ keys,
                                                         int32_t *__restrict__ indices)
{
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x)
        indices[k] = (int32_t)(keys[k] & 0xffffffffULL);
}

// key2 = tile << 44 | bin << 16 | byte offset of the pixel in the tile buffer
__global__ void __launch_bounds__(256) tile_key_kernel(long long n, int width, int th, int tiles_x,
                                                       const unsigned long long *__restrict__ keys,
                                                       unsigned long long *__restrict__ keys2)
{
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) {
        const unsigned long long key = keys[k];
        const long long p = (long long)(key & 0xffffffffULL), bin = (long long)(key >> 32);
        const int i = (int)(p / width), j = (int)(p - (long long)i * width);
        const long long tile = (long long)(i / th) * tiles_x + j / kTileW;
        const unsigned pos = (unsigned)ai_tile_pos(i % th, j % kTileW, th) * 4u;
        keys2[k] = ((unsigned long long)tile << 44) | ((unsigned long long)bin << 16) | pos;
    }
}

__global__ void __launch_bounds__(256) seg_head_kernel(long long n, const unsigned long long *__restrict__ keys2,
                                                       long long *__restrict__ head)
{
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x)
        head[k] = (k == 0 || (keys2[k] >> 16) != (keys2[k - 1] >> 16)) ? 1 : 0;
}

// per segment: first entry and (tile << 28 | bin); seg_id = exclusive scan of the head flags
__global__ void __launch_bounds__(256) seg_first_kernel(long long n, const unsigned long long *__restrict__ keys2,
                                                        const long long *__restrict__ head,
                                                        const long long *__restrict__ seg_id, int *__restrict__ seg_first,
                                                        unsigned long long *__restrict__ seg_key)
{
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x)
        if (head[k]) {
            seg_first[seg_id[k]] = (int)k;
            seg_key[seg_id[k]] = keys2[k] >> 16;
        }
}

__global__ void __launch_bounds__(256) seg_len_kernel(int nseg, long long n, const int *__restrict__ seg_first,
                                                      int *__restrict__ seg_len)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < nseg) seg_len[s] = (int)((s + 1 < nseg ? (long long)seg_first[s + 1] : n) - seg_first[s]);
}

// entries into their (padded) segments, in sorted order: position in the tile ascending
__global__ void __launch_bounds__(256) seg_scatter_kernel(long long n, const unsigned long long *__restrict__ keys2,
                                                          const float *__restrict__ vals,
                                                          const long long *__restrict__ head,
                                                          const long long *__restrict__ seg_id,
                                                          const int *__restrict__ seg_first, const int *__restrict__ seg_ptr,
                                                          float *__restrict__ tcoef, uint16_t *__restrict__ tidx)
{
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) {
        const long long s = seg_id[k] - (head[k] ? 0 : 1);       // exclusive scan: a non-head entry sees the next id
        const long long dst = (long long)seg_ptr[s] + (k - seg_first[s]);
        tcoef[dst] = vals[k];
        tidx[dst] = (uint16_t)(keys2[k] & 0xffffULL);
    }
}

// slot assignment: segments sorted by (bin, segment index) -- the segment index ascends with the tile
__global__ void __launch_bounds__(256) slot_key_kernel(int nseg, const unsigned long long *__restrict__ seg_key,
                                                       unsigned long long *__restrict__ keys3)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < nseg) keys3[s] = ((seg_key[s] & 0xfffffffULL) << 32) | (unsigned long long)s;
}
__global__ void __launch_bounds__(256) slot_runs_kernel(int nseg, const unsigned long long *__restrict__ keys3,
                                                        const int *__restrict__ seg_nruns, long long *__restrict__ runs)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nseg) runs[i] = seg_nruns[(int)(keys3[i] & 0xffffffffULL)];
}
__global__ void __launch_bounds__(256) slot_assign_kernel(int nseg, const unsigned long long *__restrict__ keys3,
                                                          const long long *__restrict__ prefix, int *__restrict__ seg_slot)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nseg) seg_slot[(int)(keys3[i] & 0xffffffffULL)] = (int)prefix[i];
}
__global__ void __launch_bounds__(256) bin_slot_kernel(int nbins, int nseg, const int *__restrict__ bin_first,
                                                       const long long *__restrict__ prefix, long long total,
                                                       int *__restrict__ bin_slot_ptr)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b <= nbins) bin_slot_ptr[b] = bin_first[b] < nseg ? (int)prefix[bin_first[b]] : (int)total;
}

int bits_for(long long v)
{
    int b = 1;
    while ((1LL << b) <= v && b < 62) ++b;
    return b;
}

// device-wide primitives with their temporary storage
struct Scratch {
    void *tmp = nullptr;
    size_t bytes = 0;
    cudaError_t need(size_t b)
    {
        if (b <= bytes) return cudaSuccess;
        cudaFree(tmp);
        tmp = nullptr;
        bytes = 0;
        cudaError_t e = cudaMalloc(&tmp, b);
        if (e == cudaSuccess) bytes = b;
        return e;
    }
    ~Scratch() { cudaFree(tmp); }
};

cudaError_t exclusive_sum(Scratch &sc, const long long *in, long long *out, long long n, cudaStream_t st)
{
    size_t b = 0;
    cudaError_t e = cub::DeviceScan::ExclusiveSum(nullptr, b, in, out, n, st);
    if (e != cudaSuccess) return e;
    if ((e = sc.need(b)) != cudaSuccess) return e;
    return cub::DeviceScan::ExclusiveSum(sc.tmp, b, in, out, n, st);
}

cudaError_t sort_pairs(Scratch &sc, const unsigned long long *kin, unsigned long long *kout, const float *vin, float *vout,
                       long long n, int end_bit, cudaStream_t st)
{
    size_t b = 0;
    cudaError_t e = cub::DeviceRadixSort::SortPairs(nullptr, b, kin, kout, vin, vout, n, 0, end_bit, st);
    if (e != cudaSuccess) return e;
    if ((e = sc.need(b)) != cudaSuccess) return e;
    return cub::DeviceRadixSort::SortPairs(sc.tmp, b, kin, kout, vin, vout, n, 0, end_bit, st);
}

cudaError_t sort_keys(Scratch &sc, const unsigned long long *kin, unsigned long long *kout, long long n, int end_bit,
                      cudaStream_t st)
{
    size_t b = 0;
    cudaError_t e = cub::DeviceRadixSort::SortKeys(nullptr, b, kin, kout, n, 0, end_bit, st);
    if (e != cudaSuccess) return e;
    if ((e = sc.need(b)) != cudaSuccess) return e;
    return cub::DeviceRadixSort::SortKeys(sc.tmp, b, kin, kout, n, 0, end_bit, st);
}

template <class T> struct DevBuf {       // freed on every return path
    T *p = nullptr;
    cudaError_t alloc(size_t n) { return cudaMalloc(&p, (n > 0 ? n : 1) * sizeof(T)); }
    ~DevBuf() { cudaFree(p); }
};

}  // namespace

// From the unsorted entries (key = bin << 32 | pixel, coefficient) to the canonical CSR and the tiled + sliced execution
// layout.  keys_a / vals_a hold the entries; keys_b / vals_b are work buffers of the same size.
static int entries_to_layouts(ai_ctx *ctx, Scratch &scr, unsigned long long *keys_a_p, unsigned long long *keys_b_p,
                              float *vals_a_p, float *vals_b_p, long long nnz, long long nbins, cudaStream_t st)
{
    const int H = ctx->height, W = ctx->width;
    TiledLayout &tl = ctx->tl;
    const int grid = 148 * 8;
    int rc = AI_OK;
    struct { unsigned long long *p; } keys_a{keys_a_p}, keys_b{keys_b_p};
    struct { float *p; } vals_a{vals_a_p}, vals_b{vals_b_p};
    (void)H;
    AI_CUDA(ctx, sort_pairs(scr, keys_a.p, keys_b.p, vals_a.p, vals_b.p, nnz, 32 + bits_for(nbins), st));
    const size_t nnz_alloc = nnz > 0 ? (size_t)nnz : 1;
    AI_CUDA(ctx, cudaMalloc(&ctx->indptr, ((size_t)nbins + 1) * sizeof(int32_t)));
    AI_CUDA(ctx, cudaMalloc(&ctx->indices, nnz_alloc * sizeof(int32_t)));
    AI_CUDA(ctx, cudaMalloc(&ctx->data, nnz_alloc * sizeof(float)));
    lower_bound_kernel<<<(int)((nbins + 256) / 256), 256, 0, st>>>(keys_b.p, nnz, 32, (int)nbins, ctx->indptr);
    csr_unpack_kernel<<<grid, 256, 0, st>>>(nnz, keys_b.p, ctx->indices);
    AI_CUDA(ctx, cudaMemcpyAsync(ctx->data, vals_b.p, (size_t)nnz * sizeof(float), cudaMemcpyDeviceToDevice, st));
    AI_CUDA(ctx, cudaGetLastError());

    // ---- the tiled layout: largest tile height whose largest blob fits the shared-memory ring ------------------------------
    DevBuf<long long> head, seg_id;
    DevBuf<int> seg_first, seg_len, tile_entries;
    DevBuf<unsigned long long> seg_key;
    AI_CUDA(ctx, head.alloc(nnz + 1));
    AI_CUDA(ctx, seg_id.alloc(nnz + 1));
    long long nseg = 0;
    int th0 = kTileHMax;
    while (th0 > 8 && th0 > ctx->tune.tile_h_max) th0 /= 2;
    for (int th = th0;; th /= 2) {
        tl.tile_h = th;
        tl.tiles_y = (H + th - 1) / th;
        tl.tiles_x = (W + kTileW - 1) / kTileW;
        tl.ntiles = tl.tiles_y * tl.tiles_x;
        if (tl.ntiles >= (1 << 20)) return ai_fail(ctx, AI_EUNSUPPORTED, "%d tiles: more than 2^20", tl.ntiles);
        // (tile, bin, position) order; keys_b / vals_b keep the CSR order for the next try
        tile_key_kernel<<<grid, 256, 0, st>>>(nnz, W, th, tl.tiles_x, keys_b.p, keys_a.p);
        DevBuf<unsigned long long> keys2;
        DevBuf<float> vals2;
        AI_CUDA(ctx, keys2.alloc(nnz));
        AI_CUDA(ctx, vals2.alloc(nnz));
        AI_CUDA(ctx, sort_pairs(scr, keys_a.p, keys2.p, vals_b.p, vals2.p, nnz, 44 + bits_for(tl.ntiles), st));
        AI_CUDA(ctx, cudaMemsetAsync(head.p + nnz, 0, sizeof(long long), st));
        seg_head_kernel<<<grid, 256, 0, st>>>(nnz, keys2.p, head.p);
        AI_CUDA(ctx, cudaGetLastError());
        AI_CUDA(ctx, exclusive_sum(scr, head.p, seg_id.p, nnz + 1, st));
        AI_CUDA(ctx, cudaMemcpyAsync(&nseg, seg_id.p + nnz, sizeof(long long), cudaMemcpyDeviceToHost, st));
        AI_CUDA(ctx, cudaStreamSynchronize(st));
        if (nseg > 0x7fffffffLL) return ai_fail(ctx, AI_EUNSUPPORTED, "%lld (tile, bin) segments", nseg);
        tl.nseg = (int)nseg;
        const size_t nseg_alloc = nseg > 0 ? (size_t)nseg : 1;
        cudaFree(seg_first.p); cudaFree(seg_len.p); cudaFree(seg_key.p); cudaFree(tile_entries.p); cudaFree(tl.tile_seg_ptr);
        seg_first.p = seg_len.p = tile_entries.p = nullptr; seg_key.p = nullptr; tl.tile_seg_ptr = nullptr;
        AI_CUDA(ctx, seg_first.alloc(nseg_alloc));
        AI_CUDA(ctx, seg_len.alloc(nseg_alloc));
        AI_CUDA(ctx, seg_key.alloc(nseg_alloc));
        AI_CUDA(ctx, tile_entries.alloc(tl.ntiles));
        AI_CUDA(ctx, cudaMalloc(&tl.tile_seg_ptr, ((size_t)tl.ntiles + 1) * sizeof(int)));
        seg_first_kernel<<<grid, 256, 0, st>>>(nnz, keys2.p, head.p, seg_id.p, seg_first.p, seg_key.p);
        seg_len_kernel<<<(tl.nseg + 255) / 256 + 1, 256, 0, st>>>(tl.nseg, nnz, seg_first.p, seg_len.p);
        lower_bound_kernel<<<(tl.ntiles + 256) / 256, 256, 0, st>>>(seg_key.p, nseg, 28, tl.ntiles, tl.tile_seg_ptr);
        pad_segments_kernel<<<(tl.ntiles + 127) / 128, 128, 0, st>>>(tl.ntiles, tl.tile_seg_ptr, seg_len.p, tile_entries.p);
        AI_CUDA(ctx, cudaGetLastError());
        int max_blob = 0;
        rc = ai_slice_max_blob(ctx, tl.ntiles, tl.tile_seg_ptr, seg_len.p, st, &max_blob);
        if (rc != AI_OK) return rc;
        const bool fits = ai_pipe_plan(max_blob, th, false, ctx->tune).fits;
        if (!fits && th > 8) continue;

        // padded segment starts, entries scattered into place
        DevBuf<long long> d_total;
        long long h_total = 0;
        AI_CUDA(ctx, d_total.alloc(1));
        AI_CUDA(ctx, cudaMalloc(&tl.seg_ptr, (nseg_alloc + 1) * sizeof(int)));
        AI_CUDA(ctx, cudaMalloc(&tl.seg_slot, nseg_alloc * sizeof(int)));
        AI_CUDA(ctx, cudaMalloc(&tl.seg_csum, nseg_alloc * sizeof(double)));
        scan_pad_kernel<<<1, 1024, 0, st>>>(tl.nseg, seg_len.p, 1, tl.seg_ptr, d_total.p);
        AI_CUDA(ctx, cudaMemcpyAsync(&h_total, d_total.p, sizeof(long long), cudaMemcpyDeviceToHost, st));
        AI_CUDA(ctx, cudaStreamSynchronize(st));
        if (h_total > 0x7fffffffLL) return ai_fail(ctx, AI_EUNSUPPORTED, "tiled layout has %lld entries", h_total);
        tl.tnnz = h_total;
        const size_t tn = h_total > 0 ? (size_t)h_total : 1;
        AI_CUDA(ctx, cudaMalloc(&tl.tcoef, tn * sizeof(float)));
        AI_CUDA(ctx, cudaMalloc(&tl.tidx, tn * sizeof(uint16_t)));
        AI_CUDA(ctx, cudaMemsetAsync(tl.tcoef, 0, tn * sizeof(float), st));
        AI_CUDA(ctx, cudaMemsetAsync(tl.tidx, 0, tn * sizeof(uint16_t), st));
        seg_scatter_kernel<<<grid, 256, 0, st>>>(nnz, keys2.p, vals2.p, head.p, seg_id.p, seg_first.p, tl.seg_ptr, tl.tcoef,
                                                 tl.tidx);
        if (tl.nseg > 0) seg_sum_kernel<<<(tl.nseg + 7) / 8, 256, 0, st>>>(tl.nseg, tl.seg_ptr, tl.tcoef, tl.seg_csum);
        AI_CUDA(ctx, cudaGetLastError());
        AI_CUDA(ctx, cudaStreamSynchronize(st));
        break;
    }

    // ---- slices and runs (build_sliced.cu), one partial slot per run, bin-major, a bin's slots by ascending tile --------------
    const size_t nseg_alloc = tl.nseg > 0 ? (size_t)tl.nseg : 1;
    DevBuf<int> seg_nruns, bin_first;
    AI_CUDA(ctx, seg_nruns.alloc(nseg_alloc));
    AI_CUDA(ctx, cudaMemsetAsync(seg_nruns.p, 0, nseg_alloc * sizeof(int), st));
    SliceScratch *sc = ai_slice_scratch_new();
    struct ScGuard { SliceScratch *s; ~ScGuard() { ai_slice_scratch_delete(s); } } sc_guard{sc};
    rc = ai_build_sliced_plan(ctx, sc, seg_nruns.p, st);
    if (rc != AI_OK) return rc;
    DevBuf<unsigned long long> keys3a, keys3b;
    DevBuf<long long> runs, prefix;
    AI_CUDA(ctx, keys3a.alloc(nseg_alloc));
    AI_CUDA(ctx, keys3b.alloc(nseg_alloc));
    AI_CUDA(ctx, runs.alloc(nseg_alloc + 1));
    AI_CUDA(ctx, prefix.alloc(nseg_alloc + 1));
    AI_CUDA(ctx, bin_first.alloc((size_t)nbins + 1));
    AI_CUDA(ctx, cudaMalloc(&tl.bin_slot_ptr, ((size_t)nbins + 1) * sizeof(int)));
    const int sblocks = (tl.nseg + 255) / 256 + 1;
    slot_key_kernel<<<sblocks, 256, 0, st>>>(tl.nseg, seg_key.p, keys3a.p);
    AI_CUDA(ctx, sort_keys(scr, keys3a.p, keys3b.p, tl.nseg, 32 + bits_for(nbins), st));
    AI_CUDA(ctx, cudaMemsetAsync(runs.p + tl.nseg, 0, sizeof(long long), st));
    slot_runs_kernel<<<sblocks, 256, 0, st>>>(tl.nseg, keys3b.p, seg_nruns.p, runs.p);
    AI_CUDA(ctx, cudaGetLastError());
    AI_CUDA(ctx, exclusive_sum(scr, runs.p, prefix.p, (long long)tl.nseg + 1, st));
    long long nslot = 0;
    AI_CUDA(ctx, cudaMemcpyAsync(&nslot, prefix.p + tl.nseg, sizeof(long long), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    if (nslot > kMetaSlotMask) return ai_fail(ctx, AI_EUNSUPPORTED, "%lld partial slots", nslot);
    tl.nslot = (int)nslot;
    slot_assign_kernel<<<sblocks, 256, 0, st>>>(tl.nseg, keys3b.p, prefix.p, tl.seg_slot);
    lower_bound_kernel<<<(int)((nbins + 256) / 256), 256, 0, st>>>(keys3b.p, tl.nseg, 32, (int)nbins, bin_first.p);
    bin_slot_kernel<<<(int)((nbins + 256) / 256), 256, 0, st>>>((int)nbins, tl.nseg, bin_first.p, prefix.p, nslot,
                                                                tl.bin_slot_ptr);
    AI_CUDA(ctx, cudaGetLastError());
    rc = ai_build_sliced_fill(ctx, sc, st);
    if (rc != AI_OK) return rc;
    return ai_tiled_finalize(ctx, st);
}

int ai_build_2d(ai_ctx *ctx, cudaStream_t st)
{
    const int H = ctx->height, W = ctx->width, npt_rad = ctx->npt_rad, npt_azim = ctx->npt_azim;
    const int64_t npix = (int64_t)H * W;
    const long long nbins = (long long)npt_rad * npt_azim;
    if (nbins > 0xfffffffLL) return ai_fail(ctx, AI_EUNSUPPORTED, "%lld bins: more than 2^28", nbins);
    TiledLayout &tl = ctx->tl;
    const int grid = 148 * 8;
    Scratch scr;

    // ---- per-pixel spans on both axes -------------------------------------------------------------------------------------
    PixelSpans sp;
    int rc = ai_build_spans(ctx, &sp, npt_rad, st);
    if (rc != AI_OK) { ai_free_spans(&sp); return rc; }
    struct SpanGuard { PixelSpans *s; ~SpanGuard() { ai_free_spans(s); } } span_guard{&sp};
    const double c0 = ctx->azim_host[0], dchi = (ctx->azim_host[1] - ctx->azim_host[0]) / (double)npt_azim;
    DevBuf<double> chi_lo, chi_w;
    DevBuf<long long> cnt, off;
    AI_CUDA(ctx, chi_lo.alloc(npix));
    AI_CUDA(ctx, chi_w.alloc(npix));
    AI_CUDA(ctx, cnt.alloc(npix + 1));
    AI_CUDA(ctx, off.alloc(npix + 1));
    chi_kernel<<<grid, 256, 0, st>>>(ctx->geo, H, W, chi_lo.p, chi_w.p);
    AI_CUDA(ctx, cudaMemsetAsync(cnt.p + npix, 0, sizeof(long long), st));
    count2d_kernel<<<grid, 256, 0, st>>>(npix, sp.nb, chi_lo.p, chi_w.p, c0, dchi, npt_azim, cnt.p);
    AI_CUDA(ctx, cudaGetLastError());
    AI_CUDA(ctx, exclusive_sum(scr, cnt.p, off.p, npix + 1, st));
    long long nnz = 0;
    AI_CUDA(ctx, cudaMemcpyAsync(&nnz, off.p + npix, sizeof(long long), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    if (nnz > 0x7fffffffLL) return ai_fail(ctx, AI_EUNSUPPORTED, "2D matrix has %lld entries", nnz);
    ctx->nnz = nnz;

    // ---- entries, sorted by (bin, pixel): the canonical CSR -----------------------------------------------------------------
    DevBuf<unsigned long long> keys_a, keys_b;
    DevBuf<float> vals_a, vals_b;
    AI_CUDA(ctx, keys_a.alloc(nnz));
    AI_CUDA(ctx, keys_b.alloc(nnz));
    AI_CUDA(ctx, vals_a.alloc(nnz));
    AI_CUDA(ctx, vals_b.alloc(nnz));
    emit2d_kernel<<<grid, 256, 0, st>>>(npix, npt_rad, npt_azim, sp.fmin, sp.fmax, sp.first, sp.nb, chi_lo.p, chi_w.p, c0,
                                        dchi, off.p, keys_a.p, vals_a.p);
    AI_CUDA(ctx, cudaGetLastError());
    return entries_to_layouts(ctx, scr, keys_a.p, keys_b.p, vals_a.p, vals_b.p, nnz, nbins, st);
}

// ======================================================================================================================
// Full pixel splitting (section 4.2): the pixel is the quadrilateral of its four corners in the (radial
// unit, chi) plane, its sides straight lines; the weight in bin b is the area of the part of the quadrilateral between
// the bin's edges -- "integrate the four functions ... over the bounds of each bin", absolute value of the sum -- over
// the area of the whole.  A pixel with the beam centre strictly inside, or with zero area in this plane, is split by its
// bounding box (section 4.1).  Same sort-based path to the layouts as the 2D matrix.
// ======================================================================================================================
namespace {

// signed integral of the line through (f_a, c_a) and (f_b, c_b) over the part of [lo, hi] it spans, along its direction
__device__ __forceinline__ double edge_integral(double f_a, double c_a, double f_b, double c_b, double lo, double hi)
{
    if (f_a == f_b) return 0.0;
    const double m = __ddiv_rn(__dsub_rn(c_b, c_a), __dsub_rn(f_b, f_a));
    const double e_lo = fmax(lo, fmin(f_a, f_b)), e_hi = fmin(hi, fmax(f_a, f_b));
    if (!(e_hi > e_lo)) return 0.0;
    const double v_lo = __dadd_rn(c_a, __dmul_rn(m, __dsub_rn(e_lo, f_a))), v_hi = __dadd_rn(c_a, __dmul_rn(m, __dsub_rn(e_hi, f_a)));
    const double area = __dmul_rn(__dmul_rn(0.5, __dadd_rn(v_lo, v_hi)), __dsub_rn(e_hi, e_lo));
    return f_b > f_a ? area : -area;
}

struct Quad {
    double f[4], chi[4];
    double f_min, f_max, total;       // total = 0: no quadrilateral (bounding-box split of [f_min, f_max])
};

__device__ __forceinline__ double quad_slice(const Quad &q, double lo, double hi)
{
    double a = 0.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) a = __dadd_rn(a, edge_integral(q.f[k], q.chi[k], q.f[(k + 1) & 3], q.chi[(k + 1) & 3], lo, hi));
    return fabs(a);
}

// corners (x_lo,y_lo) (x_hi,y_lo) (x_hi,y_hi) (x_lo,y_hi) of pixel (i, j) in bin units / radians; false if the beam
// centre is strictly inside
__device__ __forceinline__ bool pixel_quad(const ai_geometry &g, int unit, int i, int j, double u0, double delta, Quad *q)
{
    const double x_lo = __dmul_rn(__dsub_rn((double)j, g.center_x_px), g.pixel_x_m);
    const double x_hi = __dmul_rn(__dsub_rn((double)(j + 1), g.center_x_px), g.pixel_x_m);
    const double y_lo = __dmul_rn(__dsub_rn((double)i, g.center_y_px), g.pixel_y_m);
    const double y_hi = __dmul_rn(__dsub_rn((double)(i + 1), g.center_y_px), g.pixel_y_m);
    if (x_lo < 0.0 && x_hi > 0.0 && y_lo < 0.0 && y_hi > 0.0) return false;
    const double xc = __dmul_rn(0.5, __dadd_rn(x_lo, x_hi)), yc = __dmul_rn(0.5, __dadd_rn(y_lo, y_hi));
    const double chi_c = atan2(yc, xc);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double x = (k == 1 || k == 2) ? x_hi : x_lo, y = (k >= 2) ? y_hi : y_lo;
        const double r = __dsqrt_rn(__dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)));
        q->f[k] = __ddiv_rn(__dsub_rn(unit_of_r(r, g.distance_m, g.wavelength_m, unit), u0), delta);
        q->chi[k] = (x == 0.0 && y == 0.0)
                        ? chi_c
                        : __dadd_rn(chi_c, atan2(__dsub_rn(__dmul_rn(xc, y), __dmul_rn(yc, x)),
                                                 __dadd_rn(__dmul_rn(xc, x), __dmul_rn(yc, y))));
    }
    q->f_min = fmin(fmin(q->f[0], q->f[1]), fmin(q->f[2], q->f[3]));
    q->f_max = fmax(fmax(q->f[0], q->f[1]), fmax(q->f[2], q->f[3]));
    q->total = quad_slice(*q, q->f_min, q->f_max);
    return true;
}

// COUNT = true: number of entries of every pixel; false: the entries themselves at offset[p]
template <bool COUNT>
__global__ void __launch_bounds__(256) full_split_kernel(ai_geometry g, int unit, int height, int width, int npt,
                                                         const double *__restrict__ range,
                                                         const double *__restrict__ fmin_a, const double *__restrict__ fmax_a,
                                                         const int *__restrict__ first_a, const int *__restrict__ nb_a,
                                                         long long *__restrict__ cnt, const long long *__restrict__ offset,
                                                         unsigned long long *__restrict__ keys, float *__restrict__ vals)
{
    const int64_t n = (int64_t)height * width;
    const double u0 = range[0], delta = __ddiv_rn(__dsub_rn(range[1], range[0]), (double)npt);
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(p / width), j = (int)(p - (int64_t)i * width);
        Quad q;
        long long at = COUNT ? 0 : offset[p];
        int count = 0;
        const bool quad = pixel_quad(g, unit, i, j, u0, delta, &q);
        if (quad && q.total > 0.0) {
            if (q.f_max > 0.0 && q.f_min < (double)npt) {
                const int b0 = (int)floor(fmax(q.f_min, 0.0)), b1 = min((int)floor(fmin(q.f_max, (double)npt)), npt - 1);
                for (int b = b0; b <= b1; ++b) {
                    const double area = quad_slice(q, (double)b, (double)(b + 1));
                    if (!(area > 0.0)) continue;
                    if (!COUNT) {
                        keys[at] = ((unsigned long long)b << 32) | (unsigned long long)p;
                        vals[at] = (float)__ddiv_rn(area, q.total);
                        ++at;
                    }
                    ++count;
                }
            }
        } else {
            // bounding box: of the pixel rectangle (beam centre inside), or of the degenerate quadrilateral's corners
            double f_lo = fmin_a[p], f_hi = fmax_a[p];
            int first = first_a[p], nb = nb_a[p];
            if (quad) {
                f_lo = q.f_min;
                f_hi = q.f_max;
                split_span(f_lo, f_hi, npt, &first, &nb);
            }
            for (int b = first; b < first + nb; ++b) {
                if (!COUNT) {
                    keys[at] = ((unsigned long long)b << 32) | (unsigned long long)p;
                    vals[at] = (float)split_coefficient(f_lo, f_hi, b, npt);
                    ++at;
                }
                ++count;
            }
        }
        if (COUNT) cnt[p] = count;
    }
}

}  // namespace

int ai_build_full(ai_ctx *ctx, cudaStream_t st)
{
    const int H = ctx->height, W = ctx->width, npt = ctx->npt;
    const int64_t npix = (int64_t)H * W;
    const int grid = 148 * 8;
    Scratch scr;
    PixelSpans sp;                       // bounding-box spans: the automatic range, and the pixels without a quadrilateral
    int rc = ai_build_spans(ctx, &sp, npt, st);
    if (rc != AI_OK) { ai_free_spans(&sp); return rc; }
    struct SpanGuard { PixelSpans *s; ~SpanGuard() { ai_free_spans(s); } } span_guard{&sp};
    DevBuf<long long> cnt, off;
    AI_CUDA(ctx, cnt.alloc(npix + 1));
    AI_CUDA(ctx, off.alloc(npix + 1));
    AI_CUDA(ctx, cudaMemsetAsync(cnt.p + npix, 0, sizeof(long long), st));
    full_split_kernel<true><<<grid, 256, 0, st>>>(ctx->geo, (int)ctx->unit, H, W, npt, ctx->d_range, sp.fmin, sp.fmax,
                                                  sp.first, sp.nb, cnt.p, nullptr, nullptr, nullptr);
    AI_CUDA(ctx, cudaGetLastError());
    AI_CUDA(ctx, exclusive_sum(scr, cnt.p, off.p, npix + 1, st));
    long long nnz = 0;
    AI_CUDA(ctx, cudaMemcpyAsync(&nnz, off.p + npix, sizeof(long long), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    if (nnz > 0x7fffffffLL) return ai_fail(ctx, AI_EUNSUPPORTED, "matrix has %lld entries", nnz);
    ctx->nnz = nnz;
    DevBuf<unsigned long long> keys_a, keys_b;
    DevBuf<float> vals_a, vals_b;
    AI_CUDA(ctx, keys_a.alloc(nnz));
    AI_CUDA(ctx, keys_b.alloc(nnz));
    AI_CUDA(ctx, vals_a.alloc(nnz));
    AI_CUDA(ctx, vals_b.alloc(nnz));
    full_split_kernel<false><<<grid, 256, 0, st>>>(ctx->geo, (int)ctx->unit, H, W, npt, ctx->d_range, sp.fmin, sp.fmax,
                                                   sp.first, sp.nb, nullptr, off.p, keys_a.p, vals_a.p);
    AI_CUDA(ctx, cudaGetLastError());
    return entries_to_layouts(ctx, scr, keys_a.p, keys_b.p, vals_a.p, vals_b.p, nnz, npt, st);
}
