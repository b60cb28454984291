// Tiled execution layout (SURVEY.md section 8(a) B6 "derived layouts"): the same bounding-box
// coefficients as the canonical CSR, re-ordered so that all entries whose pixel lies in one
// tile_h x kTileW image tile are contiguous, grouped by bin into (tile, bin) segments, pixel stored as its 16-bit
// position inside the tile's shared-memory buffer (ai_tile_pos).  Built from the same per-pixel spans with the same
// ordered fill as the canonical CSR.  tile_h is the largest of 64, 32, 16, 8 for which the pipelined kernel's
// shared-memory plan fits (ai_pipe_plan).
#include <algorithm>
#include <vector>

#include "build_common.cuh"
#include "ctx.h"
#include "tiled_build_common.cuh"

struct SliceScratch;
int ai_slice_max_blob(ai_ctx *ctx, int ntiles, const int *tile_seg_ptr, const int *seg_len, cudaStream_t st, int *max_blob);
int ai_build_sliced_plan(ai_ctx *ctx, SliceScratch *sc, int *seg_nruns, cudaStream_t st);
int ai_build_sliced_fill(ai_ctx *ctx, SliceScratch *sc, cudaStream_t st);
SliceScratch *ai_slice_scratch_new();
void ai_slice_scratch_delete(SliceScratch *sc);

namespace {

__device__ __forceinline__ bool tile_pixel(int t, int k, int tiles_x, int th, int height, int width, int64_t *p)
{
    int ty = t / tiles_x, tx = t - ty * tiles_x;
    int y = ty * th + k / kTileW, x = tx * kTileW + k % kTileW;
    *p = (int64_t)y * width + x;
    return y < height && x < width;
}

// range of bins touched by each tile
__global__ void __launch_bounds__(256) tile_range_kernel(int tiles_x, int th, int height, int width,
                                                         const int *__restrict__ first_a, const int *__restrict__ nb_a,
                                                         int *__restrict__ tile_bmin, int *__restrict__ tile_nbins)
{
    const int t = blockIdx.x;
    int lo = 0x7fffffff, hi = -1;
    for (int k = threadIdx.x; k < th * kTileW; k += blockDim.x) {
        int64_t p;
        if (tile_pixel(t, k, tiles_x, th, height, width, &p)) {
            int nb = nb_a[p], first = first_a[p];
            if (nb > 0) { lo = min(lo, first); hi = max(hi, first + nb - 1); }
        }
    }
    __shared__ int s_lo[8], s_hi[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if ((threadIdx.x & 31) == 0) { s_lo[threadIdx.x >> 5] = lo; s_hi[threadIdx.x >> 5] = hi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { lo = min(lo, s_lo[w]); hi = max(hi, s_hi[w]); }
        tile_bmin[t] = hi >= 0 ? lo : 0;
        tile_nbins[t] = hi >= 0 ? hi - lo + 1 : 0;
    }
}

// number of entries of every (tile, bin) segment
__global__ void __launch_bounds__(256) tile_count_kernel(int tiles_x, int th, int height, int width,
                                                         const int *__restrict__ first_a, const int *__restrict__ nb_a,
                                                         const int *__restrict__ tile_bmin,
                                                         const int *__restrict__ tile_seg_ptr, int *__restrict__ seg_len)
{
    const int t = blockIdx.x;
    const int bmin = tile_bmin[t], s0 = tile_seg_ptr[t];
    for (int k = threadIdx.x; k < th * kTileW; k += blockDim.x) {
        int64_t p;
        if (tile_pixel(t, k, tiles_x, th, height, width, &p)) {
            int nb = nb_a[p], first = first_a[p];
            for (int b = first; b < first + nb; ++b) atomicAdd(&seg_len[s0 + b - bmin], 1);
        }
    }
}

struct TileChunk {
    int t, tiles_x, th, height, width, bmin, s0;
    const int *seg_ptr;
    int *seg_cur;
    float *tcoef;
    uint16_t *tidx;
    __device__ int npix() const { return th * kTileW; }
    __device__ bool pixel(int k, int64_t *p) const { return tile_pixel(t, k, tiles_x, th, height, width, p); }
    __device__ int base(int b) const { return seg_ptr[s0 + b - bmin]; }
    __device__ volatile int *cursor(int b) const { return seg_cur + s0 + b - bmin; }
    // Entries of a segment are consumed in windows of 32 by kTileLanes = 8 lanes, lane l reading entries 4l .. 4l+3
    // of the window with one 128-bit load.  Pixel-order entry j of a window is stored at (j % la) * 4 + j / la (la =
    // lanes the window occupies), so that in each of a lane's four gathers the lanes read CONSECUTIVE pixels of the
    // segment -- neighbours along the ring, which ai_tile_pos puts in different banks.
    __device__ int64_t place(int b, int64_t pos) const
    {
        const int base = seg_ptr[s0 + b - bmin], plen = seg_ptr[s0 + b - bmin + 1] - base;
        const int r = (int)(pos - base), w = r >> 5, j = r & 31;
        const int la = min(8, (plen - 32 * w) / 4);
        return (int64_t)base + 32 * w + (j % la) * 4 + j / la;
    }
    __device__ void emit(int64_t pos, int k, int64_t, float coef) const
    {
        tcoef[pos] = coef;
        tidx[pos] = (uint16_t)(ai_tile_pos(k / kTileW, k % kTileW, th) * 4);      // byte offset in the tile buffer
    }
};

__global__ void __launch_bounds__(128) fill_tiles_kernel(int ntiles, int tiles_x, int th, int height, int width, int npt,
                                                         const double *__restrict__ fmin_a,
                                                         const double *__restrict__ fmax_a,
                                                         const int *__restrict__ first_a, const int *__restrict__ nb_a,
                                                         const int *__restrict__ tile_bmin,
                                                         const int *__restrict__ tile_seg_ptr,
                                                         const int *__restrict__ seg_ptr, int *seg_cur,
                                                         float *__restrict__ tcoef, uint16_t *__restrict__ tidx)
{
    int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (t >= ntiles) return;
    TileChunk ch{t, tiles_x, th, height, width, tile_bmin[t], tile_seg_ptr[t], seg_ptr, seg_cur, tcoef, tidx};
    marching_fill(ch, fmin_a, fmax_a, first_a, nb_a, npt);
}

// number of partial slots of each bin: the runs (build_sliced.cu) of its segments over all tiles
__global__ void __launch_bounds__(128) bin_tiles_count_kernel(int npt, int ntiles, const int *__restrict__ tile_bmin,
                                                              const int *__restrict__ tile_nbins,
                                                              const int *__restrict__ tile_seg_ptr,
                                                              const int *__restrict__ seg_nruns, int *__restrict__ nslot)
{
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= npt) return;
    int c = 0;
    for (int t = 0; t < ntiles; ++t) {
        int lo = tile_bmin[t];
        if (b >= lo && b < lo + tile_nbins[t]) c += seg_nruns[tile_seg_ptr[t] + b - lo];
    }
    nslot[b] = c;
}

// first slot of every segment in the bin-major partial buffer: bin b's slots are ordered by ascending tile, the runs
// of one segment are adjacent
__global__ void __launch_bounds__(128) bin_tiles_assign_kernel(int npt, int ntiles, const int *__restrict__ tile_bmin,
                                                               const int *__restrict__ tile_nbins,
                                                               const int *__restrict__ tile_seg_ptr,
                                                               const int *__restrict__ seg_nruns,
                                                               const int *__restrict__ bin_slot_ptr,
                                                               int *__restrict__ seg_slot)
{
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= npt) return;
    int slot = bin_slot_ptr[b];
    for (int t = 0; t < ntiles; ++t) {
        int lo = tile_bmin[t];
        if (b >= lo && b < lo + tile_nbins[t]) {
            const int s = tile_seg_ptr[t] + b - lo;
            seg_slot[s] = slot;
            slot += seg_nruns[s];
        }
    }
}

}  // namespace

static void free_tiled(TiledLayout &tl)
{
    cudaFree(tl.tile_seg_ptr); cudaFree(tl.seg_ptr); cudaFree(tl.seg_slot); cudaFree(tl.seg_meta); cudaFree(tl.seg_csum);
    cudaFree(tl.tile_desc); cudaFree(tl.tile_order); cudaFree(tl.tcoef); cudaFree(tl.tidx); cudaFree(tl.bin_slot_ptr);
    cudaFree(tl.blob); cudaFree(tl.blob_desc);
    free(tl.h_first_desc);
    tl = TiledLayout{};
}

// Segment structure for one tile height: tile_seg_ptr, padded seg_len, the largest tile.  Returns AI_OK and sets *fits.
static int plan_tiles(ai_ctx *ctx, const PixelSpans &sp, int th, cudaStream_t st, int **tile_bmin, int **tile_nbins,
                      int **seg_len, bool *fits)
{
    TiledLayout &tl = ctx->tl;
    const int H = ctx->height, W = ctx->width;
    tl.tile_h = th;
    tl.tiles_y = (H + th - 1) / th;
    tl.tiles_x = (W + kTileW - 1) / kTileW;
    tl.ntiles = tl.tiles_y * tl.tiles_x;
    long long *d_total = nullptr, h_total = 0;
    int *tile_entries = nullptr;
    AI_CUDA(ctx, cudaMalloc(tile_bmin, tl.ntiles * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(tile_nbins, tl.ntiles * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&tile_entries, tl.ntiles * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&tl.tile_seg_ptr, (tl.ntiles + 1) * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&d_total, sizeof(long long)));
    tile_range_kernel<<<tl.ntiles, 256, 0, st>>>(tl.tiles_x, th, H, W, sp.first, sp.nb, *tile_bmin, *tile_nbins);
    scan_pad_kernel<<<1, 1024, 0, st>>>(tl.ntiles, *tile_nbins, 1, tl.tile_seg_ptr, d_total);
    AI_CUDA(ctx, cudaGetLastError());
    AI_CUDA(ctx, cudaMemcpyAsync(&h_total, d_total, sizeof(long long), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    cudaFree(d_total);
    if (h_total > 0x7fffffffLL) return ai_fail(ctx, AI_EUNSUPPORTED, "too many (tile, bin) segments: %lld", h_total);
    tl.nseg = (int)h_total;
    const size_t nseg_alloc = tl.nseg > 0 ? tl.nseg : 1;
    AI_CUDA(ctx, cudaMalloc(seg_len, nseg_alloc * sizeof(int)));
    AI_CUDA(ctx, cudaMemsetAsync(*seg_len, 0, nseg_alloc * sizeof(int), st));
    tile_count_kernel<<<tl.ntiles, 256, 0, st>>>(tl.tiles_x, th, H, W, sp.first, sp.nb, *tile_bmin, tl.tile_seg_ptr,
                                                 *seg_len);
    pad_segments_kernel<<<(tl.ntiles + 127) / 128, 128, 0, st>>>(tl.ntiles, tl.tile_seg_ptr, *seg_len, tile_entries);
    AI_CUDA(ctx, cudaGetLastError());
    std::vector<int> h_entries(tl.ntiles), h_nbins(tl.ntiles);
    AI_CUDA(ctx, cudaMemcpyAsync(h_entries.data(), tile_entries, tl.ntiles * sizeof(int), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaMemcpyAsync(h_nbins.data(), *tile_nbins, tl.ntiles * sizeof(int), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    cudaFree(tile_entries);
    tl.max_tile_entries = 0;
    tl.max_tile_segs = 0;
    for (int t = 0; t < tl.ntiles; ++t) {
        tl.max_tile_entries = std::max(tl.max_tile_entries, h_entries[t]);
        tl.max_tile_segs = std::max(tl.max_tile_segs, h_nbins[t]);
    }
    int max_blob = 0;
    int rc = ai_slice_max_blob(ctx, tl.ntiles, tl.tile_seg_ptr, *seg_len, st, &max_blob);
    if (rc != AI_OK) return rc;
    *fits = ai_pipe_plan(max_blob, th, false, ctx->tune).fits;
    return AI_OK;
}

int ai_build_tiled(ai_ctx *ctx, const PixelSpans &sp, cudaStream_t st)
{
    TiledLayout &tl = ctx->tl;
    const int H = ctx->height, W = ctx->width, npt = ctx->npt;
    int *tile_bmin = nullptr, *tile_nbins = nullptr, *seg_len = nullptr, *seg_cur = nullptr, *nslot = nullptr;
    long long *d_total = nullptr, h_total = 0;
    // largest tile height whose slices fit the pipelined kernel (8 is taken regardless: the direct kernel serves it)
    int th0 = kTileHMax;
    while (th0 > 8 && th0 > ctx->tune.tile_h_max) th0 /= 2;
    for (int th = th0;; th /= 2) {
        bool fits = false;
        int rc = plan_tiles(ctx, sp, th, st, &tile_bmin, &tile_nbins, &seg_len, &fits);
        if (rc != AI_OK) return rc;
        if (fits || th == 8) break;
        cudaFree(tile_bmin); cudaFree(tile_nbins); cudaFree(seg_len);
        tile_bmin = tile_nbins = seg_len = nullptr;
        free_tiled(tl);
    }
    const int th = tl.tile_h;
    const size_t nseg_alloc = tl.nseg > 0 ? tl.nseg : 1;
    AI_CUDA(ctx, cudaMalloc(&d_total, sizeof(long long)));
    AI_CUDA(ctx, cudaMalloc(&seg_cur, nseg_alloc * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&tl.seg_ptr, (nseg_alloc + 1) * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&tl.seg_slot, nseg_alloc * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&tl.seg_csum, nseg_alloc * sizeof(double)));
    AI_CUDA(ctx, cudaMemsetAsync(seg_cur, 0, nseg_alloc * sizeof(int), st));
    scan_pad_kernel<<<1, 1024, 0, st>>>(tl.nseg, seg_len, 1, tl.seg_ptr, d_total);
    AI_CUDA(ctx, cudaGetLastError());
    AI_CUDA(ctx, cudaMemcpyAsync(&h_total, d_total, sizeof(long long), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    if (h_total > 0x7fffffffLL) return ai_fail(ctx, AI_EUNSUPPORTED, "tiled layout has %lld entries", h_total);
    tl.tnnz = h_total;
    const size_t nnz_alloc = tl.tnnz > 0 ? (size_t)tl.tnnz : 1;

    AI_CUDA(ctx, cudaMalloc(&tl.tcoef, nnz_alloc * sizeof(float)));
    AI_CUDA(ctx, cudaMalloc(&tl.tidx, nnz_alloc * sizeof(uint16_t)));
    AI_CUDA(ctx, cudaMemsetAsync(tl.tcoef, 0, nnz_alloc * sizeof(float), st));       // padding: coefficient 0,
    AI_CUDA(ctx, cudaMemsetAsync(tl.tidx, 0, nnz_alloc * sizeof(uint16_t), st));     // pixel 0 of the tile
    fill_tiles_kernel<<<(tl.ntiles + 3) / 4, 128, 0, st>>>(tl.ntiles, tl.tiles_x, th, H, W, npt, sp.fmin, sp.fmax,
                                                           sp.first, sp.nb, tile_bmin, tl.tile_seg_ptr, tl.seg_ptr,
                                                           seg_cur, tl.tcoef, tl.tidx);
    if (tl.nseg > 0)
        seg_sum_kernel<<<(tl.nseg + 7) / 8, 256, 0, st>>>(tl.nseg, tl.seg_ptr, tl.tcoef, tl.seg_csum);

    // slices and runs of the sliced layout: one partial slot per run, bin-major
    int *seg_nruns = nullptr;
    AI_CUDA(ctx, cudaMalloc(&seg_nruns, nseg_alloc * sizeof(int)));
    AI_CUDA(ctx, cudaMemsetAsync(seg_nruns, 0, nseg_alloc * sizeof(int), st));
    SliceScratch *sc = ai_slice_scratch_new();
    int rc = ai_build_sliced_plan(ctx, sc, seg_nruns, st);
    if (rc != AI_OK) { ai_slice_scratch_delete(sc); return rc; }
    AI_CUDA(ctx, cudaMalloc(&nslot, (size_t)npt * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&tl.bin_slot_ptr, ((size_t)npt + 1) * sizeof(int)));
    bin_tiles_count_kernel<<<(npt + 127) / 128, 128, 0, st>>>(npt, tl.ntiles, tile_bmin, tile_nbins, tl.tile_seg_ptr,
                                                              seg_nruns, nslot);
    scan_pad_kernel<<<1, 1024, 0, st>>>(npt, nslot, 1, tl.bin_slot_ptr, d_total);
    bin_tiles_assign_kernel<<<(npt + 127) / 128, 128, 0, st>>>(npt, tl.ntiles, tile_bmin, tile_nbins, tl.tile_seg_ptr,
                                                               seg_nruns, tl.bin_slot_ptr, tl.seg_slot);
    AI_CUDA(ctx, cudaMemcpyAsync(&h_total, d_total, sizeof(long long), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    if (h_total > kMetaSlotMask) { ai_slice_scratch_delete(sc); return ai_fail(ctx, AI_EUNSUPPORTED, "%lld partial slots", h_total); }
    tl.nslot = (int)h_total;
    rc = ai_build_sliced_fill(ctx, sc, st);
    ai_slice_scratch_delete(sc);
    cudaFree(seg_nruns);
    if (rc != AI_OK) return rc;
    rc = ai_tiled_finalize(ctx, st);
    if (rc != AI_OK) return rc;
    cudaFree(tile_bmin); cudaFree(tile_nbins); cudaFree(seg_len); cudaFree(seg_cur); cudaFree(nslot); cudaFree(d_total);
    return AI_OK;
}
