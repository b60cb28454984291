// Frame-lane layout of the matrix (SURVEY.md section 8(a) B6 "derived layouts", H6): the
// bounding-box coefficients of the canonical CSR, re-ordered for the batched kernel of
// integrate_fl.cu, in which the 32 lanes of a warp are 32 pairs of frames and every matrix entry is warp-uniform.
//   - the image is cut into tiles of kFlTileW x kFlTileH pixels; a tile's entries are grouped by bin into segments;
//   - tiles are ordered by their lowest bin and cut into chunks of at most kFlChunkTilesMax tiles whose bins fit a window
//     of kFlWindow bins: the kernel keeps one shared-memory accumulator per (bin of the window, frame) and writes one
//     partial per (chunk, bin, frame);
//   - inside a chunk every bin belongs to ONE consumer warp (dealt round-robin: a tile's bins are a contiguous range, so
//     every warp gets an even sample of its short and long segments), so accumulators are never shared between warps and
//     every sum has a fixed order;
//   - a tile's blob = header {first record of each warp} + records {bin - chunk's lowest bin, pairs, first pair} +
//     entry pairs {c0, c1, byte offset of pixel 0, byte offset of pixel 1} (one 128-bit broadcast load per pair), a
//     warp's segments one after the other.
// Built from the canonical CSR on the device (count, fill: one warp per row, entries keep the row's ascending pixel
// order, no atomics on the data path); the plan in between (chunks, owners, offsets) is host work over the segment
// lengths.
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <numeric>
#include <vector>

#include "ctx.h"

namespace {

constexpr int kFlHdrBytes = 48;          // uint16 first_record[kFlCons + 1], padded
constexpr int kFlMaxPairs = 1023;        // pairs of one segment (10 bits of a record)
constexpr int kFlMaxPairOff = 16383;     // first pair of a segment inside its tile (14 bits)

__device__ __forceinline__ int fl_tile_of(int p, int width, int th, int tiles_x, int *pos)
{
    const int y = p / width, x = p - y * width;
    const int ty = y / th, tx = x / kFlTileW;
    *pos = ((y - ty * th) * kFlTileW + (x - tx * kFlTileW)) * 8;      // two frames per pixel and lane
    return ty * tiles_x + tx;
}

// bins touched by each tile; sum of each row's coefficients (fp64, fixed order)
__global__ void __launch_bounds__(256) fl_range_kernel(int npt, const int *__restrict__ indptr,
                                                       const int *__restrict__ indices, const float *__restrict__ data,
                                                       int width, int th, int tiles_x, int *__restrict__ tile_bmin,
                                                       int *__restrict__ tile_bmax, double *__restrict__ bin_csum)
{
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (b >= npt) return;
    const int beg = indptr[b], end = indptr[b + 1];
    double a = 0.0;
    int last = -1;
    for (int e = beg + lane; e < end; e += 32) {
        int pos;
        const int t = fl_tile_of(indices[e], width, th, tiles_x, &pos);
        if (t != last) {
            atomicMin(tile_bmin + t, b);
            atomicMax(tile_bmax + t, b);
            last = t;
        }
        a += (double)data[e];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if (lane == 0) bin_csum[b] = a;
}

// entries of every (tile, bin) segment.  A segment belongs to one row, a row to one warp: no atomics.
__global__ void __launch_bounds__(256) fl_count_kernel(int npt, const int *__restrict__ indptr,
                                                       const int *__restrict__ indices, int width, int th, int tiles_x,
                                                       const int *__restrict__ tile_bmin,
                                                       const int *__restrict__ tile_seg_ptr, int *seg_len)
{
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (b >= npt) return;
    const int beg = indptr[b], end = indptr[b + 1];
    for (int e0 = beg; e0 < end; e0 += 32) {
        const int e = e0 + lane;
        int seg = -1 - lane;
        if (e < end) {
            int pos;
            const int t = fl_tile_of(indices[e], width, th, tiles_x, &pos);
            seg = tile_seg_ptr[t] + b - tile_bmin[t];
        }
        const unsigned m = __match_any_sync(0xffffffffu, seg);
        if (seg >= 0 && lane == __ffs(m) - 1) seg_len[seg] += __popc(m);
        __syncwarp();
    }
}

// entries into the blobs: entry k of a segment (ascending pixel) goes to pair k / 2, half k % 2
__global__ void __launch_bounds__(256) fl_fill_kernel(int npt, const int *__restrict__ indptr,
                                                      const int *__restrict__ indices, const float *__restrict__ data,
                                                      int width, int th, int tiles_x,
                                                      const int *__restrict__ tile_bmin,
                                                      const int *__restrict__ tile_seg_ptr,
                                                      const unsigned *__restrict__ seg_dst, int *seg_cur,
                                                      unsigned char *__restrict__ blob)
{
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (b >= npt) return;
    const int beg = indptr[b], end = indptr[b + 1];
    for (int e0 = beg; e0 < end; e0 += 32) {
        const int e = e0 + lane;
        int seg = -1 - lane, pos = 0;
        if (e < end) {
            const int t = fl_tile_of(indices[e], width, th, tiles_x, &pos);
            seg = tile_seg_ptr[t] + b - tile_bmin[t];
        }
        const unsigned m = __match_any_sync(0xffffffffu, seg);
        int k = 0;
        if (seg >= 0) k = seg_cur[seg] + __popc(m & ((1u << lane) - 1u));
        __syncwarp();
        if (seg >= 0) {
            if (lane == __ffs(m) - 1) seg_cur[seg] += __popc(m);
            unsigned char *q = blob + ((size_t)seg_dst[seg] + (size_t)(k >> 1)) * 16 + (k & 1) * 4;
            *reinterpret_cast<float *>(q) = data[e];
            *reinterpret_cast<unsigned *>(q + 8) = (unsigned)pos;
        }
        __syncwarp();
    }
}

// the headers (built on the host, packed one after the other) into their blobs
__global__ void __launch_bounds__(128) fl_header_kernel(int ntiles, const int4 *__restrict__ tile_desc,
                                                        const int *__restrict__ hdr_off,
                                                        const uint4 *__restrict__ hdr, unsigned char *__restrict__ blob)
{
    const int r = blockIdx.x;
    if (r >= ntiles) return;
    const int n = hdr_off[r + 1] - hdr_off[r];
    uint4 *dst = reinterpret_cast<uint4 *>(blob + (size_t)tile_desc[r].x * 16);
    for (int k = threadIdx.x; k < n; k += blockDim.x) dst[k] = hdr[hdr_off[r] + k];
}

template <class T>
int upload(ai_ctx *ctx, T **dev, const std::vector<T> &h, cudaStream_t st)
{
    const size_t n = h.size() ? h.size() : 1;
    AI_CUDA(ctx, cudaMalloc(dev, n * sizeof(T)));
    if (h.size()) AI_CUDA(ctx, cudaMemcpyAsync(*dev, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, st));
    return AI_OK;
}

}  // namespace

void ai_free_fl(FlLayout &fl)
{
    cudaFree(fl.tile_desc); cudaFree(fl.chunk_desc); cudaFree(fl.chunk_owner); cudaFree(fl.blob);
    cudaFree(fl.bin_slot_ptr); cudaFree(fl.bin_slots); cudaFree(fl.bin_csum); cudaFree(fl.call_csum); cudaFree(fl.gone); cudaFree(fl.scale); cudaFree(fl.blob_call); cudaFree(fl.partials);
    fl = FlLayout{};
}

// Builds ctx->fl from the canonical CSR.  fl.ok stays false (AI_OK is returned) where the layout does not apply: a
// tile that touches more than kFlWindow bins, or a segment / tile beyond the record's bit fields.  Synchronises `st`.
int ai_build_fl(ai_ctx *ctx, int nframes, cudaStream_t st)
{
    FlLayout &fl = ctx->fl;
    fl.tried = true;
    fl.ok = false;
    if (ctx->npt_azim > 0 || ctx->nnz <= 0 || !ctx->indptr) return AI_OK;
    const int H = ctx->height, W = ctx->width, npt = ctx->npt;
    const int th = kFlTileH;
    const int tiles_x = (W + kFlTileW - 1) / kFlTileW, tiles_y = (H + th - 1) / th;
    const int ntiles_all = tiles_x * tiles_y;
    if (tiles_x > 0xffff || tiles_y > 0x7fff || npt > 0x7fffff) return AI_OK;
    const int wpb = 8, grid_rows = (npt + wpb - 1) / wpb;

    int *d_bmin = nullptr, *d_bmax = nullptr, *d_seg_ptr = nullptr, *d_seg_len = nullptr;
    unsigned *d_seg_dst = nullptr;
    int *d_hdr_off = nullptr;
    uint4 *d_hdr = nullptr;
    auto cleanup = [&]() {
        cudaFree(d_bmin); cudaFree(d_bmax); cudaFree(d_seg_ptr); cudaFree(d_seg_len); cudaFree(d_seg_dst);
        cudaFree(d_hdr_off); cudaFree(d_hdr);
    };
#define FL_CUDA(call)                                                                                      \
    do {                                                                                                   \
        cudaError_t e_ = (call);                                                                           \
        if (e_ != cudaSuccess) {                                                                           \
            cleanup();                                                                                     \
            ai_free_fl(fl);                                                                                \
            fl.tried = true;                                                                               \
            return ai_fail(ctx, e_ == cudaErrorMemoryAllocation ? AI_ENOMEM : AI_ECUDA, "%s: %s (%s:%d)", #call, \
                           cudaGetErrorString(e_), __FILE__, __LINE__);                                    \
        }                                                                                                  \
    } while (0)

    // 1. bins of every tile
    FL_CUDA(cudaMalloc(&d_bmin, (size_t)ntiles_all * sizeof(int)));
    FL_CUDA(cudaMalloc(&d_bmax, (size_t)ntiles_all * sizeof(int)));
    FL_CUDA(cudaMalloc(&fl.bin_csum, (size_t)npt * sizeof(double)));
    FL_CUDA(cudaMemsetAsync(d_bmin, 0x7f, (size_t)ntiles_all * sizeof(int), st));
    FL_CUDA(cudaMemsetAsync(d_bmax, 0xff, (size_t)ntiles_all * sizeof(int), st));
    fl_range_kernel<<<grid_rows, wpb * 32, 0, st>>>(npt, ctx->indptr, ctx->indices, ctx->data, W, th, tiles_x, d_bmin,
                                                    d_bmax, fl.bin_csum);
    FL_CUDA(cudaGetLastError());
    std::vector<int> bmin(ntiles_all), bmax(ntiles_all);
    FL_CUDA(cudaMemcpyAsync(bmin.data(), d_bmin, (size_t)ntiles_all * sizeof(int), cudaMemcpyDeviceToHost, st));
    FL_CUDA(cudaMemcpyAsync(bmax.data(), d_bmax, (size_t)ntiles_all * sizeof(int), cudaMemcpyDeviceToHost, st));
    FL_CUDA(cudaStreamSynchronize(st));
    std::vector<int> seg_ptr(ntiles_all + 1, 0);
    for (int t = 0; t < ntiles_all; ++t) {
        const int nb = bmax[t] >= 0 ? bmax[t] - bmin[t] + 1 : 0;
        if (nb > kFlWindow) { cleanup(); ai_free_fl(fl); fl.tried = true; return AI_OK; }
        if ((int64_t)seg_ptr[t] + nb > 0x7fffffffLL) { cleanup(); ai_free_fl(fl); fl.tried = true; return AI_OK; }
        seg_ptr[t + 1] = seg_ptr[t] + nb;
    }
    const int nseg = seg_ptr[ntiles_all];

    // 2. entries of every segment
    FL_CUDA(cudaMalloc(&d_seg_ptr, ((size_t)ntiles_all + 1) * sizeof(int)));
    FL_CUDA(cudaMalloc(&d_seg_len, (size_t)(nseg > 0 ? nseg : 1) * sizeof(int)));
    FL_CUDA(cudaMemcpyAsync(d_seg_ptr, seg_ptr.data(), ((size_t)ntiles_all + 1) * sizeof(int), cudaMemcpyHostToDevice, st));
    FL_CUDA(cudaMemsetAsync(d_seg_len, 0, (size_t)(nseg > 0 ? nseg : 1) * sizeof(int), st));
    fl_count_kernel<<<grid_rows, wpb * 32, 0, st>>>(npt, ctx->indptr, ctx->indices, W, th, tiles_x, d_bmin, d_seg_ptr,
                                                    d_seg_len);
    FL_CUDA(cudaGetLastError());
    std::vector<int> seg_len(nseg > 0 ? nseg : 1);
    FL_CUDA(cudaMemcpyAsync(seg_len.data(), d_seg_len, (size_t)(nseg > 0 ? nseg : 1) * sizeof(int), cudaMemcpyDeviceToHost, st));
    FL_CUDA(cudaStreamSynchronize(st));

    // 3. plan: tiles by lowest bin, chunks, owners, blobs
    std::vector<int> order;
    order.reserve(ntiles_all);
    for (int t = 0; t < ntiles_all; ++t)
        if (bmax[t] >= 0) order.push_back(t);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return bmin[a] < bmin[b]; });
    const int ntiles = (int)order.size();
    // tiles per chunk: large chunks mean fewer flushes and barriers, but the items (chunk x group of frames) are dealt to
    // the SMs in rounds: of the sizes 8 .. kFlChunkTilesMax take the one whose last round is fullest for the batch this
    // layout is built for (ties: the larger)
    int chunk_tiles = ctx->tune.fl_chunk;
    if (chunk_tiles <= 0) {
        const int64_t ngroups = (nframes + kFlFrames - 1) / kFlFrames, sms = ctx->sm_count > 0 ? ctx->sm_count : 148;
        double best = -1.0;
        for (int ct = kFlChunkTilesMax; ct >= 8; --ct) {
            const int64_t items = (int64_t)((ntiles + ct - 1) / ct) * ngroups, rounds = (items + sms - 1) / sms;
            const double eff = (double)items / (double)(rounds * sms) - (rounds < 4 ? 0.05 * (4 - rounds) : 0.0);
            if (eff > best + 1e-9) { best = eff; chunk_tiles = ct; }
        }
    }
    std::vector<int4> chunk_desc;
    std::vector<int> chunk_lo;
    {
        int first = 0, lo = 0, hi = -1;
        for (int r = 0; r < ntiles; ++r) {
            const int t = order[r];
            if (r > first && (r - first == chunk_tiles || std::max(hi, bmax[t]) - lo + 1 > kFlWindow)) {
                chunk_desc.push_back(make_int4(first, r - first, 0, hi - lo + 1));
                chunk_lo.push_back(lo);
                first = r;
            }
            if (r == first) { lo = bmin[t]; hi = bmax[t]; }
            else hi = std::max(hi, bmax[t]);
        }
        if (ntiles > first) {
            chunk_desc.push_back(make_int4(first, ntiles - first, 0, hi - lo + 1));
            chunk_lo.push_back(lo);
        }
    }
    const int nchunks = (int)chunk_desc.size();
    int nslot = 0;
    std::vector<int> chunk_nb(nchunks);
    for (int c = 0; c < nchunks; ++c) {
        chunk_nb[c] = chunk_desc[c].w;
        chunk_desc[c].z = nslot;
        nslot += chunk_nb[c];
        chunk_desc[c].w = chunk_lo[c] << 8 | (chunk_nb[c] - 1);
    }
    std::vector<uint8_t> owner((size_t)nchunks * kFlWindow, 0);
    std::vector<int4> tile_desc(ntiles);
    std::vector<unsigned> seg_dst(nseg > 0 ? nseg : 1, 0);
    std::vector<int> hdr_off(ntiles + 1, 0);
    std::vector<uint4> hdr;
    int64_t blob16 = 0;                      // blob bytes so far / 16
    int max_blob = 0;
    bool fits = true;
    for (int c = 0; c < nchunks && fits; ++c) {
        const int first = chunk_desc[c].x, n = chunk_desc[c].y, nb = chunk_nb[c], lo = chunk_lo[c];
        // entries per bin over the chunk; owners: longest first onto the least loaded warp
        int64_t tot[kFlWindow] = {0};
        for (int r = first; r < first + n; ++r) {
            const int t = order[r];
            for (int b = bmin[t]; b <= bmax[t]; ++b) tot[b - lo] += (seg_len[seg_ptr[t] + b - bmin[t]] + 1) / 2 + 3;
        }
        int idx[kFlWindow];
        for (int k = 0; k < nb; ++k) idx[k] = k;
        std::stable_sort(idx, idx + nb, [&](int a, int b) { return tot[a] > tot[b]; });
        int64_t load[kFlCons] = {0};
        uint8_t *own = owner.data() + (size_t)c * kFlWindow;
        for (int k = 0; k < nb; ++k) {
            int w = 0;
            for (int v = 1; v < kFlCons; ++v)
                if (load[v] < load[w]) w = v;
            // round-robin by default: a tile's bins are a contiguous range, so every warp gets an even sample of
            // the tile's short and long segments (measured better than longest-first over the chunk, which balances
            // the chunk but not its tiles)
            if (ctx->tune.fl_owner != 1) w = idx[k] % kFlCons;
            own[idx[k]] = (uint8_t)w;
            load[w] += tot[idx[k]];
        }
        for (int k = nb; k < kFlWindow; ++k) own[k] = 0xff;
        for (int r = first; r < first + n && fits; ++r) {
            const int t = order[r];
            uint16_t wptr[kFlHdrBytes / 2] = {0};
            std::vector<unsigned> recs;
            int pair_off = 0;
            for (int w = 0; w < kFlCons; ++w) {
                wptr[w] = (uint16_t)recs.size();
                for (int b = bmin[t]; b <= bmax[t]; ++b) {
                    const int s = seg_ptr[t] + b - bmin[t], len = seg_len[s];
                    if (own[b - lo] != w || len == 0) continue;
                    const int npairs = (len + 1) / 2;
                    if (npairs > kFlMaxPairs || pair_off > kFlMaxPairOff) { fits = false; break; }
                    recs.push_back((unsigned)(b - lo) << 24 | (unsigned)npairs << 14 | (unsigned)pair_off);
                    seg_dst[s] = (unsigned)pair_off;        // relative to the first pair of the tile, for now
                    pair_off += npairs;
                }
            }
            wptr[kFlCons] = (uint16_t)recs.size();
            const int hdr_bytes = (kFlHdrBytes + 4 * (int)recs.size() + 15) / 16 * 16;
            const int blob_bytes = hdr_bytes + 16 * pair_off + 32;      // two zero pairs behind: the look-ahead stays valid
            if (blob16 + blob_bytes / 16 > 0xfffffff0LL) { fits = false; break; }
            for (int b = bmin[t]; b <= bmax[t]; ++b) seg_dst[seg_ptr[t] + b - bmin[t]] += (unsigned)(blob16 + hdr_bytes / 16);
            tile_desc[r] = make_int4((int)blob16, blob_bytes, (t / tiles_x) << 16 | (t % tiles_x), pair_off);
            std::vector<unsigned char> hb(hdr_bytes, 0);
            memcpy(hb.data(), wptr, (kFlCons + 1) * sizeof(uint16_t));
            if (!recs.empty()) memcpy(hb.data() + kFlHdrBytes, recs.data(), recs.size() * 4);
            const size_t at = hdr.size();
            hdr.resize(at + hdr_bytes / 16);
            memcpy(hdr.data() + at, hb.data(), hdr_bytes);
            hdr_off[r + 1] = (int)hdr.size();
            blob16 += blob_bytes / 16;
            max_blob = std::max(max_blob, blob_bytes);
        }
    }
    if (!fits || ntiles == 0) { cleanup(); ai_free_fl(fl); fl.tried = true; return AI_OK; }
    // H5: the slots of every bin, ascending chunk
    std::vector<int> bin_slot_ptr(npt + 1, 0), bin_slots;
    {
        std::vector<int> cnt(npt, 0);
        for (int c = 0; c < nchunks; ++c)
            for (int k = 0; k < chunk_nb[c]; ++k) ++cnt[chunk_lo[c] + k];
        for (int b = 0; b < npt; ++b) bin_slot_ptr[b + 1] = bin_slot_ptr[b] + cnt[b];
        bin_slots.resize(bin_slot_ptr[npt]);
        std::fill(cnt.begin(), cnt.end(), 0);
        for (int c = 0; c < nchunks; ++c)
            for (int k = 0; k < chunk_nb[c]; ++k) {
                const int b = chunk_lo[c] + k;
                bin_slots[bin_slot_ptr[b] + cnt[b]++] = chunk_desc[c].z + k;
            }
    }

    // 4. blobs
    fl.blob_bytes = blob16 * 16;
    FL_CUDA(cudaMalloc(&fl.blob, (size_t)fl.blob_bytes));
    FL_CUDA(cudaMemsetAsync(fl.blob, 0, (size_t)fl.blob_bytes, st));
    int rc = upload(ctx, &fl.tile_desc, tile_desc, st);
    if (rc == AI_OK) rc = upload(ctx, &fl.chunk_desc, chunk_desc, st);
    if (rc == AI_OK) rc = upload(ctx, &fl.chunk_owner, owner, st);
    if (rc == AI_OK) rc = upload(ctx, &fl.bin_slot_ptr, bin_slot_ptr, st);
    if (rc == AI_OK) rc = upload(ctx, &fl.bin_slots, bin_slots, st);
    if (rc == AI_OK) rc = upload(ctx, &d_seg_dst, seg_dst, st);
    if (rc == AI_OK) rc = upload(ctx, &d_hdr_off, hdr_off, st);
    if (rc == AI_OK) rc = upload(ctx, &d_hdr, hdr, st);
    if (rc != AI_OK) { cleanup(); ai_free_fl(fl); fl.tried = true; return rc; }
    FL_CUDA(cudaMemsetAsync(d_seg_len, 0, (size_t)(nseg > 0 ? nseg : 1) * sizeof(int), st));      // now the fill cursors
    fl_fill_kernel<<<grid_rows, wpb * 32, 0, st>>>(npt, ctx->indptr, ctx->indices, ctx->data, W, th, tiles_x, d_bmin,
                                                   d_seg_ptr, d_seg_dst, d_seg_len, fl.blob);
    fl_header_kernel<<<ntiles, 128, 0, st>>>(ntiles, fl.tile_desc, d_hdr_off, d_hdr, fl.blob);
    FL_CUDA(cudaGetLastError());
    FL_CUDA(cudaStreamSynchronize(st));
#undef FL_CUDA
    cleanup();
    fl.tiles_x = tiles_x;
    fl.tiles_y = tiles_y;
    fl.ntiles = ntiles;
    fl.nchunks = nchunks;
    fl.nslot = nslot;
    fl.max_blob_bytes = max_blob;
    fl.ok = true;
    return AI_OK;
}
