// Sliced execution layout (SURVEY.md section 8(a) B6 "derived layouts"): the entries of the tiled
// layout (build_tiled.cu: same coefficients as the canonical CSR) cut into slices of at most
// kSliceMax entries and packed, 32 slices of similar length at a time, into blocks that one warp consumes with one
// lane per slice.  A tile's blocks form one blob moved to shared memory by a single bulk copy (ctx.h).
//
// Order of the slices of a tile: by descending length, within equal length in (bin, position) order.  Adjacent lanes of
// a block that belong to the same segment form a run; a run yields one partial sum per frame.
#include <stdlib.h>

#include <algorithm>
#include <vector>

#include "ctx.h"

namespace {

struct SegLens {                 // padded segment lengths either as an array or as differences of seg_ptr
    const int *len, *ptr;
    __device__ int operator()(int s) const { return len ? len[s] : ptr[s + 1] - ptr[s]; }
};

// A segment of n entries (n a multiple of 4) is cut into k = ceil(n / kSliceMax) slices of 2q or 2q + 2 steps (a step
// = 4 entries; blocks hold an even number of steps), the first r of them the longer ones: slices of a segment differ
// by at most two steps and only the last one carries padding (at most one step), so blocks of slices of equal length
// have almost no empty slots (cutting off full slices and a remainder left 8-19 % of the slots empty).
struct SegCut {
    int k, q, r, n;
    __device__ __forceinline__ int steps(int w) const { return 2 * (q + (w < r ? 1 : 0)); }
    __device__ __forceinline__ int start(int w) const { return 8 * (w * q + min(w, r)); }    // first entry of slice w
    __device__ __forceinline__ int len(int w) const { return min(4 * steps(w), n - start(w)); }   // real entries
};
__device__ __forceinline__ SegCut seg_cut(int n)
{
    SegCut c{0, 0, 0, n};
    if (n <= 0) return c;
    const int pairs = (n / 4 + 1) / 2;
    c.k = (n + kSliceMax - 1) / kSliceMax;
    c.q = pairs / c.k;
    c.r = pairs % c.k;
    return c;
}

// steps of the slice at sorted position i of a tile with cnt[r] slices of r steps (longest first)
__device__ __forceinline__ int slice_steps_at(int i, const int *cnt)
{
    for (int r = kSliceSteps; r >= 1; --r) {
        if (i < cnt[r]) return r;
        i -= cnt[r];
    }
    return 0;
}

// steps of the block whose first slice sits at sorted position i: the longest of its slices, rounded up to an even
// number (the stream kernel consumes two steps per trip without tail predicates; the extra step is zero padding)
__device__ __forceinline__ int block_steps_at(int i, const int *cnt)
{
    return (slice_steps_at(i, cnt) + 1) & ~1;
}

// cnt[1 .. kSliceSteps]: slices of the tile by number of steps; returns their total
__device__ __forceinline__ int tile_slice_counts(const SegLens &L, int s0, int s1, int *cnt)
{
    for (int r = 0; r <= kSliceSteps; ++r) cnt[r] = 0;
    int S = 0;
    for (int s = s0; s < s1; ++s) {
        const SegCut c = seg_cut(L(s));
        if (c.k == 0) continue;
        if (c.r) cnt[2 * c.q + 2] += c.r;
        cnt[2 * c.q] += c.k - c.r;
        S += c.k;
    }
    return S;
}

// per tile: number of slices, number of blocks, bytes of the blob
__global__ void __launch_bounds__(64) slice_plan_kernel(int ntiles, const int *__restrict__ tile_seg_ptr, SegLens L,
                                                        int *__restrict__ tile_nslices, int *__restrict__ tile_nblk,
                                                        int *__restrict__ tile_blob_bytes)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntiles) return;
    int cnt[kSliceSteps + 1];
    const int S = tile_slice_counts(L, tile_seg_ptr[t], tile_seg_ptr[t + 1], cnt);
    const int nblk = (S + 31) / 32;
    int bytes = (4 * (1 + nblk) + 15) / 16 * 16;
    for (int b = 0; b < nblk; ++b) bytes += block_steps_at(32 * b, cnt) * kBlkStepBytes + kBlkMetaBytes;
    tile_nslices[t] = S;
    tile_nblk[t] = nblk;
    tile_blob_bytes[t] = bytes;
}

// per tile (one thread): which (segment, window of 32 entries) every slice is, the runs, the blob header
__global__ void __launch_bounds__(64) slice_assign_kernel(int ntiles, const int *__restrict__ tile_seg_ptr, SegLens L,
                                                          const int *__restrict__ tile_slice_ptr,
                                                          const long long *__restrict__ tile_blob_off,
                                                          int *__restrict__ slice_seg, int *__restrict__ slice_win,
                                                          int *__restrict__ slice_run, int *__restrict__ seg_nruns,
                                                          unsigned char *__restrict__ blob)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntiles) return;
    const int s0 = tile_seg_ptr[t], s1 = tile_seg_ptr[t + 1];
    int cnt[kSliceSteps + 1], pos[kSliceSteps + 1];
    tile_slice_counts(L, s0, s1, cnt);
    int S = 0;
    for (int r = kSliceSteps; r >= 1; --r) { pos[r] = S; S += cnt[r]; }
    const int g0 = tile_slice_ptr[t];
    for (int s = s0; s < s1; ++s) {
        const SegCut c = seg_cut(L(s));
        for (int w = 0; w < c.k; ++w) {                  // slices of equal length: (bin, position) order
            const int i = pos[c.steps(w)]++;
            slice_seg[g0 + i] = s;
            slice_win[g0 + i] = w;
        }
        seg_nruns[s] = 0;
    }
    // runs: adjacent lanes of one block with the same segment; run index counted per segment in slice order
    int run = 0;
    for (int i = 0; i < S; ++i) {
        const int s = slice_seg[g0 + i];
        const bool head = (i & 31) == 0 || slice_seg[g0 + i - 1] != s;
        if (head) run = seg_nruns[s]++;
        slice_run[g0 + i] = run | (head ? (int)0x80000000 : 0);
    }
    // lanes of the run after this one (backwards), longest run of every block -> reduction rounds
    unsigned *hdr = reinterpret_cast<unsigned *>(blob + tile_blob_off[t]);
    const int nblk = (S + 31) / 32;
    hdr[0] = (unsigned)nblk;
    int off = (4 * (1 + nblk) + 15) / 16 * 16;
    for (int b = 0; b < nblk; ++b) {
        const int lo = 32 * b, hi = min(S, lo + 32);
        int rem = 0, maxrun = 1;
        for (int i = hi - 1; i >= lo; --i) {
            const bool last = i == hi - 1 || (slice_run[g0 + i + 1] < 0);
            rem = last ? 0 : rem + 1;
            maxrun = max(maxrun, rem + 1);
            slice_run[g0 + i] |= rem << 24;
        }
        int rounds = 0;
        while ((1 << rounds) < maxrun) ++rounds;
        const int nsteps = block_steps_at(lo, cnt);
        hdr[1 + b] = ((unsigned)(off / 16) << 8) | ((unsigned)rounds << 4) | (unsigned)nsteps;
        off += nsteps * kBlkStepBytes + kBlkMetaBytes;
    }
}

// one thread block per tile: copy the entries of every slice into its lane of its block, write the lane records
__global__ void __launch_bounds__(256) slice_fill_kernel(const int *__restrict__ tile_slice_ptr,
                                                         const long long *__restrict__ tile_blob_off,
                                                         const int *__restrict__ slice_seg,
                                                         const int *__restrict__ slice_win,
                                                         const int *__restrict__ slice_run,
                                                         const int *__restrict__ seg_ptr, const int *__restrict__ seg_slot,
                                                         const float *__restrict__ tcoef,
                                                         const uint16_t *__restrict__ tidx, unsigned char *__restrict__ blob)
{
    const int t = blockIdx.x;
    const int g0 = tile_slice_ptr[t], S = tile_slice_ptr[t + 1] - g0;
    unsigned char *tb = blob + tile_blob_off[t];
    const unsigned *hdr = reinterpret_cast<const unsigned *>(tb);
    for (int w = threadIdx.x; w < S * kSliceSteps; w += blockDim.x) {
        const int i = w / kSliceSteps, step = w % kSliceSteps, b = i >> 5, lane = i & 31;
        const unsigned h = hdr[1 + b];
        const int nsteps = h & 15;
        unsigned char *blk = tb + (size_t)(h >> 8) * 16;
        const int s = slice_seg[g0 + i], win = slice_win[g0 + i];
        const SegCut c = seg_cut(seg_ptr[s + 1] - seg_ptr[s]);
        const int len = 4 * c.steps(win);
        const int seg_end = seg_ptr[s + 1];
        // Adjacent lanes that hold slices of equal length of the same segment (consecutive windows of its entries) share
        // them interleaved: at step j lane q of m reads the four entries 4 * (j * m + q) ... of the m windows, so that
        // the lanes of one segment gather neighbouring pixels in the same step (different rows and columns of the tile
        // -> different shared-memory banks) instead of pixels a whole slice apart.
        int q = 0, m = 1;
        while (q < lane && slice_seg[g0 + i - q - 1] == s && slice_win[g0 + i - q - 1] == win - q - 1 &&
               c.steps(win - q - 1) == c.steps(win))
            ++q;
        while (lane - q + m < 32 && i - q + m < S && slice_seg[g0 + i - q + m] == s &&
               slice_win[g0 + i - q + m] == win - q + m && c.steps(win - q + m) == c.steps(win))
            ++m;
        const int src = seg_ptr[s] + c.start(win - q) + 4 * (step * m + q);
        if (step * 4 < len && src + 4 <= seg_end) {   // the rest stays zero: coefficient 0 at pixel 0 of the tile
            const float4 cf = *reinterpret_cast<const float4 *>(tcoef + src);
            const ushort4 x = *reinterpret_cast<const ushort4 *>(tidx + src);
            reinterpret_cast<float4 *>(blk)[step * 32 + lane] = cf;
            reinterpret_cast<ushort4 *>(blk + (size_t)nsteps * 512)[step * 32 + lane] = x;
        }
        if (step == 0) {
            const int r = slice_run[g0 + i];
            int2 m = make_int2(r & 0x1f000000, 0);
            if (r < 0) {
                const int rem = (r >> 24) & 31;
                double sum = 0.0;      // coefficient sum of the run, fixed order: `count` when every pixel is valid
                for (int j = 0; j <= rem; ++j) {
                    const int wj = slice_win[g0 + i + j];
                    const int bj = seg_ptr[s] + c.start(wj), lj = c.len(wj);
                    for (int e = 0; e < lj; ++e) sum += (double)tcoef[bj + e];
                }
                m.x |= (int)0x80000000 | (seg_slot[s] + (r & kMetaSlotMask));
                m.y = __float_as_int((float)sum);
            }
            reinterpret_cast<int2 *>(blk + (size_t)nsteps * kBlkStepBytes)[lane] = m;
        }
    }
}

// Bank scheduling: the ORDER in which a lane walks its entries is free (it only fixes the order of a compensated sum),
// and the pixel positions are known here -- so choose, slot by slot (slot = step * 4 + entry of the 128-bit load), for
// every lane of a block the not yet placed entry whose shared-memory bank the lanes before it use least in that slot.
// Unscheduled, the 32 lanes of a gather read unrelated pixels and fall into banks at random (2.4 wavefronts per
// gather, which makes the batched kernel shared-memory-bound).  One thread per block of the layout, greedy, one-time.
__global__ void __launch_bounds__(64) slice_schedule_kernel(const long long *__restrict__ tile_blob_off,
                                                            unsigned char *__restrict__ blob)
{
    unsigned char *tb = blob + tile_blob_off[blockIdx.x];
    const unsigned *hdr = reinterpret_cast<const unsigned *>(tb);
    const int nblk = (int)hdr[0];
    for (int b = threadIdx.x; b < nblk; b += blockDim.x) {
        const unsigned h = hdr[1 + b];
        const int nsteps = h & 15, T = nsteps * 4;
        unsigned char *blk = tb + (size_t)(h >> 8) * 16;
        float *coef = reinterpret_cast<float *>(blk);                                   // [step][lane][4]
        unsigned short *idx = reinterpret_cast<unsigned short *>(blk + (size_t)nsteps * 512);
        for (int t = 0; t < T; ++t) {
            unsigned char cnt[32];
            for (int k = 0; k < 32; ++k) cnt[k] = 0;
            for (int lane = 0; lane < 32; ++lane) {
                int best = t, bestc = 1 << 30;
                for (int k = t; k < T && bestc > 0; ++k) {
                    const int at = ((k >> 2) * 32 + lane) * 4 + (k & 3);
                    const unsigned off = idx[at];
                    // a padding entry (coefficient 0 at position 0) reads the same address in every lane: no conflict
                    const int c = (off == 0 && coef[at] == 0.0f) ? 0 : cnt[(off >> 2) & 31];
                    if (c < bestc) { bestc = c; best = k; }
                }
                const int a = ((t >> 2) * 32 + lane) * 4 + (t & 3), z = ((best >> 2) * 32 + lane) * 4 + (best & 3);
                const float cz = coef[z];
                const unsigned short xz = idx[z];
                if (best != t) {
                    coef[z] = coef[a]; idx[z] = idx[a];
                    coef[a] = cz; idx[a] = xz;
                }
                if (!(xz == 0 && cz == 0.0f)) cnt[(xz >> 2) & 31]++;
            }
        }
    }
}

}  // namespace

// Largest blob over all tiles for the segment lengths `seg_len` (padded): decides whether a tile height fits the
// shared-memory ring of the pipelined kernel.
int ai_slice_max_blob(ai_ctx *ctx, int ntiles, const int *tile_seg_ptr, const int *seg_len, cudaStream_t st,
                      int *max_blob)
{
    int *d = nullptr;
    AI_CUDA(ctx, cudaMalloc(&d, (size_t)3 * ntiles * sizeof(int)));
    slice_plan_kernel<<<(ntiles + 63) / 64, 64, 0, st>>>(ntiles, tile_seg_ptr, SegLens{seg_len, nullptr}, d, d + ntiles,
                                                         d + 2 * ntiles);
    std::vector<int> h(ntiles);
    cudaError_t e = cudaMemcpyAsync(h.data(), d + 2 * ntiles, (size_t)ntiles * sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d);
    AI_CUDA(ctx, e);
    *max_blob = 0;
    for (int t = 0; t < ntiles; ++t) *max_blob = std::max(*max_blob, h[t]);
    return AI_OK;
}

// Scratch of the sliced build, alive between its two phases.
struct SliceScratch {
    int *tile_counts = nullptr;       // [3][ntiles] slices, blocks, blob bytes
    int *tile_slice_ptr = nullptr;    // [ntiles+1]
    long long *tile_blob_off = nullptr;
    int *slice_seg = nullptr, *slice_win = nullptr, *slice_run = nullptr;
    std::vector<int> h_nblk, h_bytes;
    std::vector<long long> h_off;
    void release()
    {
        cudaFree(tile_counts); cudaFree(tile_slice_ptr); cudaFree(tile_blob_off);
        cudaFree(slice_seg); cudaFree(slice_win); cudaFree(slice_run);
        tile_counts = tile_slice_ptr = slice_seg = slice_win = slice_run = nullptr;
        tile_blob_off = nullptr;
    }
};

// Phase 1 (needs seg_ptr): slices, runs, blob headers; fills seg_nruns[nseg] so that the caller can assign partial slots.
int ai_build_sliced_plan(ai_ctx *ctx, SliceScratch *sc, int *seg_nruns, cudaStream_t st)
{
    TiledLayout &tl = ctx->tl;
    const int nt = tl.ntiles;
    AI_CUDA(ctx, cudaMalloc(&sc->tile_counts, (size_t)3 * nt * sizeof(int)));
    const SegLens L{nullptr, tl.seg_ptr};
    slice_plan_kernel<<<(nt + 63) / 64, 64, 0, st>>>(nt, tl.tile_seg_ptr, L, sc->tile_counts, sc->tile_counts + nt,
                                                     sc->tile_counts + 2 * nt);
    AI_CUDA(ctx, cudaGetLastError());
    std::vector<int> h(3 * (size_t)nt);
    AI_CUDA(ctx, cudaMemcpyAsync(h.data(), sc->tile_counts, h.size() * sizeof(int), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    std::vector<int> slice_ptr(nt + 1, 0);
    sc->h_off.assign(nt, 0);
    sc->h_nblk.assign(h.begin() + nt, h.begin() + 2 * nt);
    sc->h_bytes.assign(h.begin() + 2 * nt, h.end());
    long long off = 0, nslices = 0;
    tl.max_blob_bytes = 0;
    for (int t = 0; t < nt; ++t) {
        slice_ptr[t] = (int)nslices;
        nslices += h[t];
        sc->h_off[t] = off;
        off += sc->h_bytes[t];
        tl.max_blob_bytes = std::max(tl.max_blob_bytes, sc->h_bytes[t]);
    }
    slice_ptr[nt] = (int)nslices;
    if (nslices > 0x7fffffffLL || off / 16 > 0x7fffffffLL) return ai_fail(ctx, AI_EUNSUPPORTED, "sliced layout too large");
    tl.blob_bytes = off;
    const size_t ns = nslices > 0 ? (size_t)nslices : 1;
    AI_CUDA(ctx, cudaMalloc(&sc->tile_slice_ptr, ((size_t)nt + 1) * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&sc->tile_blob_off, (size_t)nt * sizeof(long long)));
    AI_CUDA(ctx, cudaMalloc(&sc->slice_seg, ns * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&sc->slice_win, ns * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&sc->slice_run, ns * sizeof(int)));
    AI_CUDA(ctx, cudaMalloc(&tl.blob, (size_t)(off > 0 ? off : 16)));
    AI_CUDA(ctx, cudaMemsetAsync(tl.blob, 0, (size_t)(off > 0 ? off : 16), st));
    AI_CUDA(ctx, cudaMemcpyAsync(sc->tile_slice_ptr, slice_ptr.data(), ((size_t)nt + 1) * sizeof(int), cudaMemcpyHostToDevice, st));
    AI_CUDA(ctx, cudaMemcpyAsync(sc->tile_blob_off, sc->h_off.data(), (size_t)nt * sizeof(long long), cudaMemcpyHostToDevice, st));
    slice_assign_kernel<<<(nt + 63) / 64, 64, 0, st>>>(nt, tl.tile_seg_ptr, L, sc->tile_slice_ptr, sc->tile_blob_off,
                                                       sc->slice_seg, sc->slice_win, sc->slice_run, seg_nruns, tl.blob);
    AI_CUDA(ctx, cudaGetLastError());
    AI_CUDA(ctx, cudaStreamSynchronize(st));      // slice_ptr (host vector) was the source of an async copy
    return AI_OK;
}

// Phase 2 (needs seg_slot): the blocks themselves and the longest-first schedule.
int ai_build_sliced_fill(ai_ctx *ctx, SliceScratch *sc, cudaStream_t st)
{
    TiledLayout &tl = ctx->tl;
    const int nt = tl.ntiles;
    slice_fill_kernel<<<nt, 256, 0, st>>>(sc->tile_slice_ptr, sc->tile_blob_off, sc->slice_seg, sc->slice_win,
                                          sc->slice_run, tl.seg_ptr, tl.seg_slot, tl.tcoef, tl.tidx, tl.blob);
    AI_CUDA(ctx, cudaGetLastError());
    if (!ctx->no_schedule) {
        slice_schedule_kernel<<<nt, 64, 0, st>>>(sc->tile_blob_off, tl.blob);
        AI_CUDA(ctx, cudaGetLastError());
    }
    // longest-processing-time-first order of the tiles (host sort of ntiles integers, one-time)
    std::vector<int> order(nt);
    for (int t = 0; t < nt; ++t) order[t] = t;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return sc->h_bytes[a] > sc->h_bytes[b]; });
    std::vector<int4> desc(nt);
    for (int r = 0; r < nt; ++r) {
        const int t = order[r];
        desc[r] = make_int4((int)(sc->h_off[t] / 16), sc->h_bytes[t], ((t / tl.tiles_x) << 16) | (t % tl.tiles_x), sc->h_nblk[t]);
    }
    tl.h_first_desc = static_cast<int4 *>(malloc((size_t)(nt > 0 ? nt : 1) * sizeof(int4)));
    if (!tl.h_first_desc) return ai_fail(ctx, AI_ENOMEM, "host copy of the tile descriptors");
    for (int r = 0; r < nt; ++r) tl.h_first_desc[r] = desc[r];
    AI_CUDA(ctx, cudaMalloc(&tl.blob_desc, (size_t)nt * sizeof(int4)));
    AI_CUDA(ctx, cudaMemcpyAsync(tl.blob_desc, desc.data(), (size_t)nt * sizeof(int4), cudaMemcpyHostToDevice, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    sc->release();
    return AI_OK;
}

SliceScratch *ai_slice_scratch_new() { return new SliceScratch(); }
void ai_slice_scratch_delete(SliceScratch *sc)
{
    if (!sc) return;
    sc->release();
    delete sc;
}
