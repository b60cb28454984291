// Kernels and host steps shared by the two builders of the TILED execution layout (build_tiled.cu: 1D, from the per-pixel
// spans; build_2d.cu: bidimensional, from a sorted list of entries).  Everything is `static`: each translation unit gets
// its own copy.
#pragma once
#include <algorithm>
#include <vector>

#include "ctx.h"

namespace {

// exclusive scan of ceil(len / pad) * pad over n elements, one block; out[n] = total
__global__ void __launch_bounds__(1024) scan_pad_kernel(int n, const int *__restrict__ len, int pad,
                                                        int *__restrict__ out, long long *__restrict__ total)
{
    __shared__ long long warp_sum[32];
    __shared__ long long carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int base = 0; base < n; base += blockDim.x) {
        int i = base + threadIdx.x;
        long long v = i < n ? (long long)((len[i] + pad - 1) / pad) * pad : 0;
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
            warp_sum[lane] = w;
        }
        __syncthreads();
        long long before = carry + (wid > 0 ? warp_sum[wid - 1] : 0) + (x - v);
        if (i < n) out[i] = (int)before;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry = before + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        *total = carry;
        out[n] = (int)carry;
    }
}

// per-segment coefficient sum (fp64, fixed order): the segment's `count` contribution when all its pixels are valid
__global__ void __launch_bounds__(256) seg_sum_kernel(int nseg, const int *__restrict__ seg_ptr,
                                                      const float *__restrict__ tcoef, double *__restrict__ seg_csum)
{
    int s = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (s >= nseg) return;
    double a = 0.0;
    for (int k = seg_ptr[s] + (threadIdx.x & 31); k < seg_ptr[s + 1]; k += 32) a += (double)tcoef[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if ((threadIdx.x & 31) == 0) seg_csum[s] = a;
}

// padded segment lengths: every segment a multiple of kSegPad entries (128-bit coefficient loads), every tile a
// multiple of 8 entries so that the tile's slice of the 16-bit index array starts on a 16-byte boundary (bulk copies)
__global__ void __launch_bounds__(128) pad_segments_kernel(int ntiles, const int *__restrict__ tile_seg_ptr,
                                                           int *__restrict__ seg_len, int *__restrict__ tile_entries)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntiles) return;
    const int s0 = tile_seg_ptr[t], s1 = tile_seg_ptr[t + 1];
    int total = 0;
    for (int s = s0; s < s1; ++s) {
        int p = (seg_len[s] + kSegPad - 1) / kSegPad * kSegPad;
        seg_len[s] = p;
        total += p;
    }
    if (s1 > s0 && (total & 7)) {
        seg_len[s1 - 1] += 8 - (total & 7);
        total += 8 - (total & 7);
    }
    tile_entries[t] = total;
}

// {first entry, padded end, partial slot, coefficient sum as float bits} of every segment: one 128-bit load.  The
// records of a tile are written in order of descending segment length (rank by counting, ties by bin), so that the
// lane groups of one warp, which take consecutive records, work on segments of similar length.
__global__ void __launch_bounds__(256) seg_meta_kernel(int ntiles, const int *__restrict__ tile_seg_ptr,
                                                       const int *__restrict__ seg_ptr, const int *__restrict__ seg_slot,
                                                       const double *__restrict__ seg_csum,
                                                       int4 *__restrict__ seg_meta, int4 *__restrict__ tile_desc)
{
    const int t = blockIdx.x;
    if (t >= ntiles) return;
    const int s0 = tile_seg_ptr[t], s1 = tile_seg_ptr[t + 1];
    for (int s = s0 + threadIdx.x; s < s1; s += blockDim.x) {
        const int len = seg_ptr[s + 1] - seg_ptr[s];
        int rank = 0;
        for (int o = s0; o < s1; ++o) {
            const int lo = seg_ptr[o + 1] - seg_ptr[o];
            rank += (lo > len || (lo == len && o < s)) ? 1 : 0;
        }
        seg_meta[s0 + rank] = make_int4(seg_ptr[s], seg_ptr[s + 1], seg_slot[s], __float_as_int((float)seg_csum[s]));
    }
    // {first entry, number of entries, first segment, number of segments} of the tile
    if (threadIdx.x == 0) tile_desc[t] = make_int4(seg_ptr[s0], seg_ptr[s1] - seg_ptr[s0], s0, s1 - s0);
}

}  // namespace

// Last steps of a tiled build, once seg_ptr / seg_slot / seg_csum / tile_seg_ptr are final: the per-segment records of
// the one-block-per-tile kernel and the longest-first order of the tiles.
static int ai_tiled_finalize(ai_ctx *ctx, cudaStream_t st)
{
    TiledLayout &tl = ctx->tl;
    const size_t nseg_alloc = tl.nseg > 0 ? tl.nseg : 1;
    AI_CUDA(ctx, cudaMalloc(&tl.seg_meta, nseg_alloc * sizeof(int4)));
    AI_CUDA(ctx, cudaMalloc(&tl.tile_desc, (size_t)tl.ntiles * sizeof(int4)));
    AI_CUDA(ctx, cudaMalloc(&tl.tile_order, (size_t)tl.ntiles * sizeof(int)));
    seg_meta_kernel<<<tl.ntiles, 256, 0, st>>>(tl.ntiles, tl.tile_seg_ptr, tl.seg_ptr, tl.seg_slot, tl.seg_csum,
                                               tl.seg_meta, tl.tile_desc);
    AI_CUDA(ctx, cudaGetLastError());
    // longest-processing-time-first order of the tiles (host sort of ntiles integers, one-time)
    std::vector<int4> desc(tl.ntiles);
    AI_CUDA(ctx, cudaMemcpyAsync(desc.data(), tl.tile_desc, (size_t)tl.ntiles * sizeof(int4), cudaMemcpyDeviceToHost, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    std::vector<int> order(tl.ntiles);
    for (int t = 0; t < tl.ntiles; ++t) order[t] = t;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return desc[a].y > desc[b].y; });
    // tile_desc is kept in the same longest-first order as tile_order (the pipelined kernel indexes both by rank)
    std::vector<int4> desc_lpt(tl.ntiles);
    for (int r = 0; r < tl.ntiles; ++r) desc_lpt[r] = desc[order[r]];
    AI_CUDA(ctx, cudaMemcpyAsync(tl.tile_order, order.data(), (size_t)tl.ntiles * sizeof(int), cudaMemcpyHostToDevice, st));
    AI_CUDA(ctx, cudaMemcpyAsync(tl.tile_desc, desc_lpt.data(), (size_t)tl.ntiles * sizeof(int4), cudaMemcpyHostToDevice, st));
    AI_CUDA(ctx, cudaStreamSynchronize(st));
    return AI_OK;
}
