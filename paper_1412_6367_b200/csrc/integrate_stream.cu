// The TMA-streamed kernels of the TILED layout -- the CSR SpMV of PAPER.md:174-188 on B200.
//
// tiled_stream_kernel: the whole hot path of ONE frame of 32-bit pixels in one launch (the configuration the headline
// metric is quoted on; corrected frames come here through the pre-pass of integrate_prep.cu).
//   - one persistent block per SM, 1 producer warp + kStreamCons consumer warps; float frames are gathered straight
//     from the TMA tile, integer frames are converted at gather time ("casted from integer to float");
//   - one ring whose stage holds a tile of the frame AND that tile's blob of the matrix, one full / empty mbarrier pair
//     per stage; the descriptor of the tile in a stage sits next to the barriers;
//   - tiles longest first: the first kStreamFirst of every block are dealt statically and travel in the kernel
//     parameters (their copies leave before any global load has returned), the rest are drawn from a ticket counter;
//   - pixel positions of two entries are rebased with one packed 16-bit add: the tile buffers live in the first 64 KB of
//     the shared window, so a position's low half-word is its whole shared address;
//   - H5 fused: the last blocks to arrive at a counter add the partials up (fixed order) and write the three outputs;
//   - programmatic dependent launch: the next launch's prologue and first blobs overlap this launch's tail.
// tiled_bstream_kernel: batches of plain 32-bit frames, the blob of a tile loaded once per chunk of frames, two frames
// consumed per pass.
#include <stdlib.h>

#include "pipe_common.cuh"
#include "tiled_common.cuh"

namespace {

constexpr int kStreamCons = 16;                      // consumer warps: the single-frame kernel is bound by the memory
                                                     // system, 16 keep up with it and arrive at barriers sooner than 20 or 24
constexpr int kStreamThreads = 32 * (1 + kStreamCons);
constexpr int kStreamFirst = 3;                      // descriptors per block passed by value
constexpr int kStreamMaxGrid = 160;
constexpr int kStreamMaxStages = 8;
constexpr int kStreamBarBytes = 512;                 // full[8] + empty[8], block-wide state, per-stage descriptors
constexpr int kStreamDescOffset = 256;

struct StreamFirstDescs {
    int4 d[kStreamFirst][kStreamMaxGrid];
};

struct StreamParams {
    const int4 *blob_desc;       // longest first: {blob offset / 16, blob bytes, tile row << 16 | column, blocks}
    const unsigned char *blob;
    int tile_h, ntiles, nslot;
    int stages, mat_stage_bytes, img_stage_bytes, hdr_bytes;
    int dyn_base;                // rank of the first tile handed out by ticket (the ones before are dealt statically)
    int launch_index;            // launches of this context so far, modulo 8 (development trace only)
    int track_all;               // float frames: every block skips non-finite pixels and accumulates count
    void *partials;
    // H5 fused behind a grid-wide barrier (every block is resident: one per SM, grid <= number of SMs)
    unsigned long long *grid_sync;     // [0] arrivals of all launches of this context, never reset; [1] tile tickets
    const int *bin_slot_ptr;
    const double *range;
    int npt;
    float empty;
    float *radial, *intensity, *sum_signal, *count;
};

// ---- development aid (-DAI_PIPE_TRACE): per (block, tile, warp) globaltimer stamps ------------------------------------
#ifdef AI_PIPE_TRACE
__device__ long long *g_strace = nullptr;          // [grid][16 tiles][32 warps][4]
__device__ int g_strace_div = 1;                   // trace every g_strace_div-th tile
__device__ __forceinline__ long long strace_now()
{
    long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
#define AI_STRACE_AT(row, slot, val)                                                                            \
    do {                                                                                                        \
        if (g_strace && (threadIdx.x & 31) == 0)                                                                \
            g_strace[(((((size_t)p.launch_index * gridDim.x + blockIdx.x) * 16 + (row)) * 32) + (threadIdx.x >> 5)) * 4 + (slot)] = (val); \
    } while (0)
// tiles: every g_strace_div-th one, rows 0..13; rows 14 and 15 hold the kernel-level stamps
#define AI_STRACE(item, slot, val)                                                                              \
    do {                                                                                                        \
        if ((item) % g_strace_div == 0 && (item) / g_strace_div < 14) AI_STRACE_AT((item) / g_strace_div, slot, val); \
    } while (0)
#else
#define AI_STRACE(item, slot, val) do { } while (0)
#define AI_STRACE_AT(row, slot, val) do { } while (0)
#define strace_now() 0
#endif

// n-th tile of this block: tiles (longest first) are dealt to the blocks in snake order
__device__ __forceinline__ int stream_item_at(int n)
{
    return n * gridDim.x + ((n & 1) ? gridDim.x - 1 - blockIdx.x : blockIdx.x);
}

__device__ __forceinline__ float lds_f32(unsigned addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ int lds_s32(unsigned addr)
{
    int v;
    asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

// pixel values of the four entries of one step; x holds four 16-bit byte offsets into the tile.  PACKED: `base` = low
// half-word of the tile's shared address in both halves (tile buffers inside the first 64 KB of the shared window: one
// add rebases two positions); otherwise `base` = the tile's shared address.
template <int DT, bool PACKED = true>
__device__ __forceinline__ float4 stream_gather4(const uint2 &x, unsigned base)
{
    unsigned a0, a1, a2, a3;
    if constexpr (PACKED) {
        const unsigned p0 = x.x + base, p1 = x.y + base;
        a0 = p0 & 0xffffu; a1 = p0 >> 16; a2 = p1 & 0xffffu; a3 = p1 >> 16;
    } else {
        a0 = base + (x.x & 0xffffu); a1 = base + (x.x >> 16); a2 = base + (x.y & 0xffffu); a3 = base + (x.y >> 16);
    }
    if constexpr (DT == AI_F32) {
        return make_float4(lds_f32(a0), lds_f32(a1), lds_f32(a2), lds_f32(a3));
    } else if constexpr (DT == AI_I32) {
        return make_float4((float)lds_s32(a0), (float)lds_s32(a1), (float)lds_s32(a2), (float)lds_s32(a3));
    } else {
        return make_float4((float)(unsigned)lds_s32(a0), (float)(unsigned)lds_s32(a1), (float)(unsigned)lds_s32(a2),
                           (float)(unsigned)lds_s32(a3));
    }
}

// lanes of a run are adjacent: suffix sums by doubling, the head of the run ends with the run's total
template <int ACC, bool TRACK>
__device__ __forceinline__ void stream_finish_block(Accum<ACC> &S, Accum<ACC> &C, const int2 &m, int rounds, void *part_f)
{
    const int rem = (m.x >> 24) & 31;
    for (int r = 0; r < rounds; ++r) {
        const int d = 1 << r;
        Accum<ACC> S_o = S, C_o = C;
        S_o.shfl_down(d);
        if constexpr (TRACK) C_o.shfl_down(d);
        if (rem >= d) {
            S.absorb(S_o);
            if constexpr (TRACK) C.absorb(C_o);
        }
    }
    if (m.x < 0) store_partial<ACC>(part_f, m.x & kMetaSlotMask, S, C, TRACK, (double)__int_as_float(m.y));
}

// Kahan mode, cheaper epilogue: a lane's four compensated sums are carried over to ONE double (s - c is exact in
// fp64), the lanes of a run are added in fp64 (exact to 2^-53: nothing the fp32 two-sum merge kept is lost) and the
// run's total goes out as the same (hi, lo) float pair.  A third of the instructions of the fp32 merges.
__device__ __forceinline__ double kahan_total_d(const AccumQ<AI_ACC_F32_KAHAN> &q)
{
    return (((double)q.a.s - (double)q.a.c) + ((double)q.b.s - (double)q.b.c)) +
           (((double)q.c.s - (double)q.c.c) + ((double)q.d.s - (double)q.d.c));
}
template <bool TRACK>
__device__ __forceinline__ void stream_finish_d(double S, double C, const int2 &m, int rounds, void *part_f)
{
    const int rem = (m.x >> 24) & 31;
    for (int r = 0; r < rounds; ++r) {
        const int d = 1 << r;
        const double S_o = __shfl_down_sync(AI_FULL_MASK, S, d);
        double C_o = 0.0;
        if constexpr (TRACK) C_o = __shfl_down_sync(AI_FULL_MASK, C, d);
        if (rem >= d) {
            S += S_o;
            if constexpr (TRACK) C += C_o;
        }
    }
    if (m.x < 0) {
        if constexpr (!TRACK) C = (double)__int_as_float(m.y);       // every pixel valid: the build-time coefficient sum
        const float s_hi = (float)S, c_hi = (float)C;
        reinterpret_cast<float4 *>(part_f)[m.x & kMetaSlotMask] =
            make_float4(s_hi, (float)(S - (double)s_hi), c_hi, (float)(C - (double)c_hi));
    }
}

// One block of 32 slices against the staged tile: lane = slice, two steps (8 entries) per trip, the loads of the next
// trip issued before the current one is consumed.  Blocks hold an even number of steps (build_sliced.cu) and the
// stage has slack behind the blob, so the look-ahead needs no predicate.  Float frames are not screened: a
// non-finite lane sum anywhere in the warp means a non-finite pixel may have been gathered; nothing is stored and
// true is returned (the caller repeats the block with stream_block_tracked).
template <int DT, int ACC, bool PACKED = true>
__device__ __noinline__ bool stream_block(unsigned rebase, const unsigned char *blob, unsigned h, void *part_f, int lane)
{
    const int nsteps = h & 15, rounds = (h >> 4) & 7;
    const unsigned char *blk = blob + (size_t)(h >> 8) * 16;
    const float4 *cp = reinterpret_cast<const float4 *>(blk) + lane;
    const uint2 *xp = reinterpret_cast<const uint2 *>(blk + nsteps * 512) + lane;
    const int2 m = reinterpret_cast<const int2 *>(blk + nsteps * kBlkStepBytes)[lane];
    AccumQ<ACC> S2, C2;
    float4 c0 = cp[0], c1 = cp[32];
    uint2 x0 = xp[0], x1 = xp[32];
#pragma unroll 1
    for (int j = 2; j <= nsteps; j += 2) {
        const float4 n0 = cp[j * 32], n1 = cp[j * 32 + 32];
        const uint2 y0 = xp[j * 32], y1 = xp[j * 32 + 32];
        const float4 v0 = stream_gather4<DT, PACKED>(x0, rebase), v1 = stream_gather4<DT, PACKED>(x1, rebase);
        accumulate4<ACC, false>(c0, v0, S2, C2);
        accumulate4<ACC, false>(c1, v1, S2, C2);
        c0 = n0; c1 = n1; x0 = y0; x1 = y1;
    }
    if constexpr (ACC == AI_ACC_F32_KAHAN) {
        const double S = kahan_total_d(S2);
        if constexpr (DT == AI_F32) {
            if (__any_sync(AI_FULL_MASK, !finite_f((float)S))) return true;
        }
        stream_finish_d<false>(S, 0.0, m, rounds, part_f);
    } else {
        Accum<ACC> S = S2.total(), C = C2.total();
        if constexpr (DT == AI_F32) {
            if (__any_sync(AI_FULL_MASK, !finite_f((float)S.s))) return true;
        }
        stream_finish_block<ACC, false>(S, C, m, rounds, part_f);
    }
    return false;
}

// the same block with non-finite pixels skipped and count accumulated (float frames: the pre-pass marks invalid
// pixels with NaN, raw frames may carry NaN / Inf); same two-steps-per-trip pipeline
template <int ACC, bool PACKED = true>
__device__ __noinline__ void stream_block_tracked(unsigned rebase, const unsigned char *blob, unsigned h, void *part_f,
                                                  int lane)
{
    const int nsteps = h & 15, rounds = (h >> 4) & 7;
    const unsigned char *blk = blob + (size_t)(h >> 8) * 16;
    const float4 *cp = reinterpret_cast<const float4 *>(blk) + lane;
    const uint2 *xp = reinterpret_cast<const uint2 *>(blk + nsteps * 512) + lane;
    const int2 m = reinterpret_cast<const int2 *>(blk + nsteps * kBlkStepBytes)[lane];
    AccumQ<ACC> S2, C2;
    float4 c0 = cp[0], c1 = cp[32];
    uint2 x0 = xp[0], x1 = xp[32];
#pragma unroll 1
    for (int j = 2; j <= nsteps; j += 2) {
        const float4 n0 = cp[j * 32], n1 = cp[j * 32 + 32];
        const uint2 y0 = xp[j * 32], y1 = xp[j * 32 + 32];
        const float4 v0 = stream_gather4<AI_F32, PACKED>(x0, rebase), v1 = stream_gather4<AI_F32, PACKED>(x1, rebase);
        accumulate4<ACC, true>(c0, v0, S2, C2);
        accumulate4<ACC, true>(c1, v1, S2, C2);
        c0 = n0; c1 = n1; x0 = y0; x1 = y1;
    }
    if constexpr (ACC == AI_ACC_F32_KAHAN) {
        stream_finish_d<true>(kahan_total_d(S2), kahan_total_d(C2), m, rounds, part_f);
    } else {
        Accum<ACC> S = S2.total(), C = C2.total();
        stream_finish_block<ACC, true>(S, C, m, rounds, part_f);
    }
}

// Batches (H6): the same block against the tiles of TWO frames at once.  Coefficients and positions are loaded and
// unpacked once and serve both frames; the two sets of accumulators double the independent work per lane.  Returns
// true (nothing stored) if a non-finite lane sum shows that either tile may hold a non-finite pixel.
template <int DT, int ACC>
__device__ __noinline__ bool stream_block2(unsigned tile_a, unsigned tile_b, const unsigned char *blob, unsigned h,
                                           void *part_a, void *part_b, int lane)
{
    const int nsteps = h & 15, rounds = (h >> 4) & 7;
    const unsigned char *blk = blob + (size_t)(h >> 8) * 16;
    const float4 *cp = reinterpret_cast<const float4 *>(blk) + lane;
    const uint2 *xp = reinterpret_cast<const uint2 *>(blk + nsteps * 512) + lane;
    const int2 m = reinterpret_cast<const int2 *>(blk + nsteps * kBlkStepBytes)[lane];
    AccumQ<ACC> SA, SB, C2;
    float4 c0 = cp[0], c1 = cp[32];
    uint2 x0 = xp[0], x1 = xp[32];
#pragma unroll 1
    for (int j = 2; j <= nsteps; j += 2) {
        const float4 n0 = cp[j * 32], n1 = cp[j * 32 + 32];
        const uint2 y0 = xp[j * 32], y1 = xp[j * 32 + 32];
        const float4 a0 = stream_gather4<DT, false>(x0, tile_a), b0 = stream_gather4<DT, false>(x0, tile_b);
        const float4 a1 = stream_gather4<DT, false>(x1, tile_a), b1 = stream_gather4<DT, false>(x1, tile_b);
        accumulate4<ACC, false>(c0, a0, SA, C2);
        accumulate4<ACC, false>(c0, b0, SB, C2);
        accumulate4<ACC, false>(c1, a1, SA, C2);
        accumulate4<ACC, false>(c1, b1, SB, C2);
        c0 = n0; c1 = n1; x0 = y0; x1 = y1;
    }
    if constexpr (ACC == AI_ACC_F32_KAHAN) {
        const double Sa = kahan_total_d(SA), Sb = kahan_total_d(SB);
        if constexpr (DT == AI_F32) {
            if (__any_sync(AI_FULL_MASK, !finite_f((float)Sa) || !finite_f((float)Sb))) return true;
        }
        stream_finish_d<false>(Sa, 0.0, m, rounds, part_a);
        stream_finish_d<false>(Sb, 0.0, m, rounds, part_b);
    } else {
        Accum<ACC> Sa = SA.total(), Sb = SB.total(), C = C2.total();
        if constexpr (DT == AI_F32) {
            if (__any_sync(AI_FULL_MASK, !finite_f((float)Sa.s) || !finite_f((float)Sb.s))) return true;
        }
        Accum<ACC> Ca = C;
        stream_finish_block<ACC, false>(Sa, Ca, m, rounds, part_a);
        stream_finish_block<ACC, false>(Sb, C, m, rounds, part_b);
    }
    return false;
}

template <int DT, int ACC>
__global__ void __launch_bounds__(kStreamThreads, 1) tiled_stream_kernel(const __grid_constant__ CUtensorMap tmap,
                                                                         const __grid_constant__ StreamFirstDescs first,
                                                                         const StreamParams p)
{
    // [tile stages][barriers, per-stage tile descriptors][matrix stages]
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *img_base = smem;
    unsigned char *hdr = smem + (size_t)p.stages * p.img_stage_bytes;
    uint64_t *full = reinterpret_cast<uint64_t *>(hdr);              // tile + blob landed (complete_tx)
    uint64_t *empty = full + kStreamMaxStages;                        // every consumer warp is done with the stage
    int4 *stage_desc = reinterpret_cast<int4 *>(hdr + kStreamDescOffset);   // descriptor of the tile in each stage
    unsigned char *mat_base = hdr + p.hdr_bytes;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    AI_STRACE_AT(15, 0, strace_now());

    // Tiles, longest first: the first npre of every block are dealt statically (snake order; their descriptors came
    // with the launch), the rest are handed out by a ticket counter to whichever block has a free stage -- the blocks
    // do not finish their static shares at the same time (the memory system serves them unevenly).
    int npre = 0;
    while (npre < min(kStreamFirst, p.stages) && stream_item_at(npre) < p.ntiles) ++npre;

    // Launch chain (programmatic dependent launch): this grid may start while the previous kernel of the stream is
    // still running.  Nothing that kernel may still read or write is touched before griddepcontrol.wait: until then
    // only the matrix (static since ai_build_csr) is fetched -- the blobs of the block's first tiles -- together with
    // barriers and the tensor map; the frame is read, tickets are drawn and the partials are written after it.
    auto issue_blob = [&](int stage, const int4 &d) {
        stage_desc[stage] = d;
        mbar_arrive_expect_tx(full + stage, (uint32_t)(p.img_stage_bytes + d.y));
        bulk_g2s(mat_base + (size_t)stage * p.mat_stage_bytes, p.blob + (size_t)d.x * 16, (uint32_t)d.y, full + stage);
    };
    auto issue_tile = [&](int stage, const int4 &d) {
        unsigned char *tile = img_base + (size_t)stage * p.img_stage_bytes;
        const int ty = d.z >> 16, tx = d.z & 0xffff;
        tma_box(tile, &tmap, tx * kTileW, ty * p.tile_h, 0, full + stage);
        tma_box(tile + p.img_stage_bytes / 2, &tmap, tx * kTileW + 32, ty * p.tile_h, 0, full + stage);
    };

    if (threadIdx.x == 0) {
        // the packed rebase needs every tile buffer inside the first 64 KB of the shared window
        if (smem_u32(img_base) + (unsigned)(p.stages * p.img_stage_bytes) > 0x10000u) __trap();
        for (int s = 0; s < kStreamMaxStages; ++s) {
            mbar_init(full + s, 1);
            mbar_init(empty + s, kStreamCons);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        // the tensor map is first used after the grid dependency has resolved: have the TMA unit fetch it now
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap) : "memory");
        // first blobs, from descriptors that came with the launch: in flight before any global load returns
        int stage = 0;
        for (int n = 0; n < npre; ++n) {
            const int4 d = first.d[n][blockIdx.x];
            if (d.w == 0) continue;
            issue_blob(stage++, d);
        }
    }
    // static data read late in the kernel, pulled into L2 now: the descriptors of the ticketed tiles (each block its
    // share of the array) and the slot ranges of the bins (H5)
    for (int k = p.dyn_base + (blockIdx.x * kStreamThreads + threadIdx.x) * 8; k < p.ntiles; k += gridDim.x * kStreamThreads * 8)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(p.blob_desc + k));
    for (int k = threadIdx.x * 32; k <= p.npt; k += kStreamThreads * 32)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(p.bin_slot_ptr + k));
    // the next kernel of the stream may be scheduled as SMs free up
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    AI_STRACE_AT(14, 1, strace_now());
    if (threadIdx.x == 0) {
        int stage = 0;
        for (int n = 0; n < npre; ++n) {
            const int4 d = first.d[n][blockIdx.x];
            if (d.w == 0) continue;
            issue_tile(stage++, d);
        }
    }
    __syncthreads();
    AI_STRACE_AT(15, 1, strace_now());

    Ring r;
    if (warp == 0) {
        // ===== producer ================================================================================================
        int issued = 0;
        for (int n = 0; n < npre; ++n) {                  // stages taken by the static tiles
            if (first.d[n][blockIdx.x].w == 0) continue;
            ++issued;
            r.next(p.stages);
        }
        // Ticketed tiles, two draws ahead so that neither the atomic nor the descriptor load is waited for: in every
        // trip lane 0 takes the descriptor loaded in the previous trip, loads the one for the ticket drawn in the
        // previous trip and draws a new ticket; only the block count is shared with the warp (uniform control flow).
        const unsigned long long nticket = p.dyn_base < p.ntiles ? (unsigned long long)(p.ntiles - p.dyn_base) : 0ULL;
        auto fetch = [&](unsigned long long t) {
            return t < nticket ? __ldg(p.blob_desc + p.dyn_base + (int)t) : make_int4(0, 0, 0, -1);
        };
        unsigned long long t_next = ~0ULL;
        int4 d_next = make_int4(0, 0, 0, -1);
        if (lane == 0 && nticket) {
            const unsigned long long t0 = atomicAdd(p.grid_sync + 1, 1ULL);
            t_next = atomicAdd(p.grid_sync + 1, 1ULL);
            d_next = fetch(t0);
        }
        int n = npre;
        while (true) {
            const int4 d = d_next;
            if (lane == 0 && nticket) {
                d_next = fetch(t_next);
                t_next = atomicAdd(p.grid_sync + 1, 1ULL);
            }
            const int nblk = __shfl_sync(AI_FULL_MASK, d.w, 0);
            if (nblk < 0) break;
            if (nblk == 0) continue;                      // tile without entries: never published
            AI_STRACE(n, 0, strace_now());
            if (issued >= p.stages) mbar_wait(empty + r.stage, r.parity ^ 1u);
            if (lane == 0) {
                issue_blob(r.stage, d);
                issue_tile(r.stage, d);
            }
            AI_STRACE(n, 1, strace_now());
            ++issued;
            ++n;
            r.next(p.stages);
        }
        // no tile left: a descriptor with a negative block count ends the consumers' loop
        if (issued >= p.stages) mbar_wait(empty + r.stage, r.parity ^ 1u);
        if (lane == 0) {
            stage_desc[r.stage] = make_int4(0, 0, 0, -1);
            mbar_arrive(full + r.stage);
        }
    } else {
        // ===== consumers: a tile's blocks are dealt round-robin to the warps, continuing across tiles ===================
        const int cw = warp - 1;
        int firstb = cw;
        for (int n = 0;; ++n) {
            // every warp waits on and arrives at every stage, also when it holds no block of the tile: no warp is
            // ever a whole phase away from a barrier
            AI_STRACE(n, 0, strace_now());
            mbar_wait(full + r.stage, r.parity);
            AI_STRACE(n, 1, strace_now());
            const int4 d = stage_desc[r.stage];
            if (d.w < 0) break;
            if (firstb < d.w) {
                const unsigned char *blob = mat_base + (size_t)r.stage * p.mat_stage_bytes;
                const unsigned *bh = reinterpret_cast<const unsigned *>(blob) + 1;
                const unsigned rebase = (smem_u32(img_base + (size_t)r.stage * p.img_stage_bytes) & 0xffffu) * 0x10001u;
                for (int b = firstb; b < d.w; b += kStreamCons) {
                    const unsigned h = bh[b];
                    if constexpr (DT == AI_F32) {
                        // track_all: the frame comes from the correction pre-pass and is expected to hold NaN marks
                        if (p.track_all || stream_block<DT, ACC>(rebase, blob, h, p.partials, lane))
                            stream_block_tracked<ACC>(rebase, blob, h, p.partials, lane);
                    } else {
                        stream_block<DT, ACC>(rebase, blob, h, p.partials, lane);
                    }
                }
                __syncwarp();
                AI_STRACE(n, 2, strace_now());
                AI_STRACE(n, 3, (long long)((d.w - firstb + kStreamCons - 1) / kStreamCons));
            }
            if (lane == 0) mbar_arrive(empty + r.stage);
            firstb -= d.w % kStreamCons;
            if (firstb < 0) firstb += kStreamCons;
            r.next(p.stages);
        }
    }
    AI_STRACE_AT(15, 2, strace_now());

    // ===== H5: the last blocks to finish add up the partials ===========================================================
    // Every block publishes its partials (block barrier, then one thread: fence + atomic arrival).  A launch adds
    // exactly gridDim.x arrivals to the context's counter, so old / gridDim.x is the launch's generation and
    // old % gridDim.x the block's place in the order of arrival.  All but the last `nfin` blocks to arrive leave at once
    // -- their SMs go to the next kernel of the stream; the last ones wait for the stragglers among themselves (all
    // blocks of the grid are resident: one per SM), then share the bins: one warp per bin, fixed summation order.
    volatile int *fin_rank = reinterpret_cast<volatile int *>(empty + kStreamMaxStages);   // spare bytes of the header
    const int nwarps = kStreamThreads / 32;
    const int nfin = min((int)gridDim.x, max(1, (p.npt + nwarps - 1) / nwarps));           // one bin per warp if possible
    unsigned long long target = 0;
    __syncthreads();
    if (threadIdx.x == 0) {
        // release: the block's partials (ordered before this thread by the barrier above) are visible to whoever
        // observes the arrival; acquire: the last block to arrive sees everybody's
        unsigned long long old;
        asm volatile("atom.add.acq_rel.gpu.global.u64 %0, [%1], 1;" : "=l"(old) : "l"(p.grid_sync) : "memory");
        const int place = (int)(old % gridDim.x);
        target = (old / gridDim.x + 1ULL) * gridDim.x;
        if (old + 1 == target) {                                 // the last block to arrive has nothing to wait for,
            target = 0;
            p.grid_sync[1] = 0ULL;                               // and every producer is done: tickets start over
        }
        *fin_rank = place >= (int)gridDim.x - nfin ? place - ((int)gridDim.x - nfin) : -1;
    }
    __syncthreads();
    const int rank = *fin_rank;
    if (rank < 0) return;
    // the slot ranges of the warp's first two bins are fetched while thread 0 waits for the stragglers
    const int stride = nfin * nwarps;
    int b = rank + nfin * warp;
    int beg0 = 0, end0 = 0, beg1 = 0, end1 = 0;
    if (b < p.npt) { beg0 = __ldg(p.bin_slot_ptr + b); end0 = __ldg(p.bin_slot_ptr + b + 1); }
    if (b + stride < p.npt) { beg1 = __ldg(p.bin_slot_ptr + b + stride); end1 = __ldg(p.bin_slot_ptr + b + stride + 1); }
    if (threadIdx.x == 0 && target) {
        unsigned spin = 0;
        while (true) {
            unsigned long long now;
            asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(now) : "l"(p.grid_sync) : "memory");
            if (now >= target) break;
            if (++spin > (1u << 24)) __trap();               // a lost block traps instead of hanging the device
        }
    }
    __syncthreads();
    AI_STRACE_AT(15, 3, strace_now());
    while (b < p.npt) {
        const bool two = b + stride < p.npt;
        const int bn = b + 2 * stride;
        int nb0 = 0, ne0 = 0, nb1 = 0, ne1 = 0;
        if (bn < p.npt) { nb0 = __ldg(p.bin_slot_ptr + bn); ne0 = __ldg(p.bin_slot_ptr + bn + 1); }
        if (bn + stride < p.npt) { nb1 = __ldg(p.bin_slot_ptr + bn + stride); ne1 = __ldg(p.bin_slot_ptr + bn + stride + 1); }
        finish_bins<ACC>(p.partials, b, beg0, end0, two, b + stride, beg1, end1, lane, p.empty, p.intensity, p.sum_signal,
                         p.count);
        if (lane == 0 && p.radial) {
            const double u0 = p.range[0], delta = (p.range[1] - p.range[0]) / (double)p.npt;
            p.radial[b] = (float)(u0 + ((double)b + 0.5) * delta);
            if (two) p.radial[b + stride] = (float)(u0 + ((double)(b + stride) + 0.5) * delta);
        }
        b = bn; beg0 = nb0; end0 = ne0; beg1 = nb1; end1 = ne1;
    }
    AI_STRACE_AT(14, 0, strace_now());
}

// ---- batches (H6): tiled_bstream_kernel ---------------------------------------------------------------------------------
// A work item = (tile, chunk of consecutive frames): the tile's blob is loaded ONCE into a matrix stage and serves
// every frame of the chunk (the batched variant that amortises the matrix read across frames); the frames' tiles stream
// through a ring of image stages and are consumed two frames at a time (stream_block2).  Writes one partial per run
// and frame; tiled_stage2_kernel adds them up.
constexpr int kBatchCons = 20;                       // consumer warps: the batch kernel is bound by the consumers' issue rate
constexpr int kBatchThreads = 32 * (1 + kBatchCons);
constexpr int kBatchMaxImgStages = 8;
constexpr int kBatchMaxMatStages = 2;

struct BatchParams {
    const int4 *blob_desc;
    const unsigned char *blob;
    int tile_h, ntiles, nslot;
    int img_stages, mat_stages, img_stage_bytes, mat_stage_bytes, hdr_bytes;
    int nframes, frames_per_item, nitems;
    void *partials;
};

template <int DT, int ACC>
__global__ void __launch_bounds__(kBatchThreads, 1) tiled_bstream_kernel(const __grid_constant__ CUtensorMap tmap,
                                                                          const BatchParams p)
{
    // [image stages][barriers, item descriptors][matrix stages]
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *img_base = smem;
    unsigned char *hdr = smem + (size_t)p.img_stages * p.img_stage_bytes;
    uint64_t *img_full = reinterpret_cast<uint64_t *>(hdr);
    uint64_t *img_empty = img_full + kBatchMaxImgStages;
    uint64_t *mat_full = img_empty + kBatchMaxImgStages;
    uint64_t *mat_empty = mat_full + kBatchMaxMatStages;
    int4 *desc_s = reinterpret_cast<int4 *>(hdr + kStreamBarBytes);
    unsigned char *mat_base = hdr + p.hdr_bytes;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    int nmine = 0;
    while (stream_item_at(nmine) < p.nitems) ++nmine;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kBatchMaxImgStages; ++s) {
            mbar_init(img_full + s, 1);
            mbar_init(img_empty + s, kBatchCons);
        }
        for (int s = 0; s < kBatchMaxMatStages; ++s) {
            mbar_init(mat_full + s, 1);
            mbar_init(mat_empty + s, kBatchCons);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int k = threadIdx.x; k < nmine; k += kBatchThreads) {
        const int w = stream_item_at(k);
        int4 d = __ldg(p.blob_desc + w % p.ntiles);
        d.x = d.w ? d.x : 0;
        desc_s[k] = d;
    }
    asm volatile("griddepcontrol.launch_dependents;");       // stage 2 may be scheduled as SMs free up
    __syncthreads();

    Ring ir, mr;
    if (warp == 0) {
        // ===== producer: blob of the item, then the tiles of its frames ==================================================
        int nblob = 0, nimg = 0;
        for (int n = 0; n < nmine; ++n) {
            const int4 d = desc_s[n];
            if (d.w == 0) continue;
            const int chunk = stream_item_at(n) / p.ntiles;
            const int f0 = chunk * p.frames_per_item, f1 = min(p.nframes, f0 + p.frames_per_item);
            const int ty = d.z >> 16, tx = d.z & 0xffff;
            if (nblob >= p.mat_stages) mbar_wait(mat_empty + mr.stage, mr.parity ^ 1u);
            if (lane == 0) {
                mbar_arrive_expect_tx(mat_full + mr.stage, (uint32_t)d.y);
                bulk_g2s(mat_base + (size_t)mr.stage * p.mat_stage_bytes, p.blob + (size_t)d.x * 16, (uint32_t)d.y,
                         mat_full + mr.stage);
            }
            ++nblob;
            mr.next(p.mat_stages);
            for (int f = f0; f < f1; ++f) {
                if (nimg >= p.img_stages) mbar_wait(img_empty + ir.stage, ir.parity ^ 1u);
                if (lane == 0) {
                    unsigned char *tile = img_base + (size_t)ir.stage * p.img_stage_bytes;
                    mbar_arrive_expect_tx(img_full + ir.stage, (uint32_t)p.img_stage_bytes);
                    tma_box(tile, &tmap, tx * kTileW, ty * p.tile_h, f, img_full + ir.stage);
                    tma_box(tile + p.img_stage_bytes / 2, &tmap, tx * kTileW + 32, ty * p.tile_h, f, img_full + ir.stage);
                }
                ++nimg;
                ir.next(p.img_stages);
            }
        }
    } else {
        // ===== consumers: blocks dealt round-robin to the warps, continuing across frame pairs and items ==================
        const int cw = warp - 1;
        int firstb = cw;
        for (int n = 0; n < nmine; ++n) {
            const int4 d = desc_s[n];
            if (d.w == 0) continue;
            const int chunk = stream_item_at(n) / p.ntiles;
            const int f0 = chunk * p.frames_per_item, f1 = min(p.nframes, f0 + p.frames_per_item);
            mbar_wait(mat_full + mr.stage, mr.parity);
            const unsigned char *blob = mat_base + (size_t)mr.stage * p.mat_stage_bytes;
            const unsigned *bh = reinterpret_cast<const unsigned *>(blob) + 1;
            for (int f = f0; f < f1; f += 2) {
                const bool two = f + 1 < f1;
                const int sa = ir.stage;
                mbar_wait(img_full + sa, ir.parity);
                ir.next(p.img_stages);
                const int sb = ir.stage;
                if (two) {
                    mbar_wait(img_full + sb, ir.parity);
                    ir.next(p.img_stages);
                }
                if (firstb < d.w) {
                    const unsigned ta = smem_u32(img_base + (size_t)sa * p.img_stage_bytes);
                    const unsigned tb = smem_u32(img_base + (size_t)sb * p.img_stage_bytes);
                    char *pa = reinterpret_cast<char *>(p.partials) + (int64_t)f * p.nslot * 16;
                    char *pb = pa + (int64_t)p.nslot * 16;
                    for (int b = firstb; b < d.w; b += kBatchCons) {
                        const unsigned h = bh[b];
                        if (two && !stream_block2<DT, ACC>(ta, tb, blob, h, pa, pb, lane)) continue;
                        // one frame left, or a non-finite pixel somewhere: frame by frame
                        if (stream_block<DT, ACC, false>(ta, blob, h, pa, lane)) {
                            if constexpr (DT == AI_F32) stream_block_tracked<ACC, false>(ta, blob, h, pa, lane);
                        }
                        if (two && stream_block<DT, ACC, false>(tb, blob, h, pb, lane)) {
                            if constexpr (DT == AI_F32) stream_block_tracked<ACC, false>(tb, blob, h, pb, lane);
                        }
                    }
                    __syncwarp();
                }
                if (lane == 0) {
                    mbar_arrive(img_empty + sa);
                    if (two) mbar_arrive(img_empty + sb);
                }
                firstb -= d.w % kBatchCons;
                if (firstb < 0) firstb += kBatchCons;
            }
            if (lane == 0) mbar_arrive(mat_empty + mr.stage);
            mr.next(p.mat_stages);
        }
    }
}

template <int DT, int ACC>
int launch_stream(ai_ctx *ctx, const CUtensorMap &map, const StreamFirstDescs &first, const StreamParams &p, size_t smem,
                  int grid, cudaStream_t st)
{
    static int configured_device = -1;            // per instantiation: opt in to the large dynamic shared memory once
    if (configured_device != ctx->device) {
        AI_CUDA(ctx, cudaFuncSetAttribute(tiled_stream_kernel<DT, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          kPipeSmemBudget));
        configured_device = ctx->device;
    }
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kStreamThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ai_prof_begin(ctx, st);
    AI_CUDA(ctx, cudaLaunchKernelEx(&cfg, tiled_stream_kernel<DT, ACC>, map, first, p));
    ai_prof_end(ctx, st);
    return AI_OK;
}

template <int DT>
int launch_stream_dt(ai_ctx *ctx, const CUtensorMap &map, const StreamFirstDescs &first, const StreamParams &p,
                     size_t smem, int grid, cudaStream_t st)
{
    switch (ctx->accum) {
    case AI_ACC_F32_KAHAN: return launch_stream<DT, AI_ACC_F32_KAHAN>(ctx, map, first, p, smem, grid, st);
    case AI_ACC_F32_PLAIN: return launch_stream<DT, AI_ACC_F32_PLAIN>(ctx, map, first, p, smem, grid, st);
    default: return launch_stream<DT, AI_ACC_F64>(ctx, map, first, p, smem, grid, st);
    }
}

}  // namespace

#ifdef AI_PIPE_TRACE
extern "C" int ai_debug_set_stream_trace(void *dev_buffer, int div)
{
    cudaMemcpyToSymbol(g_strace_div, &div, sizeof(int));
    return (int)cudaMemcpyToSymbol(g_strace, &dev_buffer, sizeof(void *));
}
#endif

// shared-memory plan: [tile stages][barriers + descriptors][blob stages]; false if fewer than two stages fit
static bool stream_plan(const ai_ctx *ctx, int grid, StreamParams *p)
{
    const TiledLayout &tl = ctx->tl;
    p->img_stage_bytes = tl.tile_h * kTileW * 4;
    p->mat_stage_bytes = ai_align_up(tl.max_blob_bytes + 1024, 1024);     // slack: the look-ahead reads past a blob's end
    p->hdr_bytes = ai_align_up(kStreamBarBytes, 1024);
    int stages = (kPipeSmemBudget - p->hdr_bytes) / (p->img_stage_bytes + p->mat_stage_bytes);
    if (stages > kStreamMaxStages) stages = kStreamMaxStages;
    if (ctx->tune.stream_stages > 0 && stages > ctx->tune.stream_stages) stages = ctx->tune.stream_stages;
    while (stages * p->img_stage_bytes > 0xf000) --stages;    // tile buffers stay inside the first 64 KB (packed rebase)
    p->stages = stages;
    return stages >= 2;
}

int ai_stream_stages(const ai_ctx *ctx)
{
    const TiledLayout &tl = ctx->tl;
    if (tl.ntiles < 1 || !tl.blob) return 0;
    const int sms = ctx->sm_count > 0 ? ctx->sm_count : 148;
    const int grid = tl.ntiles < sms ? tl.ntiles : sms;
    StreamParams p{};
    return grid <= kStreamMaxGrid && stream_plan(ctx, grid, &p) ? p.stages : 0;
}

// Launches the single-frame fast path when it applies (*handled = true): one frame of 32-bit pixels, no correction
// arrays, rows on 16-byte boundaries, and at least two (tile + blob) stages fitting the shared memory of an SM.
// The kernel is the whole hot path of the frame: stage 1 and, behind a grid barrier, H5 (no second launch).
int ai_launch_stream_stage1(ai_ctx *ctx, const FrameArgs &a, int vec_ok, int track_all, cudaStream_t st, bool *handled)
{
    const TiledLayout &tl = ctx->tl;
    *handled = false;
    if (a.nframes != 1 || tl.ntiles < 1 || !tl.blob || !tl.h_first_desc || !ctx->grid_sync || ctx->no_tma || ctx->no_stream)
        return AI_OK;
    const bool plain = !a.dark && !a.flat && !a.solidangle && !a.polarization && !a.mask;
    const bool is32 = a.dtype == AI_F32 || a.dtype == AI_I32 || a.dtype == AI_U32;
    if (!plain || !is32 || !vec_ok || (reinterpret_cast<uintptr_t>(a.image) % 16) != 0) return AI_OK;
    const int sms = ctx->sm_count > 0 ? ctx->sm_count : 148;
    const int grid = tl.ntiles < sms ? tl.ntiles : sms;
    if (grid > kStreamMaxGrid) return AI_OK;

    StreamParams p{};
    if (!stream_plan(ctx, grid, &p)) return AI_OK;
    const int stages = p.stages;
    p.blob_desc = tl.blob_desc;
    p.blob = tl.blob;
    p.tile_h = tl.tile_h;
    p.ntiles = tl.ntiles;
    p.nslot = tl.nslot;
    p.partials = ctx->partials;
    p.dyn_base = (p.stages < kStreamFirst ? p.stages : kStreamFirst) * grid;
    p.track_all = track_all;
    static unsigned launches = 0;                  // development trace only: which of 8 trace buffers the launch writes
    p.launch_index = launches++ & 7;
    p.grid_sync = ctx->grid_sync;
    p.bin_slot_ptr = tl.bin_slot_ptr;
    p.range = ctx->d_range;
    p.npt = ctx->npt;
    p.empty = ctx->empty_value;
    p.radial = a.radial;
    p.intensity = a.intensity;
    p.sum_signal = a.sum_signal;
    p.count = a.count;
    const size_t smem = (size_t)stages * (p.img_stage_bytes + p.mat_stage_bytes) + p.hdr_bytes;

    // descriptors of the first tiles of every block (host copy kept by the builder), assembled once per context
    if (!ctx->stream_first || ctx->stream_first_grid != grid) {
        free(ctx->stream_first);
        ctx->stream_first = calloc(1, sizeof(StreamFirstDescs));
        if (!ctx->stream_first) return ai_fail(ctx, AI_ENOMEM, "first-tile descriptors");
        StreamFirstDescs *fd = static_cast<StreamFirstDescs *>(ctx->stream_first);
        for (int n = 0; n < kStreamFirst; ++n)
            for (int b = 0; b < grid; ++b) {
                const int w = n * grid + ((n & 1) ? grid - 1 - b : b);
                fd->d[n][b] = w < tl.ntiles ? tl.h_first_desc[w] : make_int4(0, 0, 0, 0);
            }
        ctx->stream_first_grid = grid;
    }
    const StreamFirstDescs &first = *static_cast<const StreamFirstDescs *>(ctx->stream_first);
    CUtensorMap map{};
    int rc = ai_make_frame_map(ctx, a, tl.tile_h, &map);
    if (rc != AI_OK) return rc;
    rc = AI_EINVAL;
    switch (a.dtype) {
    case AI_F32: rc = launch_stream_dt<AI_F32>(ctx, map, first, p, smem, grid, st); break;
    case AI_I32: rc = launch_stream_dt<AI_I32>(ctx, map, first, p, smem, grid, st); break;
    case AI_U32: rc = launch_stream_dt<AI_U32>(ctx, map, first, p, smem, grid, st); break;
    default: break;
    }
    if (rc == AI_OK) *handled = true;
    return rc;
}

namespace {

template <int DT, int ACC>
int launch_bstream(ai_ctx *ctx, const CUtensorMap &map, const BatchParams &p, size_t smem, int grid, cudaStream_t st)
{
    static int configured_device = -1;
    if (configured_device != ctx->device) {
        AI_CUDA(ctx, cudaFuncSetAttribute(tiled_bstream_kernel<DT, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          kPipeSmemBudget));
        configured_device = ctx->device;
    }
    ai_prof_begin(ctx, st);
    tiled_bstream_kernel<DT, ACC><<<grid, kBatchThreads, smem, st>>>(map, p);
    ai_prof_end(ctx, st);
    AI_CUDA(ctx, cudaGetLastError());
    return AI_OK;
}

template <int DT>
int launch_bstream_dt(ai_ctx *ctx, const CUtensorMap &map, const BatchParams &p, size_t smem, int grid, cudaStream_t st)
{
    switch (ctx->accum) {
    case AI_ACC_F32_KAHAN: return launch_bstream<DT, AI_ACC_F32_KAHAN>(ctx, map, p, smem, grid, st);
    case AI_ACC_F32_PLAIN: return launch_bstream<DT, AI_ACC_F32_PLAIN>(ctx, map, p, smem, grid, st);
    default: return launch_bstream<DT, AI_ACC_F64>(ctx, map, p, smem, grid, st);
    }
}

}  // namespace

// Stage 1 of a batch of plain 32-bit frames (*handled = true when it applies); the caller launches stage 2.
int ai_launch_bstream_stage1(ai_ctx *ctx, const FrameArgs &a, int vec_ok, cudaStream_t st, bool *handled)
{
    const TiledLayout &tl = ctx->tl;
    *handled = false;
    if (a.nframes < 2 || tl.ntiles < 1 || !tl.blob || ctx->no_tma || ctx->no_stream) return AI_OK;
    const bool plain = !a.dark && !a.flat && !a.solidangle && !a.polarization && !a.mask;
    const bool is32 = a.dtype == AI_F32 || a.dtype == AI_I32 || a.dtype == AI_U32;
    if (!plain || !is32 || !vec_ok || (reinterpret_cast<uintptr_t>(a.image) % 16) != 0) return AI_OK;
    const int sms = ctx->sm_count > 0 ? ctx->sm_count : 148;

    BatchParams p{};
    // items: every tile once per chunk of frames; enough chunks that each block gets several items, even chunks
    int nchunks = (8 * sms + tl.ntiles - 1) / tl.ntiles;
    if (nchunks > a.nframes / 2) nchunks = a.nframes / 2;
    if (nchunks < 1) nchunks = 1;
    p.frames_per_item = (a.nframes + nchunks - 1) / nchunks;
    p.frames_per_item += p.frames_per_item & 1;
    nchunks = (a.nframes + p.frames_per_item - 1) / p.frames_per_item;
    const int64_t nitems = (int64_t)tl.ntiles * nchunks;
    if (nitems > 0x3fffffffLL) return AI_OK;
    p.nitems = (int)nitems;
    const int grid = p.nitems < sms ? p.nitems : sms;
    const int items_max = (p.nitems + grid - 1) / grid;
    p.img_stage_bytes = tl.tile_h * kTileW * 4;
    p.mat_stage_bytes = ai_align_up(tl.max_blob_bytes + 1024, 1024);
    p.hdr_bytes = ai_align_up(kStreamBarBytes + 16 * items_max, 1024);
    const int room = kPipeSmemBudget - p.hdr_bytes;
    p.mat_stages = (room - 2 * p.mat_stage_bytes) / p.img_stage_bytes >= 4 ? 2 : 1;
    p.img_stages = (room - p.mat_stages * p.mat_stage_bytes) / p.img_stage_bytes;
    if (p.img_stages > kBatchMaxImgStages) p.img_stages = kBatchMaxImgStages;
    if (p.img_stages < 2) return AI_OK;
    p.blob_desc = tl.blob_desc;
    p.blob = tl.blob;
    p.tile_h = tl.tile_h;
    p.ntiles = tl.ntiles;
    p.nslot = tl.nslot;
    p.nframes = a.nframes;
    p.partials = ctx->partials;
    const size_t smem = (size_t)p.img_stages * p.img_stage_bytes + p.hdr_bytes + (size_t)p.mat_stages * p.mat_stage_bytes;
    CUtensorMap map{};
    int rc = ai_make_frame_map(ctx, a, tl.tile_h, &map);
    if (rc != AI_OK) return rc;
    rc = AI_EINVAL;
    switch (a.dtype) {
    case AI_F32: rc = launch_bstream_dt<AI_F32>(ctx, map, p, smem, grid, st); break;
    case AI_I32: rc = launch_bstream_dt<AI_I32>(ctx, map, p, smem, grid, st); break;
    case AI_U32: rc = launch_bstream_dt<AI_U32>(ctx, map, p, smem, grid, st); break;
    default: break;
    }
    if (rc == AI_OK) *handled = true;
    return rc;
}
