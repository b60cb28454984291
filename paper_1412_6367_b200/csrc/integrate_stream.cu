// The TMA-streamed kernels of the TILED layout -- the CSR SpMV of PAPER.md:174-188 on B200.
//
// tiled_stream_kernel: H1 + H4 of ONE frame of 32-bit pixels (the configuration the headline metric is quoted on;
// corrected frames come here through the pre-pass of integrate_prep.cu); H5 is tiled_stage2_kernel (integrate_tiled.cu).
//   - one persistent block per SM, 1 producer warp + kStreamCons consumer warps; float frames are gathered straight
//     from the TMA tile, integer frames are converted at gather time ("casted from integer to float");
//   - one ring whose stage holds a tile of the frame AND that tile's blob of the matrix, one full / empty mbarrier pair
//     per stage; the descriptor of the tile in a stage sits next to the barriers;
//   - tiles longest first: the first kStreamFirst of every block are dealt statically and travel in the kernel
//     parameters (their copies leave before any global load has returned), the rest are drawn from a ticket counter;
//   - pixel positions of two entries are rebased with one packed 16-bit add: the tile buffers live in the first 64 KB of
//     the shared window, so a position's low half-word is its whole shared address;
//   - one partial record per run of the sliced layout, in the set of partials of this launch's parity;
//   - programmatic dependent launch: along a stream of calls the next call's kernel streams while this one drains and
//     the small finish kernel in between adds up this one's partials (see the kernel).
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
constexpr int kStreamBarBytes = 512;                 // full[8] + empty[8], per-stage descriptors
constexpr int kStreamDescOffset = 256;
constexpr int kBatchBarBytes = 512;                  // tiled_bstream_kernel: barriers, then the item descriptors

struct StreamFirstDescs {
    int4 d[kStreamFirst][kStreamMaxGrid];
};

struct StreamParams {
    const int4 *blob_desc;       // longest first: {blob offset / 16, blob bytes, tile row << 16 | column, blocks}
    const unsigned char *blob;
    const unsigned char *blob_orig;   // held corrections: `blob` is the held copy, this one the matrix's own
    int tile_h, ntiles, nslot;
    int stages, mat_stage_bytes, img_stage_bytes, hdr_bytes;
    int tile_bytes;              // bytes of a frame tile (= img_stage_bytes without held corrections)
    int dk;                      // held corrections: the dark tiles of all stages follow the frame tiles of all stages; a
                                 // stage's dark tile lies dk = stages x tile_bytes behind its frame tile (a multiple of 1024:
                                 // same 128-byte swizzle phase); img_stage_bytes = 2 tile_bytes
    int dyn_base;                // rank of the first tile handed out by ticket (the ones before are dealt statically)
    int launch_index;            // launches of this context so far, modulo 8 (not read by the kernel; kept so that the
                                 // parameter block, and with it ptxas's allocation, stays what was measured)
    int track_all;               // float frames: every block skips non-finite pixels and accumulates count
    void *partials;
    unsigned long long *tickets;       // tile tickets of this launch (zero at its start)
    unsigned long long *tickets_reset; // the counter the context's next launch uses: zeroed by this one
    int full_grid;                     // one block on every SM: a block of this launch runs where the previous
                                       // launch's block has left, so the launch before that one is complete
    int overlap;                       // stream before the grid dependency is resolved (see the kernel)
    const unsigned long long *chain_done;   // overlap: the finish kernel that read this launch's set of partials last has
    unsigned long long chain_target;        // ended when *chain_done >= chain_target
};


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

// held corrections: the pixel minus the held dark current, whose tile lies `dk` bytes behind the frame's
template <int DT>
__device__ __forceinline__ float4 stream_gather4_held(const uint2 &x, unsigned base, unsigned dk)
{
    const unsigned p0 = x.x + base, p1 = x.y + base;
    const unsigned a0 = p0 & 0xffffu, a1 = p0 >> 16, a2 = p1 & 0xffffu, a3 = p1 >> 16;
    float4 v;
    if constexpr (DT == AI_F32) {
        v = make_float4(lds_f32(a0), lds_f32(a1), lds_f32(a2), lds_f32(a3));
    } else if constexpr (DT == AI_I32) {
        v = make_float4((float)lds_s32(a0), (float)lds_s32(a1), (float)lds_s32(a2), (float)lds_s32(a3));
    } else {
        v = make_float4((float)(unsigned)lds_s32(a0), (float)(unsigned)lds_s32(a1), (float)(unsigned)lds_s32(a2),
                        (float)(unsigned)lds_s32(a3));
    }
    return make_float4(__fsub_rn(v.x, lds_f32(a0 + dk)), __fsub_rn(v.y, lds_f32(a1 + dk)), __fsub_rn(v.z, lds_f32(a2 + dk)),
                       __fsub_rn(v.w, lds_f32(a3 + dk)));
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
template <int DT, int ACC, bool PACKED = true, bool HELD = false>
__device__ __noinline__ bool stream_block(unsigned rebase, const unsigned char *blob, unsigned h, void *part_f, int lane,
                                          unsigned dk = 0)
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
        float4 v0, v1;
        if constexpr (HELD) {
            v0 = stream_gather4_held<DT>(x0, rebase, dk);
            v1 = stream_gather4_held<DT>(x1, rebase, dk);
        } else {
            v0 = stream_gather4<DT, PACKED>(x0, rebase);
            v1 = stream_gather4<DT, PACKED>(x1, rebase);
        }
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

// Held corrections (hold.cu), a block that met a non-finite I - dark (a non-finite pixel of a float frame): the staged
// coefficients carry 1 / den, so the weight a valid pixel adds to count is read from the matrix's own blob (`orig`, global
// memory, same offsets).  A pixel that is invalid for every frame has a zero staged coefficient and adds nothing: its
// weight is not in the run sums of the held blob either.
template <int DT>
__device__ __noinline__ void stream_block_tracked_held(unsigned rebase, const unsigned char *blob, const unsigned char *orig,
                                                       unsigned h, void *part_f, int lane, unsigned dk)
{
    const int nsteps = h & 15, rounds = (h >> 4) & 7;
    const unsigned char *blk = blob + (size_t)(h >> 8) * 16;
    const float4 *cp = reinterpret_cast<const float4 *>(blk) + lane;
    const float4 *op = reinterpret_cast<const float4 *>(orig + (size_t)(h >> 8) * 16) + lane;
    const uint2 *xp = reinterpret_cast<const uint2 *>(blk + nsteps * 512) + lane;
    const int2 m = reinterpret_cast<const int2 *>(blk + nsteps * kBlkStepBytes)[lane];
    AccumQ<AI_ACC_F32_KAHAN> S2, C2;
#pragma unroll 1
    for (int j = 0; j < nsteps; ++j) {
        const float4 c = cp[j * 32], o = __ldg(op + j * 32);
        const float4 v = stream_gather4_held<DT>(xp[j * 32], rebase, dk);
        const bool k0 = finite_f(v.x), k1 = finite_f(v.y), k2 = finite_f(v.z), k3 = finite_f(v.w);
        S2.a.add(c.x, k0 ? v.x : 0.0f);
        S2.b.add(c.y, k1 ? v.y : 0.0f);
        S2.c.add(c.z, k2 ? v.z : 0.0f);
        S2.d.add(c.w, k3 ? v.w : 0.0f);
        C2.a.add1(k0 && c.x != 0.0f ? o.x : 0.0f);
        C2.b.add1(k1 && c.y != 0.0f ? o.y : 0.0f);
        C2.c.add1(k2 && c.z != 0.0f ? o.z : 0.0f);
        C2.d.add1(k3 && c.w != 0.0f ? o.w : 0.0f);
    }
    stream_finish_d<true>(kahan_total_d(S2), kahan_total_d(C2), m, rounds, part_f);
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

template <int DT, int ACC, bool HELD = false>
__global__ void __launch_bounds__(kStreamThreads, 1) tiled_stream_kernel(const __grid_constant__ CUtensorMap tmap,
                                                                         const __grid_constant__ CUtensorMap dmap,
                                                                         const __grid_constant__ StreamFirstDescs first,
                                                                         const StreamParams p)
{
    // [frame tile stages (, HELD: dark tile stages)][barriers, per-stage tile descriptors][matrix stages]
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *img_base = smem;
    unsigned char *hdr = smem + (size_t)p.stages * p.img_stage_bytes;
    uint64_t *full = reinterpret_cast<uint64_t *>(hdr);              // tile + blob landed (complete_tx)
    uint64_t *empty = full + kStreamMaxStages;                        // every consumer warp is done with the stage
    int4 *stage_desc = reinterpret_cast<int4 *>(hdr + kStreamDescOffset);   // descriptor of the tile in each stage
    unsigned char *mat_base = hdr + p.hdr_bytes;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    // Tiles, longest first: the first npre of every block are dealt statically (snake order; their descriptors came
    // with the launch), the rest are handed out by a ticket counter to whichever block has a free stage -- the blocks
    // do not finish their static shares at the same time (the memory system serves them unevenly).
    int npre = 0;
    while (npre < min(kStreamFirst, p.stages) && stream_item_at(npre) < p.ntiles) ++npre;

    auto issue_blob = [&](int stage, const int4 &d) {
        stage_desc[stage] = d;
        mbar_arrive_expect_tx(full + stage, (uint32_t)((HELD ? 2 : 1) * p.tile_bytes + d.y));
        bulk_g2s(mat_base + (size_t)stage * p.mat_stage_bytes, p.blob + (size_t)d.x * 16, (uint32_t)d.y, full + stage);
    };
    auto issue_tile = [&](int stage, const int4 &d) {
        unsigned char *tile = img_base + (size_t)stage * p.tile_bytes;
        const int ty = d.z >> 16, tx = d.z & 0xffff;
        tma_box(tile, &tmap, tx * kTileW, ty * p.tile_h, 0, full + stage);
        tma_box(tile + p.tile_bytes / 2, &tmap, tx * kTileW + 32, ty * p.tile_h, 0, full + stage);
        if constexpr (HELD) {
            // the held dark current of the same pixels, behind the frame tile
            tma_box(tile + p.dk, &dmap, tx * kTileW, ty * p.tile_h, 0, full + stage);
            tma_box(tile + p.dk + p.tile_bytes / 2, &dmap, tx * kTileW + 32, ty * p.tile_h, 0, full + stage);
        }
    };

    // Launch chain (programmatic dependent launch).  A call is two launches, this kernel (S) and the finish kernel (F,
    // tiled_stage2_kernel: it waits for S, adds the partials of every bin up and writes the caller's outputs); both
    // let their dependents start at once, so along a stream of calls S_k, F_k, S_k+1, F_k+1 ... the blocks of S_k+1 take
    // the SMs as the blocks of S_k leave them (one S block per SM: registers), while F_k, a few small blocks that fit
    // beside them, waits for the last block of S_k.
    //   p.overlap (the grid fills the GPU and the frame is not written by the kernel right before this one): S runs
    //     WITHOUT waiting for its predecessors.  It reads the matrix and the frame and writes only this launch's set
    //     of partial sums and tickets (alternating sets).  Before it leaves, every block waits for the grid dependency
    //     (free by then): S_k completes after F_k-1, so a block of S_k+1 -- resident only where a block of S_k has
    //     left -- finds the set of partials it shares with S_k-1 read out and S_k-1's ticket counter idle.
    //   otherwise nothing but static data (barriers, tensor map, first blobs) is touched before griddepcontrol.wait.
    if (threadIdx.x == 0) {
        // the packed rebase needs every tile buffer inside the first 64 KB of the shared window
        if (smem_u32(img_base) + (unsigned)(p.stages * p.tile_bytes) > 0x10000u) __trap();
        for (int s = 0; s < kStreamMaxStages; ++s) {
            mbar_init(full + s, 1);
            mbar_init(empty + s, kStreamCons);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap) : "memory");
        if constexpr (HELD) asm volatile("prefetch.tensormap [%0];" ::"l"(&dmap) : "memory");
        if (p.full_grid && blockIdx.x == 0) {
            // tickets of the context's next launch (last used by the launch before the previous one, complete: see
            // above): zero before any block of that launch can exist, i.e. before this block lets dependents start
            *p.tickets_reset = 0ULL;
            fence_acq_rel_gpu();
        }
        // first blobs (and tiles), from descriptors that came with the launch: in flight before any global load returns
        int stage = 0;
        for (int n = 0; n < npre; ++n) {
            const int4 d = first.d[n][blockIdx.x];
            if (d.w == 0) continue;
            issue_blob(stage, d);
            if (p.overlap) issue_tile(stage, d);
            ++stage;
        }
    }
    // overlap: nothing of this block writes partial sums before the finish kernel of the call before the previous one
    // has read the set they share.  With the GPU to itself the chain guarantees it (see below); checked because another
    // tenant may have let this block in out of turn.  One thread of a consumer warp, while thread 0 sets the block up.
    if (threadIdx.x == 32 && p.overlap) wait_count_at_least(p.chain_done, p.chain_target);
    // the descriptors of the ticketed tiles (each block its share of the array), pulled into L2 now
    for (int k = p.dyn_base + (blockIdx.x * kStreamThreads + threadIdx.x) * 8; k < p.ntiles; k += gridDim.x * kStreamThreads * 8)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(p.blob_desc + k));
    __syncthreads();
    // the next kernel of the stream may be scheduled as SMs free up
    asm volatile("griddepcontrol.launch_dependents;");
    if (!p.overlap) {
        asm volatile("griddepcontrol.wait;" ::: "memory");
        if (threadIdx.x == 0) {
            int stage = 0;
            for (int n = 0; n < npre; ++n) {
                const int4 d = first.d[n][blockIdx.x];
                if (d.w == 0) continue;
                issue_tile(stage++, d);
            }
            if (!p.full_grid && blockIdx.x == 0) *p.tickets_reset = 0ULL;     // everything before this launch is complete
        }
    }

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
            const unsigned long long t0 = atomicAdd(p.tickets, 1ULL);
            t_next = atomicAdd(p.tickets, 1ULL);
            d_next = fetch(t0);
        }
        while (true) {
            const int4 d = d_next;
            if (lane == 0 && nticket) {
                d_next = fetch(t_next);
                t_next = atomicAdd(p.tickets, 1ULL);
            }
            const int nblk = __shfl_sync(AI_FULL_MASK, d.w, 0);
            if (nblk < 0) break;
            if (nblk == 0) continue;                      // tile without entries: never published
            if (issued >= p.stages) mbar_wait(empty + r.stage, r.parity ^ 1u);
            if (lane == 0) {
                issue_blob(r.stage, d);
                issue_tile(r.stage, d);
            }
            ++issued;
            r.next(p.stages);
        }
        // no tile left: a descriptor with a negative block count ends the consumers' loop
        if (issued >= p.stages) mbar_wait(empty + r.stage, r.parity ^ 1u);
        if (lane == 0) {
            stage_desc[r.stage] = make_int4(0, 0, 0, -1);
            mbar_arrive(full + r.stage);
        }
        // overlap: the block (hence the grid) completes after everything before it in the stream
        if (p.overlap) asm volatile("griddepcontrol.wait;" ::: "memory");
    } else {
        // ===== consumers: a tile's blocks are dealt round-robin to the warps, continuing across tiles ===================
        const int cw = warp - 1;
        int firstb = cw;
        for (int n = 0;; ++n) {
            // every warp waits on and arrives at every stage, also when it holds no block of the tile: no warp is
            // ever a whole phase away from a barrier
            mbar_wait(full + r.stage, r.parity);
            const int4 d = stage_desc[r.stage];
            if (d.w < 0) break;
            if (firstb < d.w) {
                const unsigned char *blob = mat_base + (size_t)r.stage * p.mat_stage_bytes;
                const unsigned *bh = reinterpret_cast<const unsigned *>(blob) + 1;
                const unsigned rebase = (smem_u32(img_base + (size_t)r.stage * p.tile_bytes) & 0xffffu) * 0x10001u;
                for (int b = firstb; b < d.w; b += kStreamCons) {
                    const unsigned h = bh[b];
                    if constexpr (HELD) {
                        if (stream_block<DT, ACC, true, true>(rebase, blob, h, p.partials, lane, (unsigned)p.dk))
                            stream_block_tracked_held<DT>(rebase, blob, p.blob_orig + (size_t)d.x * 16, h, p.partials, lane,
                                                          (unsigned)p.dk);
                    } else if constexpr (DT == AI_F32) {
                        // track_all: the frame comes from the correction pre-pass and is expected to hold NaN marks
                        if (p.track_all || stream_block<DT, ACC>(rebase, blob, h, p.partials, lane))
                            stream_block_tracked<ACC>(rebase, blob, h, p.partials, lane);
                    } else {
                        stream_block<DT, ACC>(rebase, blob, h, p.partials, lane);
                    }
                }
                __syncwarp();
            }
            if (lane == 0) mbar_arrive(empty + r.stage);
            firstb -= d.w % kStreamCons;
            if (firstb < 0) firstb += kStreamCons;
            r.next(p.stages);
        }
    }
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
    int single_units;            // a consumer warp's work unit is (block, one frame) instead of (block, two frames)
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
    int4 *desc_s = reinterpret_cast<int4 *>(hdr + kBatchBarBytes);
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
                // work units of the pass, dealt round-robin to the warps and continuing across passes: (block, both
                // frames) -- coefficients and positions serve two frames -- or, when a tile has fewer blocks than half
                // the warps (p.single_units, an experiment switch), (block, one frame): twice as many units
                const int nunits = p.single_units && two ? 2 * d.w : d.w;
                if (firstb < nunits) {
                    const unsigned ta = smem_u32(img_base + (size_t)sa * p.img_stage_bytes);
                    const unsigned tb = smem_u32(img_base + (size_t)sb * p.img_stage_bytes);
                    char *pa = reinterpret_cast<char *>(p.partials) + (int64_t)f * p.nslot * 16;
                    char *pb = pa + (int64_t)p.nslot * 16;
                    for (int u = firstb; u < nunits; u += kBatchCons) {
                        if (p.single_units && two) {
                            const unsigned h = bh[u >> 1];
                            const unsigned t = (u & 1) ? tb : ta;
                            char *pp = (u & 1) ? pb : pa;
                            if (stream_block<DT, ACC, false>(t, blob, h, pp, lane)) {
                                if constexpr (DT == AI_F32) stream_block_tracked<ACC, false>(t, blob, h, pp, lane);
                            }
                            continue;
                        }
                        const unsigned h = bh[u];
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
                firstb -= nunits % kBatchCons;
                if (firstb < 0) firstb += kBatchCons;
            }
            if (lane == 0) mbar_arrive(mat_empty + mr.stage);
            mr.next(p.mat_stages);
        }
    }
}

template <int DT, int ACC, bool HELD = false>
int launch_stream(ai_ctx *ctx, const CUtensorMap &map, const CUtensorMap &dmap, const StreamFirstDescs &first, StreamParams p,
                  size_t smem, int grid, cudaStream_t st)
{
    const uint64_t bit = 1ULL << (HELD ? 45 + (DT == AI_F32 ? 0 : DT == AI_I32 ? 1 : 2) : DT * 3 + ACC);      // per context and instantiation: opt in to the large
    if (!(ctx->smem_opt_in & bit)) {                      // dynamic shared memory once
        AI_CUDA(ctx, cudaFuncSetAttribute(tiled_stream_kernel<DT, ACC, HELD>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          kPipeSmemBudget));
        // the launch chain (see the kernel) relies on ONE block of this kernel per SM
        int per_sm = 0;
        AI_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, tiled_stream_kernel<DT, ACC, HELD>, kStreamThreads, smem));
        if (per_sm != 1) ctx->stream_shared_sm |= bit;
        ctx->smem_opt_in |= bit;
    }
    if (ctx->stream_shared_sm & bit) p.full_grid = p.overlap = 0;
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
    AI_CUDA(ctx, cudaLaunchKernelEx(&cfg, tiled_stream_kernel<DT, ACC, HELD>, map, dmap, first, p));
    ai_prof_end(ctx, st);
    return AI_OK;
}

template <int DT>
int launch_stream_dt(ai_ctx *ctx, const CUtensorMap &map, const CUtensorMap *dmap, const StreamFirstDescs &first,
                     const StreamParams &p, size_t smem, int grid, cudaStream_t st)
{
    if (dmap) return launch_stream<DT, AI_ACC_F32_KAHAN, true>(ctx, map, *dmap, first, p, smem, grid, st);
    switch (ctx->accum) {
    case AI_ACC_F32_KAHAN: return launch_stream<DT, AI_ACC_F32_KAHAN>(ctx, map, map, first, p, smem, grid, st);
    case AI_ACC_F32_PLAIN: return launch_stream<DT, AI_ACC_F32_PLAIN>(ctx, map, map, first, p, smem, grid, st);
    default: return launch_stream<DT, AI_ACC_F64>(ctx, map, map, first, p, smem, grid, st);
    }
}

}  // namespace


// shared-memory plan: [tile stages][barriers + descriptors][blob stages]; false if fewer than two stages fit
static bool stream_plan(const ai_ctx *ctx, int grid, StreamParams *p, bool held = false)
{
    const TiledLayout &tl = ctx->tl;
    p->tile_bytes = tl.tile_h * kTileW * 4;
    p->img_stage_bytes = held ? 2 * p->tile_bytes : p->tile_bytes;
    p->mat_stage_bytes = ai_align_up(tl.max_blob_bytes + 1024, 1024);     // slack: the look-ahead reads past a blob's end
    p->hdr_bytes = ai_align_up(kStreamBarBytes, 1024);
    // (4 KB of the SM's shared memory stay free: the finish kernel's blocks must fit beside a block of this kernel or the
    // launch chain stalls -- measured with a 226 KB variant: 13.6 -> 15.3 us per step on the headline)
    int stages = (kPipeSmemBudget - 4096 - p->hdr_bytes) / (p->img_stage_bytes + p->mat_stage_bytes);
    if (stages > kStreamMaxStages) stages = kStreamMaxStages;
    if (ctx->tune.stream_stages > 0 && stages > ctx->tune.stream_stages) stages = ctx->tune.stream_stages;
    while (stages * p->tile_bytes > 0xf000) --stages;    // frame tile buffers stay inside the first 64 KB (packed rebase)
    p->stages = stages;
    p->dk = held ? stages * p->tile_bytes : 0;
    if (held && p->tile_bytes % 1024 != 0) return false;
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

int ai_stream_full_grid(const ai_ctx *ctx)
{
    const int sms = ctx->sm_count > 0 ? ctx->sm_count : 148;
    return ai_stream_stages(ctx) >= 2 && ctx->tl.ntiles >= sms && !ctx->stream_shared_sm;
}

// Launches the single-frame fast path when it applies (*handled = true): one frame of 32-bit pixels, no correction
// arrays, rows on 16-byte boundaries, and at least two (tile + blob) stages fitting the shared memory of an SM.
// Stage 1 of the frame (H1 + H4); the caller launches stage 2 (H5) on *partials_used.
// image_dep: the frame is written by the kernel launched right before this one (the correction pre-pass).
int ai_launch_stream_stage1(ai_ctx *ctx, const FrameArgs &a, int vec_ok, int track_all, int image_dep, cudaStream_t st,
                            bool *handled, const void **partials_used)
{
    const TiledLayout &tl = ctx->tl;
    *handled = false;
    // held corrections (hold.cu): the held copy of the blobs, the dark tile behind every frame tile
    const bool held = a.held;
    if (held && (!ctx->held.on || !ctx->held.tl_ready || ctx->accum != AI_ACC_F32_KAHAN || ctx->width % 4 != 0)) return AI_OK;
    if (a.nframes != 1 || tl.ntiles < 1 || !tl.blob || !tl.h_first_desc || !ctx->grid_sync || !ctx->stream_partials ||
        ctx->no_tma || ctx->no_stream)
        return AI_OK;
    const bool plain = held || (!a.dark && !a.flat && !a.solidangle && !a.polarization && !a.mask);
    const bool is32 = a.dtype == AI_F32 || a.dtype == AI_I32 || a.dtype == AI_U32;
    if (!plain || !is32 || !vec_ok || (reinterpret_cast<uintptr_t>(a.image) % 16) != 0) return AI_OK;
    const int sms = ctx->sm_count > 0 ? ctx->sm_count : 148;
    const int grid = tl.ntiles < sms ? tl.ntiles : sms;
    if (grid > kStreamMaxGrid) return AI_OK;

    StreamParams p{};
    if (!stream_plan(ctx, grid, &p, held)) return AI_OK;
    const int stages = p.stages;
    p.blob_desc = tl.blob_desc;
    p.blob = held ? ctx->held.tl_blob : tl.blob;
    p.blob_orig = tl.blob;
    p.tile_h = tl.tile_h;
    p.ntiles = tl.ntiles;
    p.nslot = tl.nslot;
    // alternating sets of partial sums, three ticket counters in rotation: see the kernel
    const unsigned seq = ctx->stream_launches;
    p.partials = static_cast<char *>(ctx->stream_partials) + (size_t)(seq & 1) * (size_t)(tl.nslot > 0 ? tl.nslot : 1) * 16;
    p.dyn_base = (p.stages < kStreamFirst ? p.stages : kStreamFirst) * grid;
    p.track_all = track_all;
    p.launch_index = (int)(ctx->stream_launches & 7);
    p.tickets = ctx->grid_sync + seq % 3;
    p.tickets_reset = ctx->grid_sync + (seq + 1) % 3;
    p.full_grid = grid == sms;
    p.overlap = p.full_grid && !image_dep && !ctx->tune.no_overlap;
    p.chain_done = ctx->chain_done;
    p.chain_target = ctx->tune.no_chain_guard ? 0ULL : ctx->fin_cum_prev;

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
    CUtensorMap map{}, dmap{};
    int rc = ai_make_frame_map(ctx, a, tl.tile_h, &map);
    if (rc != AI_OK) return rc;
    if (held) {
        FrameArgs dk{};
        dk.image = ctx->held.dark;
        dk.dtype = AI_F32;
        dk.nframes = 1;
        dk.frame_stride = (int64_t)ctx->height * ctx->width;
        rc = ai_make_frame_map(ctx, dk, tl.tile_h, &dmap);
        if (rc != AI_OK) return rc;
    }
    const CUtensorMap *dm = held ? &dmap : nullptr;
    rc = AI_EINVAL;
    switch (a.dtype) {
    case AI_F32: rc = launch_stream_dt<AI_F32>(ctx, map, dm, first, p, smem, grid, st); break;
    case AI_I32: rc = launch_stream_dt<AI_I32>(ctx, map, dm, first, p, smem, grid, st); break;
    case AI_U32: rc = launch_stream_dt<AI_U32>(ctx, map, dm, first, p, smem, grid, st); break;
    default: break;
    }
    if (rc == AI_OK) {
        *handled = true;
        *partials_used = p.partials;
        ++ctx->stream_launches;
    }
    return rc;
}

namespace {

template <int DT, int ACC>
int launch_bstream(ai_ctx *ctx, const CUtensorMap &map, const BatchParams &p, size_t smem, int grid, cudaStream_t st)
{
    const uint64_t bit = 1ULL << (15 + DT * 3 + ACC);
    if (!(ctx->smem_opt_in & bit)) {
        AI_CUDA(ctx, cudaFuncSetAttribute(tiled_bstream_kernel<DT, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          kPipeSmemBudget));
        ctx->smem_opt_in |= bit;
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
    p.hdr_bytes = ai_align_up(kBatchBarBytes + 16 * items_max, 1024);
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
    p.single_units = ctx->tune.batch_units == 1;      // measured slower on cfg2 x 64 and cfg4 (0.375 / 2.18 ms against 0.325 / 1.82 ms)
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
