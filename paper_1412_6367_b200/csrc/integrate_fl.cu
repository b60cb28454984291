// Batches of plain 32-bit frames on the frame-lane layout (H6 of SURVEY.md section 8(a): "a batched multi-frame variant
// that amortises the matrix read across frames"; PAPER.md:11 detectors streaming thousands of frames per second;
// DESIGN.md section 5.4).
//
// fl_batch_kernel: lane = two frames.  A work item is (chunk of tiles, group of 64 frames); one persistent block per SM.
//   - kFlLoad loader warps bring a tile (32 x 8 pixels) of the group's 64 frames in with 128-bit loads (the lines were
//     pulled into L2 three tiles earlier by one tensor-map prefetch per tile), cast them (H1) and store the two frames of
//     lane l interleaved pixel by pixel, lane l shifted by 2 l words (lane pitch = tile bytes + 8): the 32 lanes of a
//     gather -- same pixel, 64 frames -- fall into 32 different bank pairs.  The tile's blob of the matrix arrives by one
//     bulk copy.  One ring of (tile + blob) stages, one full / empty mbarrier pair per stage.
//   - kFlCons consumer warps: every (tile, bin) segment belongs to the warp that owns the bin inside the chunk.  An
//     entry pair {c0, c1, pixel 0, pixel 1} is one broadcast 128-bit shared load for the whole warp; each lane gathers
//     its two frames' pixel with one 64-bit load and adds the two products with two Kahan recurrences
//     carried in packed fp32x2 arithmetic (FFMA2 / FADD2, the coefficient a scalar operand).  The running (sum,
//     compensation) of every (bin, frame) of the chunk lives in shared memory, touched by its owner warp only: fixed
//     order of every sum, no atomics, bit-reproducible.
//   - at the end of an item the owner warps write one (sum, compensation) pair per (chunk, bin, frame).
// fl_finish_kernel (H5): adds a bin's partials over the chunks in fp64 and writes the three outputs.
// Float frames: the loaders flag a tile that holds a non-finite pixel; its segments then take the variant that skips
// such pixels and adds their weight -- in 2^-40 fixed point, so that the atomic sums do not depend on their order -- to
// a (bin, frame) array which H5 subtracts from the row's coefficient sum.
#include "common.cuh"
#include "pipe_common.cuh"

namespace {

constexpr int kFlLoad = 8;                           // loader warps: warp w stages lanes 4w .. 4w+3 (frames 8w .. 8w+7 of the group)
constexpr int kFlThreads = 32 * (kFlLoad + kFlCons);
constexpr int kFlMaxStages = 4;
constexpr int kFlBarBytes = 512;                     // full[8], empty[8], flags[kFlMaxStages][kFlLoad]
constexpr int kFlFlagOffset = 128;
constexpr int kFlHdrBytes = 48;                      // as build_fl.cu
constexpr int kFlTilePix = kFlTileW * kFlTileH;
constexpr int kFlLaneBytes = kFlTilePix * 8 + 8;     // a lane's two frames of the tile, and the shift
constexpr int kFlImgBytes = 32 * kFlLaneBytes;
constexpr int kFlPassRows = 4;                       // rows of the tile a loader holds in registers at a time
constexpr int kFlPrefetchAhead = 3;                  // tiles between the L2 prefetch and the loads
constexpr int kFlMinFrames = 32;         // a context builds the layout for a batch that sends at least this many frames here
constexpr int kFlCorBytes = 2 * kFlTilePix * 4;                  // corrected variant, per stage: the tile's dark current
                                                                 // (float) and keep words (float frames)
constexpr float kFlFix = 1099511627776.0f;           // 2^40: weights of invalid pixels as integers

struct FlParams {
    const int4 *tile_desc, *chunk_desc;
    const uint8_t *chunk_owner;
    const unsigned char *blob;                       // (corrected variant: the copy with the coefficients scaled for this call)
    const unsigned char *frames;
    int64_t frame_stride_bytes;
    int height, width;
    int nframes, ngroups, nitems;
    int stages, stage_bytes, prefetch_ahead;
    const float *dark;                               // corrected variant: the call's dark current and keep words, per pixel
    const uint32_t *keep;                            // (hold.cu: hold_prep_kernel)
    const unsigned char *blob_orig;                  // the layout's own blobs
    int64_t pad_;                                    // measured: with this struct at exactly 128 bytes ptxas 12.9 allocates the
                                                     // plain variant's loader loop differently (a spill, 16 more instructions)
                                                     // and 1024 cfg4 frames take 1.205 instead of 1.14 ms
    float2 *part_s;
    unsigned long long *part_d;                      // float frames and corrected batches only
    int64_t nfp;                                     // frames rounded up to a multiple of kFlFrames
};

__device__ __forceinline__ unsigned long long pack2(float lo, float hi)
{
    return (unsigned long long)__float_as_uint(lo) | ((unsigned long long)__float_as_uint(hi) << 32);
}
__device__ __forceinline__ float lo_of(unsigned long long v) { return __uint_as_float((unsigned)v); }
__device__ __forceinline__ float hi_of(unsigned long long v) { return __uint_as_float((unsigned)(v >> 32)); }
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ unsigned long long add2(unsigned long long a, unsigned long long b)
{
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ unsigned long long sub2(unsigned long long a, unsigned long long b)
{
    unsigned long long d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ unsigned long long lds_u64(unsigned addr)
{
    unsigned long long v;
    asm volatile("ld.shared.b64 %0, [%1];" : "=l"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint4 lds_v4(unsigned addr)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts_v4(unsigned addr, const uint4 &v)
{
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void sts_f2(unsigned addr, float a, float b)
{
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(a), "f"(b) : "memory");
}
// Waits of the frame-lane kernel: bounded (20 s of wall time) like mbar_wait, but a timed-out wait raises its error with a
// store to address 0 followed by exit instead of trap.  With a trap instruction in a branch, ptxas keeps that branch at
// the launch-time register count and ignores its setmaxnreg (measured on the corrected variant: the loaders spilled their
// in-flight 128-bit loads to local memory at 80 registers and stalled on them every tile, 12.2 us per cfg3 frame; without
// the trap they use up to 108 registers, no spills, 8.6 us).  (A try_wait with a long suspend-time hint was measured to
// oversleep by microseconds once the waiting side is the faster one: plain try_wait.)
__device__ __forceinline__ void mbar_wait_fl(uint64_t *bar, uint32_t parity)
{
    unsigned long long t0 = 0;
    for (uint32_t spin = 1; !mbar_try_wait(bar, parity); ++spin) {
        if ((spin & 0xfffu) == 0) {
            const unsigned long long now = globaltimer_ns();
            if (t0 == 0) t0 = now;
            else if (now - t0 > 20000000000ULL)
                asm volatile("st.global.u32 [%0], %1;\n\texit;" ::"l"(0ULL), "r"(spin) : "memory");
        }
    }
}

// One Kahan step for the two frames of a lane, the compensation carried as e = -(running error):
// the carried value is s + e.  c2 = the coefficient in both halves.
__device__ __forceinline__ void kahan2(unsigned long long &s, unsigned long long &e, unsigned long long c2,
                                       unsigned long long v)
{
    const unsigned long long y = fma2(c2, v, e);
    // (FFMA2 / FADD2 run on one of the SM's two fp32 pipes, ~4 cycles per warp instruction; doing the two middle steps as
    // scalar adds for the other pipe was measured no faster: the kernel is bound by shared-memory wavefronts)
    const unsigned long long t = add2(s, y);
    e = add2(sub2(s, t), y);
    s = t;
}

// position in the sequence of (item, tile) this block walks: items blockIdx.x, + gridDim.x, ...; an item is a chunk of
// tiles for one group of frames, chunk-major so that neighbouring blocks share the chunk's blobs in L2
struct FlWalk {
    int item, r, r_end, group, chunk;
    bool done;
};
__device__ __forceinline__ void fl_enter(FlWalk &w, const FlParams &p)
{
    w.done = w.item >= p.nitems;
    if (w.done) return;
    w.chunk = w.item / p.ngroups;
    w.group = w.item - w.chunk * p.ngroups;
    const int4 cd = __ldg(p.chunk_desc + w.chunk);
    w.r = cd.x;
    w.r_end = cd.x + cd.y;
}
__device__ __forceinline__ void fl_next(FlWalk &w, const FlParams &p)
{
    if (++w.r < w.r_end) return;
    w.item += gridDim.x;
    fl_enter(w, p);
}

template <int DT>
__device__ __forceinline__ float fl_cast(unsigned v)
{
    if constexpr (DT == AI_F32) return __uint_as_float(v);
    else if constexpr (DT == AI_I32) return (float)(int)v;
    else return (float)v;
}

// COR: the batch carries correction arrays and / or a mask (one set for all frames).  sum c (I - dark) / den
// is computed as sum (c / den) (I - dark): the division is folded into a per-call copy of the coefficients
// (fl_scale_blob_kernel), the loaders subtract the dark current as they stage a tile.  A pixel that is invalid for every
// frame -- masked, or with a zero / non-finite denominator -- is stored as 0 (its scaled coefficients are 0 too) and its
// weight is taken off the bins' counts once per call (fl_static_count_kernel); a pixel whose I - dark is not finite is
// stored as NaN and handled per frame like a non-finite pixel of a float frame.
template <int DT, bool COR>
__global__ void __launch_bounds__(kFlThreads, 1) fl_batch_kernel(const __grid_constant__ CUtensorMap tmap, const FlParams p)
{
    constexpr bool TRACK = DT == AI_F32;      // (integer frames minus a finite dark current are finite)
    // [accumulators][barriers, flags][stages: tile of 64 frames, blob]
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *bar = smem + kFlWindow * 32 * 16;
    uint64_t *full = reinterpret_cast<uint64_t *>(bar);
    uint64_t *empty = full + 8;
    int *flags = reinterpret_cast<int *>(bar + kFlFlagOffset);
    unsigned char *stage0 = bar + kFlBarBytes;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < 8; ++s) {
            mbar_init(full + s, kFlLoad + 1);
            mbar_init(empty + s, kFlCons);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    Ring ring;
    FlWalk cur;
    cur.item = blockIdx.x;
    fl_enter(cur, p);
    if (warp < kFlLoad) {
        // ===== loaders =================================================================================================
        // two passes of 128-bit loads in registers.  The corrected variant takes what it needs (108); the plain one is held
        // at 80: it was measured 5-10 % slower with more (80 / 88 / 96 / 104 / 112 registers: 1.17 / 1.25 / 1.23 / 1.25 / 1.28 ms per
        // 1024 frames of configs[3] before the last round of changes; ptxas schedules the loads differently)
        if constexpr (COR) asm volatile("setmaxnreg.inc.sync.aligned.u32 112;");
        else asm volatile("setmaxnreg.inc.sync.aligned.u32 80;");
        // lane = (lane of the consumers, 16-byte piece of a tile row): lanes 4 lw .. 4 lw + 3 x pieces 0..7, so that the
        // 8 lanes of a 128-bit load phase read one 128-byte line.  Stores are 64-bit (one pixel of the lane's two
        // frames); pieces 4..7 store their pixels in the order 2, 3, 0, 1, which puts the 16 lanes of a store phase into
        // 16 different bank pairs.
        const int lw = warp, piece = lane & 7, cl = lw * 4 + (lane >> 3);
        const bool swap = piece >= 4;
        const int d2 = swap ? -16 : 16;
        const unsigned dst_lane = (unsigned)cl * kFlLaneBytes + (unsigned)piece * 32 + (swap ? 16u : 0u);
        const int64_t row_bytes = (int64_t)p.width * 4;
        const int tid = threadIdx.x;                                   // 0 .. 255 among the loaders
        if (tid == 0) asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap) : "memory");
        // L2 prefetch of a tile: ONE instruction (a tensor-map box of 32 pixels x 8 rows x 64 frames) by one thread
        auto prefetch_tile = [&](const FlWalk &w) {
            if (tid != 0) return;
            const int4 d = __ldg(p.tile_desc + w.r);
            asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];"
                         ::"l"(&tmap), "r"((d.z & 0xffff) * kFlTileW), "r"((d.z >> 16) * kFlTileH), "r"(w.group * kFlFrames) : "memory");
        };
        FlWalk ahead = cur;
        for (int k = 0; k < p.prefetch_ahead && !ahead.done; ++k) {
            prefetch_tile(ahead);
            fl_next(ahead, p);
        }
        // 128-bit loads of rows 4 h .. 4 h + 3 of a tile for the lane's two frames; `src` = the lane's piece of row 0
        struct Src {
            const unsigned char *p;
            int rows;                    // rows of the tile inside the image
            bool in_a, in_b, in_x;
        };
        auto locate = [&](const FlWalk &w, int4 &d) {
            d = __ldg(p.tile_desc + w.r);
            const int x = (d.z & 0xffff) * kFlTileW + piece * 4, y0 = (d.z >> 16) * kFlTileH;
            const int fa = w.group * kFlFrames + 2 * cl;
            Src s;
            s.p = p.frames + (int64_t)fa * p.frame_stride_bytes + ((int64_t)y0 * p.width + x) * 4;
            s.rows = p.height - y0;
            s.in_x = x < p.width;
            s.in_a = fa < p.nframes && s.in_x;
            s.in_b = fa + 1 < p.nframes && s.in_x;
            return s;
        };
        auto issue = [&](const Src &s, int h, uint4 (&a)[kFlPassRows], uint4 (&b)[kFlPassRows]) {
#pragma unroll
            for (int u = 0; u < kFlPassRows; ++u) {
                const int row = h * kFlPassRows + u;
                const unsigned char *q = s.p + row * row_bytes;
                a[u] = b[u] = make_uint4(0, 0, 0, 0);
                if (s.in_a && row < s.rows) a[u] = __ldcs(reinterpret_cast<const uint4 *>(q));
                if (s.in_b && row < s.rows) b[u] = __ldcs(reinterpret_cast<const uint4 *>(q + p.frame_stride_bytes));
            }
        };
        // corrected variant: the tile's dark current (0 for a pixel that is invalid for every frame: fl_prep_kernel) and,
        // for float frames, its keep words (0 for such a pixel, else all ones) travel like the frames -- loaded into
        // registers one tile ahead (one 16-byte chunk per thread: 64 threads the dark current, 64 the keep words), stored
        // into the stage when it is free; chunks outside the image read as 0
        constexpr int kCorThreads = DT == AI_F32 ? 128 : 64;
        uint4 cq = make_uint4(0, 0, 0, 0);
        auto issue_cor = [&](const FlWalk &w) {
            if constexpr (COR) {
                cq = make_uint4(0, 0, 0, 0);
                if (tid < kCorThreads) {
                    const int4 dd = __ldg(p.tile_desc + w.r);
                    const int k = tid & 63;
                    const int y = (dd.z >> 16) * kFlTileH + (k >> 3), x = (dd.z & 0xffff) * kFlTileW + (k & 7) * 4;
                    const float *src = tid < 64 ? p.dark : reinterpret_cast<const float *>(p.keep);
                    if (y < p.height && x < p.width) cq = __ldg(reinterpret_cast<const uint4 *>(src + (int64_t)y * p.width + x));
                }
            }
        };
        auto store_cor = [&](unsigned cor_s) {
            if constexpr (COR) {
                if (tid < kCorThreads) sts_v4(cor_s + (unsigned)tid * 16, cq);
                asm volatile("bar.sync 2, %0;" ::"n"(32 * kFlLoad) : "memory");      // every loader reads what these staged
            }
        };
        bool bad = false;
        auto store = [&](unsigned dst, int h, const uint4 (&a)[kFlPassRows], const uint4 (&b)[kFlPassRows], unsigned cor_s) {
#pragma unroll
            for (int u = 0; u < kFlPassRows; ++u) {
                const unsigned o = dst + (unsigned)((h * kFlPassRows + u) * kFlTileW * 8);
                float a0, a1, a2, a3, b0, b1, b2, b3;
                if constexpr (COR) {
                    // I - dark of the lane's four pixels of the row (the division is in the call's coefficients).  A pixel
                    // that is invalid for every frame gives 0 - 0 (float frames: its bits are cleared first, integer
                    // frames are finite anyway); a difference that is not finite invalidates the pixel for this frame
                    const unsigned pix = (unsigned)((h * kFlPassRows + u) * kFlTileW + piece * 4);
                    const uint4 dku = lds_v4(cor_s + pix * 4);
                    uint4 ka = a[u], kb = b[u];
                    if constexpr (DT == AI_F32) {
                        const uint4 keep = lds_v4(cor_s + kFlTilePix * 4 + pix * 4);
                        ka = make_uint4(ka.x & keep.x, ka.y & keep.y, ka.z & keep.z, ka.w & keep.w);
                        kb = make_uint4(kb.x & keep.x, kb.y & keep.y, kb.z & keep.z, kb.w & keep.w);
                    }
                    a0 = __fsub_rn(fl_cast<DT>(ka.x), __uint_as_float(dku.x)); b0 = __fsub_rn(fl_cast<DT>(kb.x), __uint_as_float(dku.x));
                    a1 = __fsub_rn(fl_cast<DT>(ka.y), __uint_as_float(dku.y)); b1 = __fsub_rn(fl_cast<DT>(kb.y), __uint_as_float(dku.y));
                    a2 = __fsub_rn(fl_cast<DT>(ka.z), __uint_as_float(dku.z)); b2 = __fsub_rn(fl_cast<DT>(kb.z), __uint_as_float(dku.z));
                    a3 = __fsub_rn(fl_cast<DT>(ka.w), __uint_as_float(dku.w)); b3 = __fsub_rn(fl_cast<DT>(kb.w), __uint_as_float(dku.w));
                } else {
                    a0 = fl_cast<DT>(a[u].x); a1 = fl_cast<DT>(a[u].y); a2 = fl_cast<DT>(a[u].z); a3 = fl_cast<DT>(a[u].w);
                    b0 = fl_cast<DT>(b[u].x); b1 = fl_cast<DT>(b[u].y); b2 = fl_cast<DT>(b[u].z); b3 = fl_cast<DT>(b[u].w);
                }
                if constexpr (TRACK)
                    bad = bad || !finite_f(a0) || !finite_f(a1) || !finite_f(a2) || !finite_f(a3) || !finite_f(b0) ||
                          !finite_f(b1) || !finite_f(b2) || !finite_f(b3);
                sts_f2(o, swap ? a2 : a0, swap ? b2 : b0);
                sts_f2(o + 8, swap ? a3 : a1, swap ? b3 : b1);
                sts_f2(o + d2, swap ? a0 : a2, swap ? b0 : b2);
                sts_f2(o + d2 + 8, swap ? a1 : a3, swap ? b1 : b3);
            }
        };
        // Steady state: both halves of the next tile are loaded (two register sets) while the current tile is cast and
        // stored, and the loader then waits for the stage of the next tile with its loads in flight.
        static_assert(kFlTileH == 2 * kFlPassRows, "a tile is two loader passes");
        uint4 a0[kFlPassRows], b0[kFlPassRows], a1[kFlPassRows], b1[kFlPassRows];
        int4 d = make_int4(0, 0, 0, 0), dn = d;
        int issued = 0;
        if (!cur.done) {
            const Src s = locate(cur, d);
            issue(s, 0, a0, b0);
            issue(s, 1, a1, b1);
            issue_cor(cur);
        }
        while (!cur.done) {
            FlWalk nxt = cur;
            fl_next(nxt, p);
            if (!ahead.done) {
                prefetch_tile(ahead);
                fl_next(ahead, p);
            }
            Src sn{};
            if (!nxt.done) sn = locate(nxt, dn);
            unsigned char *stage = stage0 + (size_t)ring.stage * p.stage_bytes;
            if (issued >= p.stages) mbar_wait_fl(empty + ring.stage, ring.parity ^ 1u);
            if (lw == 0 && lane == 0) {
                mbar_arrive_expect_tx(full + ring.stage, (uint32_t)d.y);
                bulk_g2s(stage + kFlImgBytes, p.blob + (size_t)d.x * 16, (uint32_t)d.y, full + ring.stage);
            }
            const unsigned dst = smem_u32(stage) + dst_lane;
            bad = false;
            const unsigned cor_s = smem_u32(stage) + (unsigned)(p.stage_bytes - kFlCorBytes);
            store_cor(cor_s);
            if (!nxt.done) issue_cor(nxt);            // (its registers are free again: a whole tile of time to arrive)
            store(dst, 0, a0, b0, cor_s);
            if (!nxt.done) issue(sn, 0, a0, b0);
            store(dst, 1, a1, b1, cor_s);
            if (!nxt.done) issue(sn, 1, a1, b1);
            if constexpr (TRACK) {
                const bool any = __any_sync(AI_FULL_MASK, bad);
                if (lane == 0) flags[ring.stage * kFlLoad + lw] = any ? 1 : 0;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(full + ring.stage);
            ++issued;
            ring.next(p.stages);
            d = dn;
            cur = nxt;
        }
    } else {
        // ===== consumers ===============================================================================================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
        const int cw = warp - kFlLoad;
        const unsigned acc = smem_u32(smem) + (unsigned)lane * 16;     // + bin * 512: {s of the two frames, e of the two}
        while (!cur.done) {
            // bins of this chunk's window that this warp owns
            const int4 cd = __ldg(p.chunk_desc + cur.chunk);
            const int nb = (cd.w & 0xff) + 1, bin_lo = cd.w >> 8;
            unsigned own[kFlWindow / 32];
#pragma unroll
            for (int k = 0; k < kFlWindow / 32; ++k) {
                const int bl = 32 * k + lane;
                own[k] = __ballot_sync(AI_FULL_MASK, bl < nb && __ldg(p.chunk_owner + (size_t)cur.chunk * kFlWindow + bl) == cw);
            }
#pragma unroll
            for (int k = 0; k < kFlWindow / 32; ++k)
                for (unsigned m = own[k]; m; m &= m - 1) sts_v4(acc + (unsigned)(32 * k + __ffs(m) - 1) * 512, make_uint4(0, 0, 0, 0));
            const int item = cur.item, group = cur.group;
            const int fa = group * kFlFrames + 2 * lane;
            while (!cur.done && cur.item == item) {
                mbar_wait_fl(full + ring.stage, ring.parity);
                const unsigned char *stage = stage0 + (size_t)ring.stage * p.stage_bytes;
                const unsigned char *blob = stage + kFlImgBytes;
                const unsigned short *wptr = reinterpret_cast<const unsigned short *>(blob);
                const int s0 = wptr[cw], s1 = wptr[cw + 1], nrec = wptr[kFlCons];
                const unsigned recs = smem_u32(blob) + kFlHdrBytes;
                const unsigned pairs = smem_u32(blob) + (unsigned)((kFlHdrBytes + 4 * nrec + 15) & ~15);
                const unsigned img = smem_u32(stage) + (unsigned)lane * kFlLaneBytes;
                bool tracked = false;
                if constexpr (TRACK) {
                    const int4 *fp = reinterpret_cast<const int4 *>(flags + ring.stage * kFlLoad);
                    const int4 f0 = fp[0], f1 = fp[1];
                    tracked = (f0.x | f0.y | f0.z | f0.w | f1.x | f1.y | f1.z | f1.w) != 0;
                }
                if (s0 < s1 && !tracked) {
                    // the warp's segments are contiguous in the blob: the look-ahead (entry pair two ahead, pixels one
                    // ahead) runs on across segment boundaries; two zero pairs stand behind the last one
                    unsigned rec = 0;
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(rec) : "r"(recs + 4 * s0));
                    unsigned q = pairs + (rec & 16383u) * 16;
                    uint4 w0 = lds_v4(q), w1 = lds_v4(q + 16);
                    unsigned long long v0 = lds_u64(img + w0.z), v1 = lds_u64(img + w0.w);
                    for (int s = s0; s < s1; ++s) {
                        const int np = (rec >> 14) & 1023;
                        const unsigned a_addr = acc + (rec >> 24) * 512;
                        unsigned rec_n = 0;
                        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(rec_n) : "r"(recs + 4 * s + 4));   // (one past the end: an entry pair)
                        const uint4 a = lds_v4(a_addr);
                        unsigned long long s2 = (unsigned long long)a.x | ((unsigned long long)a.y << 32);
                        unsigned long long e2 = (unsigned long long)a.z | ((unsigned long long)a.w << 32);
#pragma unroll 2
                        for (int k = 0; k < np; ++k) {
                            const uint4 w2 = lds_v4(q + 32);
                            const unsigned long long n0 = lds_u64(img + w1.z), n1 = lds_u64(img + w1.w);
                            kahan2(s2, e2, pack2(__uint_as_float(w0.x), __uint_as_float(w0.x)), v0);
                            kahan2(s2, e2, pack2(__uint_as_float(w0.y), __uint_as_float(w0.y)), v1);
                            w0 = w1; w1 = w2; v0 = n0; v1 = n1;
                            q += 16;
                        }
                        sts_v4(a_addr, make_uint4((unsigned)s2, (unsigned)(s2 >> 32), (unsigned)e2, (unsigned)(e2 >> 32)));
                        rec = rec_n;
                    }
                } else if (s0 < s1) {
                    if constexpr (TRACK) {
                        for (int s = s0; s < s1; ++s) {
                            unsigned rec;
                            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(rec) : "r"(recs + 4 * s));
                            const int np = (rec >> 14) & 1023, bl = rec >> 24;
                            const unsigned q = pairs + (rec & 16383u) * 16, a_addr = acc + bl * 512;
                            const uint4 a = lds_v4(a_addr);
                            unsigned long long s2 = (unsigned long long)a.x | ((unsigned long long)a.y << 32);
                            unsigned long long e2 = (unsigned long long)a.z | ((unsigned long long)a.w << 32);
                            unsigned long long *dd = p.part_d + (int64_t)(bin_lo + bl) * p.nfp + fa;
                            // (corrected variant: the weight that leaves the count is the matrix coefficient, not the
                            // scaled one of the stage: read from the layout's own blob)
                            const float *c_orig = reinterpret_cast<const float *>(
                                p.blob_orig + (size_t)__ldg(p.tile_desc + cur.r).x * 16 + (q - smem_u32(blob)));
                            for (int k = 0; k < 2 * np; ++k) {
                                const uint4 w = lds_v4(q + 16 * (k >> 1));
                                const float c = __uint_as_float((k & 1) ? w.y : w.x);
                                const unsigned long long v = lds_u64(img + ((k & 1) ? w.w : w.z));
                                const bool oka = finite_f(lo_of(v)), okb = finite_f(hi_of(v));
                                kahan2(s2, e2, pack2(c, c), pack2(oka ? lo_of(v) : 0.f, okb ? hi_of(v) : 0.f));
                                if (c != 0.f && !(oka && okb)) {
                                    const float cw = COR ? __ldg(c_orig + 4 * (k >> 1) + (k & 1)) : c;
                                    const unsigned long long fix = __float2ull_rn(cw * kFlFix);
                                    if (!oka && fa < p.nframes) atomicAdd(dd, fix);
                                    if (!okb && fa + 1 < p.nframes) atomicAdd(dd + 1, fix);
                                }
                            }
                            sts_v4(a_addr, make_uint4((unsigned)s2, (unsigned)(s2 >> 32), (unsigned)e2, (unsigned)(e2 >> 32)));
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + ring.stage);
                ring.next(p.stages);
                fl_next(cur, p);
            }
            // one partial per (chunk, bin, frame), written by the bin's owner: {s, e} of frame 2 lane, {s, e} of the next
#pragma unroll
            for (int k = 0; k < kFlWindow / 32; ++k)
                for (unsigned m = own[k]; m; m &= m - 1) {
                    const int bl = 32 * k + __ffs(m) - 1;
                    const uint4 a = lds_v4(acc + (unsigned)bl * 512);
                    if (fa < p.nframes)
                        *reinterpret_cast<uint4 *>(p.part_s + (int64_t)(cd.z + bl) * p.nfp + fa) = make_uint4(a.x, a.z, a.y, a.w);
                }
            // the next item deals the window's accumulators to the warps afresh: every warp must be done with this one
            asm volatile("bar.sync 1, %0;" ::"n"(32 * kFlCons) : "memory");
        }
    }
}

// Corrected batches, once per call.  (1) ai_launch_corr_prep (hold.cu): per pixel, the byte "invalid for every frame"
// (masked, zero / non-finite denominator or reciprocal, non-finite dark current), the factor its coefficients take (the
// reciprocal of flat x solid angle x polarisation, 0 for an invalid pixel), the dark current the loaders subtract (0 for
// an invalid pixel) and the keep word they AND float frames with (0 for an invalid pixel, else all ones).
// (2) fl_scale_blob_kernel: the call's copy of the tile blobs with every coefficient multiplied by its pixel's factor.
// (3) fl_static_count_kernel: the count every frame of the call starts from -- the sum of a row's coefficients over the
// pixels that are not invalid for every frame; one block per row (fp64, fixed order; a row with nothing but such pixels
// gives exactly 0).  With held corrections (ai_hold_corrections) all three are done once and kept.

// one block per tile: header and records copied, pairs {c0, c1, pos0, pos1} scaled (pos = 8 x pixel within the tile)
__global__ void __launch_bounds__(128) fl_scale_blob_kernel(const int4 *__restrict__ tile_desc,
                                                            const unsigned char *__restrict__ blob,
                                                            const float *__restrict__ scale, int width, int height,
                                                            unsigned char *__restrict__ blob_call)
{
    const int4 d = __ldg(tile_desc + blockIdx.x);
    const uint4 *src = reinterpret_cast<const uint4 *>(blob) + d.x;
    uint4 *dst = reinterpret_cast<uint4 *>(blob_call) + d.x;
    const int nq = d.y >> 4, first_pair = nq - 2 - d.w;
    const int x0 = (d.z & 0xffff) * kFlTileW, y0 = (d.z >> 16) * kFlTileH;
    auto factor = [&](unsigned pos) {
        const int pix = (int)(pos >> 3), y = y0 + pix / kFlTileW, x = x0 + pix % kFlTileW;
        return (y < height && x < width) ? __ldg(scale + (int64_t)y * width + x) : 0.f;
    };
    for (int i = threadIdx.x; i < nq; i += blockDim.x) {
        uint4 q = __ldg(src + i);
        if (i >= first_pair && i < nq - 2) {
            q.x = __float_as_uint(__fmul_rn(__uint_as_float(q.x), factor(q.z)));
            q.y = __float_as_uint(__fmul_rn(__uint_as_float(q.y), factor(q.w)));
        }
        dst[i] = q;
    }
}

__global__ void __launch_bounds__(128) fl_static_count_kernel(int npt, const int *__restrict__ indptr,
                                                              const int *__restrict__ indices,
                                                              const float *__restrict__ data,
                                                              const uint8_t *__restrict__ gone,
                                                              double *__restrict__ call_csum)
{
    __shared__ double part[4];
    const int b = blockIdx.x, lane = threadIdx.x & 31;
    double a = 0.0;
    for (int e = __ldg(indptr + b) + threadIdx.x, end = __ldg(indptr + b + 1); e < end; e += 128)
        a += __ldg(gone + __ldg(indices + e)) ? 0.0 : (double)__ldg(data + e);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if (lane == 0) part[threadIdx.x >> 5] = a;
    __syncthreads();
    if (threadIdx.x == 0) call_csum[b] = (part[0] + part[1]) + (part[2] + part[3]);
}

// H5: block = 32 bins x 32 frames; lane = frame while the partials are added (coalesced over frames), lane = bin when
// the outputs are written ([frame][bin] rows)
template <bool TRACK>
__global__ void __launch_bounds__(256) fl_finish_kernel(const int *__restrict__ bin_slot_ptr,
                                                        const int *__restrict__ bin_slots,
                                                        const double *__restrict__ bin_csum, int npt, int nframes,
                                                        int64_t nfp, const float2 *__restrict__ part_s,
                                                        const unsigned long long *__restrict__ part_d, float empty,
                                                        float *__restrict__ intensity, float *__restrict__ sum_signal,
                                                        float *__restrict__ count)
{
    __shared__ float t_i[32][33], t_s[32][33], t_c[32][33];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int b0 = blockIdx.x * 32, f0 = blockIdx.y * 32;
    for (int i = w; i < 32; i += 8) {
        const int b = b0 + i, f = f0 + lane;
        double S = 0.0, C = 0.0;
        if (b < npt && f < nframes) {
            const int beg = __ldg(bin_slot_ptr + b), end = __ldg(bin_slot_ptr + b + 1);
            for (int k = beg; k < end; ++k) {
                const float2 v = __ldcg(part_s + (int64_t)__ldg(bin_slots + k) * nfp + f);
                S += (double)v.x + (double)v.y;
            }
            const double csum = __ldg(bin_csum + b);
            C = csum;
            if constexpr (TRACK) {
                C = csum - (double)__ldcg(part_d + (int64_t)b * nfp + f) * (1.0 / (double)kFlFix);
                // all of a bin's pixels invalid: the two sums of the same coefficients differ by rounding only
                if (fabs(C) <= 1e-10 * csum) C = 0.0;
            }
        }
        t_s[i][lane] = (float)S;
        t_c[i][lane] = (float)C;
        t_i[i][lane] = C > 0.0 ? (float)(S / C) : empty;
    }
    __syncthreads();
    for (int j = w; j < 32; j += 8) {
        const int f = f0 + j, b = b0 + lane;
        if (f < nframes && b < npt) {
            const int64_t o = (int64_t)f * npt + b;
            intensity[o] = t_i[lane][j];
            sum_signal[o] = t_s[lane][j];
            count[o] = t_c[lane][j];
        }
    }
}

template <int DT, bool COR>
int launch_fl(ai_ctx *ctx, const CUtensorMap &map, const FlParams &p, size_t smem, int grid, cudaStream_t st)
{
    const uint64_t bit = 1ULL << (50 + DT + (COR ? 5 : 0));     // (bits 0..44: the other kernels' instantiations)
    if (!(ctx->smem_opt_in & bit)) {
        AI_CUDA(ctx, cudaFuncSetAttribute(fl_batch_kernel<DT, COR>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPipeSmemBudget));
        ctx->smem_opt_in |= bit;
    }
    ai_prof_begin(ctx, st);
    fl_batch_kernel<DT, COR><<<grid, kFlThreads, smem, st>>>(map, p);
    ai_prof_end(ctx, st);
    AI_CUDA(ctx, cudaGetLastError());
    return AI_OK;
}

}  // namespace

// ai_prepare_batch (include/azint.h), the frame-lane part: builds the layout now (for batches of up to `max_frames`) and
// allocates everything ai_launch_fl would otherwise allocate on the call that first needs it -- the partial sums for the
// largest batch (with the invalid-pixel weights of float frames), the per-call arrays of corrected batches, the scaled
// blobs of a held set.  Nothing here is needed for correctness: a later, larger batch still grows the buffers.
int ai_prepare_fl(ai_ctx *ctx, int max_frames, cudaStream_t st)
{
    if (max_frames < 2 || ctx->no_fl || ctx->no_tma || ctx->no_stream || ctx->npt_azim > 0 ||
        ctx->accum != AI_ACC_F32_KAHAN || ctx->layout != AI_LAYOUT_TILED)
        return AI_OK;
    if (!ctx->force_fl && max_frames < kFlMinFrames) return AI_OK;
    FlLayout &fl = ctx->fl;
    if (!fl.tried) {
        int rc = ai_build_fl(ctx, max_frames, st);
        if (rc != AI_OK) return rc;
    }
    if (!fl.ok) return AI_OK;
    const size_t nfp = (size_t)((max_frames + kFlFrames - 1) / kFlFrames) * kFlFrames;
    const size_t need = (size_t)fl.nslot * nfp * sizeof(float2) + (size_t)ctx->npt * nfp * sizeof(unsigned long long);
    if (fl.partials_bytes < need) {
        if (fl.partials) AI_CUDA(ctx, cudaFree(fl.partials));
        fl.partials = nullptr;
        fl.partials_bytes = 0;
        AI_CUDA(ctx, cudaMalloc(&fl.partials, need));
        fl.partials_bytes = need;
    }
    const int64_t npix = (int64_t)ctx->height * ctx->width;
    if (!fl.call_csum) AI_CUDA(ctx, cudaMalloc(&fl.call_csum, (size_t)ctx->npt * sizeof(double)));
    if (!fl.gone) AI_CUDA(ctx, cudaMalloc(&fl.gone, (size_t)npix));
    if (!fl.scale) AI_CUDA(ctx, cudaMalloc(&fl.scale, 3 * (size_t)npix * sizeof(float)));
    if (!fl.blob_call) AI_CUDA(ctx, cudaMalloc(&fl.blob_call, (size_t)fl.blob_bytes));
    if (ctx->held.on) {
        if (!ctx->held.fl_csum) AI_CUDA(ctx, cudaMalloc(&ctx->held.fl_csum, (size_t)ctx->npt * sizeof(double)));
        if (!ctx->held.fl_blob) AI_CUDA(ctx, cudaMalloc(&ctx->held.fl_blob, (size_t)fl.blob_bytes));
    }
    return AI_OK;
}

// Batches of 32-bit frames, Kahan accumulation, 1D: *taken = the number of leading frames of the batch the frame-lane
// kernel took (both launches); the caller sends the rest through the other kernels.  The first call that takes frames
// builds the layout (one-time; synchronises `st`).
//
// Which frames (measured, us per frame on B200).  The kernel works on groups of 64 frames and a group costs
// nearly the same full or half empty (cfg3's matrix: 365 + 0.7 per frame; cfg2's: 225 + 1.3 per frame), so full groups
// always go here and the frames behind the last full group only if there are enough of them to beat the alternative:
//   plain frames, against the slice-per-lane batch kernel (cfg3 9.8, cfg2 5.1, cfg5 29 per frame): 44 frames on matrices
//     with more than 2.2 entries per pixel, 60 below;
//   frames with per-call correction arrays, against frame-by-frame calls (cfg3 43, cfg2's matrix 34): 14 frames;
//   frames against held corrections, against frame-by-frame calls (cfg3 25, cfg2's matrix 12.5): 24 frames.
// A context that has not built the layout yet builds it for 32 frames or more.  ai_path_options.force_fl takes every batch
// (testing), ai_path_options.no_fl none.
int ai_launch_fl(ai_ctx *ctx, const FrameArgs &a0, int vec_ok, cudaStream_t st, int *taken)
{
    *taken = 0;
    if (a0.nframes < 2 || ctx->no_fl || ctx->no_tma || ctx->no_stream || ctx->npt_azim > 0 ||
        ctx->accum != AI_ACC_F32_KAHAN || ctx->layout != AI_LAYOUT_TILED)
        return AI_OK;
    const bool plain = !a0.dark && !a0.flat && !a0.solidangle && !a0.polarization && !a0.mask;
    int take = a0.nframes;
    if (!ctx->force_fl) {
        const bool heavy = (double)ctx->nnz >= 2.2 * (double)ctx->height * ctx->width;
        const int tail_min = !plain ? (a0.held ? 24 : 14) : (heavy ? 44 : 60);
        const int full = a0.nframes / kFlFrames * kFlFrames, tail = a0.nframes - full;
        take = full + (tail >= tail_min ? tail : 0);
        if (!(ctx->fl.tried && ctx->fl.ok) && take < kFlMinFrames) take = 0;
    }
    if (take < 2) return AI_OK;
    FrameArgs a = a0;
    a.nframes = take;
    const bool is32 = a.dtype == AI_F32 || a.dtype == AI_I32 || a.dtype == AI_U32;
    // (vec_ok: every array, the correction arrays and the mask included, on its 4-pixel vector boundary)
    if (!is32 || !vec_ok || (reinterpret_cast<uintptr_t>(a.image) % 16) != 0) return AI_OK;
    if (a.row_pitch != 0 && a.row_pitch != ctx->width) return AI_OK;
    FlLayout &fl = ctx->fl;
    if (!fl.tried) {
        int rc = ai_build_fl(ctx, a.nframes, st);
        if (rc != AI_OK) return rc;
    }
    if (!fl.ok) return AI_OK;
    const bool track = a.dtype == AI_F32;
    const int sms = ctx->sm_count > 0 ? ctx->sm_count : 148;

    FlParams p{};
    p.stage_bytes = kFlImgBytes + ai_align_up(fl.max_blob_bytes, 16) + (plain ? 0 : ai_align_up(kFlCorBytes, 16));
    const int acc_bytes = kFlWindow * 32 * 16;
    int stages = (kPipeSmemBudget - acc_bytes - kFlBarBytes) / p.stage_bytes;
    if (stages > kFlMaxStages) stages = kFlMaxStages;
    if (ctx->tune.fl_stages > 0 && stages > ctx->tune.fl_stages) stages = ctx->tune.fl_stages;
    if (stages < 2) return AI_OK;
    p.stages = stages;
    p.prefetch_ahead = ctx->tune.fl_prefetch > 0 ? ctx->tune.fl_prefetch : kFlPrefetchAhead;
    p.ngroups = (a.nframes + kFlFrames - 1) / kFlFrames;
    const int64_t nitems = (int64_t)fl.nchunks * p.ngroups;
    if (nitems > 0x3fffffffLL) return AI_OK;
    p.nitems = (int)nitems;
    p.nfp = (int64_t)p.ngroups * kFlFrames;
    const size_t part_bytes = (size_t)fl.nslot * (size_t)p.nfp * sizeof(float2);
    const size_t d_bytes = track ? (size_t)ctx->npt * (size_t)p.nfp * sizeof(unsigned long long) : 0;
    const size_t need = part_bytes + d_bytes;
    if (fl.partials_bytes < need) {
        // grown on demand; cudaFree synchronises the device, so work in flight on the old buffer has finished
        if (fl.partials) AI_CUDA(ctx, cudaFree(fl.partials));
        fl.partials = nullptr;
        fl.partials_bytes = 0;
        AI_CUDA(ctx, cudaMalloc(&fl.partials, need));
        fl.partials_bytes = need;
    }
    p.part_s = static_cast<float2 *>(fl.partials);
    p.part_d = track ? reinterpret_cast<unsigned long long *>(static_cast<char *>(fl.partials) + part_bytes) : nullptr;
    if (track) AI_CUDA(ctx, cudaMemsetAsync(p.part_d, 0, d_bytes, st));
    p.tile_desc = fl.tile_desc;
    p.chunk_desc = fl.chunk_desc;
    p.chunk_owner = fl.chunk_owner;
    p.blob = fl.blob;
    p.blob_orig = fl.blob;
    p.frames = static_cast<const unsigned char *>(a.image);
    p.frame_stride_bytes = a.frame_stride * 4;
    p.height = ctx->height;
    p.width = ctx->width;
    p.nframes = a.nframes;
    const int grid = p.nitems < sms ? p.nitems : sms;
    const size_t smem = (size_t)acc_bytes + kFlBarBytes + (size_t)stages * p.stage_bytes;
    CUtensorMap map{};
    int rc = ai_make_frame_map(ctx, a, kFlTileH, &map, kFlFrames);      // boxes of 64 frames: the L2 prefetch of a tile
    if (rc != AI_OK) return rc;
    // corrected batches: the count all frames share, without the pixels that are invalid for every frame
    const double *csum = fl.bin_csum;
    int launches = 0;
    if (!plain && a.held && ctx->held.on) {
        // held corrections (hold.cu): the per-pixel arrays exist; the scaled blobs and the static count are made with the
        // first batch after ai_hold_corrections and kept
        HeldCorrections &h = ctx->held;
        if (!h.fl_ready) {
            if (!h.fl_csum) AI_CUDA(ctx, cudaMalloc(&h.fl_csum, (size_t)ctx->npt * sizeof(double)));
            if (!h.fl_blob) AI_CUDA(ctx, cudaMalloc(&h.fl_blob, (size_t)fl.blob_bytes));
            fl_scale_blob_kernel<<<fl.ntiles, 128, 0, st>>>(fl.tile_desc, fl.blob, h.scale, ctx->width, ctx->height, h.fl_blob);
            fl_static_count_kernel<<<ctx->npt, 128, 0, st>>>(ctx->npt, ctx->indptr, ctx->indices, ctx->data, h.gone, h.fl_csum);
            AI_CUDA(ctx, cudaGetLastError());
            h.fl_ready = true;
            launches = 2;
        }
        csum = h.fl_csum;
        p.blob = h.fl_blob;
        p.dark = h.dark;
        p.keep = h.keep;
    } else if (!plain) {
        const int64_t npix = (int64_t)ctx->height * ctx->width;
        if (!fl.call_csum) AI_CUDA(ctx, cudaMalloc(&fl.call_csum, (size_t)ctx->npt * sizeof(double)));
        if (!fl.gone) AI_CUDA(ctx, cudaMalloc(&fl.gone, (size_t)npix));
        if (!fl.scale) AI_CUDA(ctx, cudaMalloc(&fl.scale, 3 * (size_t)npix * sizeof(float)));
        float *dark_call = fl.scale + npix;
        uint32_t *keep = reinterpret_cast<uint32_t *>(fl.scale + 2 * npix);
        if (!fl.blob_call) AI_CUDA(ctx, cudaMalloc(&fl.blob_call, (size_t)fl.blob_bytes));
        rc = ai_launch_corr_prep(ctx, a.dark, a.flat, a.solidangle, a.polarization, a.mask, fl.gone, fl.scale, dark_call, keep,
                                 nullptr, st);
        if (rc != AI_OK) return rc;
        fl_scale_blob_kernel<<<fl.ntiles, 128, 0, st>>>(fl.tile_desc, fl.blob, fl.scale, ctx->width, ctx->height, fl.blob_call);
        fl_static_count_kernel<<<ctx->npt, 128, 0, st>>>(ctx->npt, ctx->indptr, ctx->indices, ctx->data, fl.gone, fl.call_csum);
        AI_CUDA(ctx, cudaGetLastError());
        csum = fl.call_csum;
        p.blob = fl.blob_call;
        p.dark = dark_call;
        p.keep = keep;
        launches = 3;
    }
    rc = AI_EINVAL;
    switch (a.dtype) {
    case AI_F32: rc = plain ? launch_fl<AI_F32, false>(ctx, map, p, smem, grid, st) : launch_fl<AI_F32, true>(ctx, map, p, smem, grid, st); break;
    case AI_I32: rc = plain ? launch_fl<AI_I32, false>(ctx, map, p, smem, grid, st) : launch_fl<AI_I32, true>(ctx, map, p, smem, grid, st); break;
    case AI_U32: rc = plain ? launch_fl<AI_U32, false>(ctx, map, p, smem, grid, st) : launch_fl<AI_U32, true>(ctx, map, p, smem, grid, st); break;
    default: break;
    }
    if (rc != AI_OK) return rc;
    *taken = take;
    ctx->last_launches = launches + 1;
    if (ctx->stage1_only) return AI_OK;
    const dim3 g2((ctx->npt + 31) / 32, (a.nframes + 31) / 32);
    if (track)
        fl_finish_kernel<true><<<g2, 256, 0, st>>>(fl.bin_slot_ptr, fl.bin_slots, csum, ctx->npt, a.nframes, p.nfp,
                                                   p.part_s, p.part_d, ctx->empty_value, a.intensity, a.sum_signal, a.count);
    else
        fl_finish_kernel<false><<<g2, 256, 0, st>>>(fl.bin_slot_ptr, fl.bin_slots, csum, ctx->npt, a.nframes, p.nfp,
                                                    p.part_s, p.part_d, ctx->empty_value, a.intensity, a.sum_signal, a.count);
    AI_CUDA(ctx, cudaGetLastError());
    ctx->last_launches = launches + 2;
    return AI_OK;
}
