// Internal state of an ai_ctx and the declarations shared by the translation units of libazint.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/azint.h"

// Tile of the detector staged in shared memory by the TILED layout: kTileW pixels wide and
// tile_h rows high, tile_h chosen at build time (64, 32, 16 or 8) so that two tiles' slices of the matrix plus the
// image ring fit the shared memory of one SM.
constexpr int kTileW = 64;
constexpr int kTileHMax = 64;
constexpr int kTilePixMax = kTileHMax * kTileW;
constexpr int kSegPad = 4;   // segments are padded to a multiple of 4 entries (one 128-bit coefficient load)

// Position (in floats) of pixel (ly, lx) of a tile inside its shared-memory buffer.  The buffer is the image of two TMA
// boxes of 32 pixels x tile_h rows loaded with the 128-byte swizzle: left half first, each row 128 bytes, the 16-byte
// chunk index of a row XORed with (row & 7).  Pixels above each other (a ring crossing the tile vertically) fall in
// different banks over 8 rows; every aligned group of 4 pixels stays contiguous for 128-bit stores.  The matrix
// stores these positions (as byte offsets), so the register-staged path writes the same arrangement.
__host__ __device__ inline int ai_tile_pos(int ly, int lx, int th)
{
    return (lx >> 5) * th * 32 + ly * 32 + (((((lx >> 2) & 7) ^ (ly & 7))) << 2) + (lx & 3);
}

// ---- sliced execution layout of a tile's part of the matrix --------------------------------
// Every (tile, bin) segment is cut into slices of at most kSliceMax entries; one lane of a warp owns one slice and
// walks it four entries (one 128-bit coefficient load) per step.  32 slices of similar length form a block:
//   coef  [nsteps][32] float4     idx [nsteps][32] ushort4 (byte offsets into the tile buffer)     meta [32] int2
// A tile's blocks plus a header (number of blocks, then per block  byte offset / 16 << 8 | rounds << 4 | nsteps)
// are one contiguous 16-byte aligned blob, moved to shared memory by one bulk copy.
constexpr int kSliceMax = 32;
constexpr int kSliceSteps = kSliceMax / 4;
constexpr int kBlkStepBytes = 32 * 16 + 32 * 8;     // one step of a block: 32 float4 + 32 ushort4
constexpr int kBlkMetaBytes = 32 * 8;
// meta.x: bit 31 = this lane heads a run (adjacent lanes of one segment), bits 24..28 = lanes of the run after this
// one, bits 0..23 = partial slot of the run (head only); meta.y = float bits of the run's coefficient sum (head only)
constexpr int kMetaSlotMask = 0xffffff;

// Shared-memory plan of the pipelined stage-1 kernel (integrate_pipe.cu), needed by the builder to pick tile_h.
constexpr int kPipeSmemBudget = 227 * 1024;
constexpr int kPipeHeaderBytes = 1024;
constexpr int kPipeMaxMatStages = 8;
constexpr int kPipeMaxImgStages = 8;
constexpr int kPipeMinImgStages = 3;
struct PipePlan {
    int mat_stage_bytes, mat_stages, img_stage_bytes, img_stages;
    size_t smem;
    bool fits;
};
inline int ai_align_up(int x, int a) { return (x + a - 1) / a * a; }
// Tunables (defaults chosen by measurement; ai_set_path_options reaches the few that tests
// need): largest tile height tried, caps on the matrix / image stages, tiles in flight per block.
struct PipeTune {
    int tile_h_max = 64;
    int mat_stages = 3, img_stages = 6;        // single frame
    int batch_mat_stages = 2, batch_img_stages = kPipeMaxImgStages;
    int inflight = 0;                          // 0 = as many as there are stages
    int stream_stages = 0;                     // cap on the (tile + blob) stages of the single-frame kernel, 0 = none
    int no_chain_guard = 0;                    // measurement: the stream kernel does not wait for the count of ended finish blocks
    int fin_blocks_per_sm = 0;                 // finish kernel of the single-frame chain: blocks per SM at most, 0 = default
    int no_overlap = 0;                        // single-frame kernel: never stream ahead of the grid dependency
    int batch_units = 0;                       // batched kernel: 1 = (block, frame) units, 2 = (block, two frames), 0 = by layout
    int fl_stages = 0;                         // frame-lane kernel: cap on the stages, 0 = none
    int fl_prefetch = 0;                       // frame-lane kernel: tiles between the L2 prefetch and the loads, 0 = default
    int fl_owner = 0;                          // frame-lane layout: 1 = bins dealt to the warps longest-first instead of round-robin
    int fl_chunk = 0;                          // frame-lane layout: tiles per chunk, 0 = by the size of the first batch
};
inline PipePlan ai_pipe_plan(int max_blob_bytes, int tile_h, bool batch, const PipeTune &tune = PipeTune())
{
    PipePlan p{};
    p.mat_stage_bytes = ai_align_up(max_blob_bytes > 16 ? max_blob_bytes : 16, 1024);   // image stages stay 1 KB aligned
    p.img_stage_bytes = tile_h * kTileW * 4;
    int ms_max = batch ? tune.batch_mat_stages : tune.mat_stages;
    int is_max = batch ? tune.batch_img_stages : tune.img_stages;
    ms_max = ms_max < 2 ? 2 : (ms_max > kPipeMaxMatStages ? kPipeMaxMatStages : ms_max);
    is_max = is_max < kPipeMinImgStages ? kPipeMinImgStages : (is_max > kPipeMaxImgStages ? kPipeMaxImgStages : is_max);
    for (p.mat_stages = ms_max; p.mat_stages >= 2; --p.mat_stages) {
        const int room = kPipeSmemBudget - kPipeHeaderBytes - p.mat_stages * p.mat_stage_bytes;
        p.img_stages = room > 0 ? room / p.img_stage_bytes : 0;
        if (p.img_stages > is_max) p.img_stages = is_max;
        if (p.img_stages >= kPipeMinImgStages) break;
    }
    if (p.mat_stages < 2) p.mat_stages = 2;
    p.fits = p.img_stages >= kPipeMinImgStages;
    p.smem = (size_t)kPipeHeaderBytes + (size_t)p.mat_stages * p.mat_stage_bytes + (size_t)p.img_stages * p.img_stage_bytes;
    return p;
}

struct TiledLayout {
    int tile_h = 0;                // rows per tile
    int tiles_y = 0, tiles_x = 0, ntiles = 0;
    int nseg = 0;                  // number of (tile, bin) segments
    int64_t tnnz = 0;              // padded number of entries
    int *tile_seg_ptr = nullptr;   // [ntiles+1] first segment of each tile
    int *seg_ptr = nullptr;        // [nseg+1]   first entry of each segment (multiple of kSegPad), segments in bin order
    int *seg_slot = nullptr;       // [nseg]     slot of the segment's partial in the bin-major partial buffer
    int4 *seg_meta = nullptr;      // [nseg]     {first entry, padded end, partial slot, float bits of the coefficient
                                   //            sum}; within a tile ordered by descending length (lanes of a warp work
                                   //            on segments of similar length)
    int4 *tile_desc = nullptr;     // [ntiles]   {first entry, number of entries, first segment, number of segments}
    int *tile_order = nullptr;     // [ntiles]   tiles by descending number of entries (longest first scheduling)
    int max_tile_entries = 0, max_tile_segs = 0;
    // sliced layout (pipelined kernel)
    unsigned char *blob = nullptr; // all tiles' blobs, tile t at 16 * blob_desc[rank].x
    int4 *blob_desc = nullptr;     // [ntiles] longest first: {blob offset / 16, blob bytes, tile row << 16 | tile column, number of blocks}
    int4 *h_first_desc = nullptr;  // HOST copy of blob_desc (the single-frame kernel takes each block's first tiles by value)
    int64_t blob_bytes = 0;
    int max_blob_bytes = 0;
    double *seg_csum = nullptr;    // [nseg]     sum of the segment's coefficients (count when every pixel is valid)
    float *tcoef = nullptr;        // [tnnz]     coefficient
    uint16_t *tidx = nullptr;      // [tnnz]     ai_tile_pos of the pixel inside the tile
    int *bin_slot_ptr = nullptr;   // [npt+1]    partial slots of bin b are [bin_slot_ptr[b], bin_slot_ptr[b+1])
    int nslot = 0;                 // number of partials per frame: one per run of the sliced layout
};

// ---- frame-lane layout (build_fl.cu, integrate_fl.cu): batches of plain 32-bit frames ----------
// The batched kernel turns the problem by 90 degrees: a warp's 32 lanes are 32 PAIRS OF FRAMES, an entry (coefficient,
// pixel) is warp-uniform and serves all 64 of them.  Tiles of kFlTileW x kFlTileH pixels of 64 frames are staged in
// shared memory (the two frames of a lane interleaved pixel by pixel, lane l shifted by 2 l words: the 32 lanes of a
// gather fall into 32 different bank pairs); tiles are taken in order of their lowest bin and cut into chunks whose
// bins fit a window of kFlWindow shared-memory accumulators per frame, so that one partial per (chunk, bin, frame)
// leaves the SM instead of one per (tile, bin, frame).
constexpr int kFlTileW = 32, kFlTileH = 8;
constexpr int kFlFrames = 64;       // frames per group = two per lane of a warp
constexpr int kFlWindow = 128;      // bins a chunk may touch
constexpr int kFlCons = 16;         // consumer warps; a bin of a chunk belongs to one of them
constexpr int kFlChunkTilesMax = 64; // tiles per chunk at most (fewer where the window would overflow, or for small batches)
struct FlLayout {
    bool tried = false, ok = false;
    int tiles_x = 0, tiles_y = 0;
    int ntiles = 0;                 // tiles that hold entries
    int nchunks = 0, nslot = 0;
    int4 *tile_desc = nullptr;      // [ntiles] in chunk order: {blob offset / 16, blob bytes, tile row << 16 | column, pairs}
    int4 *chunk_desc = nullptr;     // [nchunks] {first tile, tiles, first slot, lowest bin << 8 | bins in the window - 1}
    uint8_t *chunk_owner = nullptr; // [nchunks][kFlWindow] consumer warp that owns bin (lowest bin of the chunk + k)
    unsigned char *blob = nullptr;
    int64_t blob_bytes = 0;
    int max_blob_bytes = 0;
    int *bin_slot_ptr = nullptr;    // [npt+1] H5: partial slots of bin b are bin_slots[bin_slot_ptr[b] .. bin_slot_ptr[b+1])
    int *bin_slots = nullptr;       //         ascending chunk
    double *bin_csum = nullptr;     // [npt] sum of the row's coefficients (count when every pixel is valid)
    double *call_csum = nullptr;    // [npt] corrected batches: the same without the pixels invalid for every frame, per call
    uint8_t *gone = nullptr;        // [npix] corrected batches: 1 = the pixel is invalid for every frame of the call
    float *scale = nullptr;         // [3][npix] corrected batches, per call: 1 / (flat x solid angle x polarisation) (0 where
                                    // gone), dark current (0 where gone), keep word (0 where gone, else all ones)
    unsigned char *blob_call = nullptr;   // corrected batches: blob with the coefficients times scale, rewritten per call
    void *partials = nullptr;       // [nslot][frames rounded up to 64] float2 (sum, compensation), then, for float
                                    // frames, [npt][frames rounded up] uint64: weight of the invalid pixels, 2^-40 units
    size_t partials_bytes = 0;
};

// ---- held corrections (hold.cu) ----------------------------------------------------------------------------------------
struct HeldCorrections {
    bool on = false;
    uint8_t *gone = nullptr;        // [npix] 1 = invalid for every frame
    float *scale = nullptr;         // [4][npix], one allocation: 1 / den (0 where gone), then
    float *dark = nullptr;          //   the dark current (0 where gone),
    uint32_t *keep = nullptr;       //   the keep word (all ones, 0 where gone),
    float *den = nullptr;           //   the denominator (0 where gone)
    unsigned char *tl_blob = nullptr;   // tiled blobs: coefficients x scale, run sums without the gone pixels
    bool tl_ready = false;
    unsigned char *fl_blob = nullptr;   // frame-lane blobs, coefficients x scale (built with the first frame-lane batch)
    double *fl_csum = nullptr;          // [npt] the frame-lane finish kernel's count without the gone pixels
    bool fl_ready = false;
};

struct ai_ctx {
    ai_geometry geo{};
    int height = 0, width = 0, npt = 0;   // npt = number of bins = rows of the matrix (2D: npt_azim * npt_rad)
    int npt_rad = 0, npt_azim = 0;        // bidimensional integration (ai_setup2d): row = a * npt_rad + r; 1D: npt_azim = 0
    double azim_host[2] = {-3.14159265358979323846, 3.14159265358979323846};   // azimuthal range, radians
    float *axes2d = nullptr;              // [npt_rad + npt_azim] bin centres of the two axes (device)
    ai_unit unit = AI_R_MM;
    bool user_range = false;
    double range_host[2] = {0.0, 0.0};   // valid after build
    ai_layout layout = AI_LAYOUT_TILED;
    ai_accum accum = AI_ACC_F32_KAHAN;
    ai_norm norm = AI_NORM_PIXEL;
    ai_split split = AI_SPLIT_BBOX;
    float *norm_scratch = nullptr;        // [2 * npt] throw-away outputs of the two passes of AI_NORM_SPLIT
    float empty_value = 0.0f;
    int device = 0;
    int sm_count = 0;
    bool built = false;
    int last_launches = 0;
    char err[512] = {0};

    // canonical CSR
    int64_t nnz = 0;
    int32_t *indptr = nullptr;    // [npt+1]
    int32_t *indices = nullptr;   // [nnz]
    float *data = nullptr;        // [nnz]
    float *row_csum = nullptr;    // [npt] sum of each row's coefficients
    double *d_range = nullptr;    // [2] u0, u1 on the device

    // segments of the canonical CSR's rows for AI_LAYOUT_CSR (integrate_csr.cu), built on first use
    void *csr_seg = nullptr;              // int4 {row, first entry, end entry, -}
    int *csr_row_seg_ptr = nullptr;       // [npt+1]
    int csr_nseg = 0;
    void *csr_partials = nullptr;         // [nframes][csr_nseg] double2
    size_t csr_partials_bytes = 0;
    // AI_LAYOUT_SCATTER (integrate_scatter.cu): 12 bytes of split geometry per pixel, built on first use
    int *scat_first_nb = nullptr;
    void *scat_gw = nullptr;              // float2 {lower bound relative to the first bin, width in bins}
    // padded LUT, row-major: entry j of bin b at [b * lut_width + j], lut_width a multiple of 4
    int lut_width = 0;
    float *lut_coef = nullptr;
    int32_t *lut_idx = nullptr;

    TiledLayout tl;
    FlLayout fl;
    HeldCorrections held;

    // per-call scratch
    void *partials = nullptr;       // tiled stage-1 output, bin-major
    size_t partials_bytes = 0;
    void *staging = nullptr;        // device copy of a host frame (ai_integrate1d_host)
    size_t staging_bytes = 0;
    float *out_dev = nullptr;       // [3*npt] device outputs of ai_integrate1d_host
    // ai_integrate1d_host_frames: double-buffered upload
    void *stage2[2] = {nullptr, nullptr};
    size_t stage2_bytes = 0, out2_floats = 0;
    bool host_frames_ready = false;
    float *out2[2] = {nullptr, nullptr};
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t h2d_done[2] = {nullptr, nullptr}, slot_free[2] = {nullptr, nullptr};
    void *stream_first = nullptr;   // HOST: descriptors of every block's first tiles, as the single-frame kernel takes them
    int stream_first_grid = 0;
    float *corrected[2] = {nullptr, nullptr};   // corrected float32 frames (integrate_prep.cu), alternating, allocated on first use
    unsigned prep_launches = 0;
    // single-frame kernel: tile-ticket counters and partial records in alternating sets (two launches of a context may
    // be resident at a time, integrate_stream.cu)
    unsigned long long *grid_sync = nullptr;   // [3] tile tickets, used in rotation
    void *stream_partials = nullptr;           // [2][nslot] partial records
    unsigned stream_launches = 0;              // single-frame launches of this context so far
    // Blocks of finish kernels of this context that have ended, ever increasing.  The launch chain re-uses a set of
    // partial sums (and a corrected frame) every second call on the argument that a block of the stream kernel only
    // becomes resident where a block of the previous launch has left; another tenant of the GPU (a second context on a
    // second stream) frees SMs out of turn, so the kernels that re-use check this count as well (normally long reached).
    unsigned long long *chain_done = nullptr;  // device
    unsigned long long fin_cum = 0, fin_cum_prev = 0;   // the count after every finish kernel launched so far / all but the last
    uint64_t stream_shared_sm = 0;             // bit k: instantiation k of the kernel does NOT have an SM to itself
    // tensor map of the last frame buffer seen by the TMA kernels (encoding one costs the host ~1-2 us per call)
    struct MapEntry {
        alignas(64) unsigned char map[128];
        const void *image = nullptr;
        int dtype = -1, tile_h = 0, nframes = 0;
        int64_t pitch = 0, stride = 0;
    } map_cache[8];
    unsigned map_next = 0;          // entry replaced next (round robin)
    uint64_t smem_opt_in = 0;       // bit k: kernel instantiation k was given its dynamic shared-memory size (per context:
                                    // no function-local static state, two host threads may drive two contexts)

    // measurement hook (ai_profile_enable): events around the dominant kernel of the last call
    PipeTune tune;
    bool no_tma = false;            // ai_path_options.no_tma: stage raw frames through registers even where TMA applies (testing)
    bool no_schedule = false;       // ai_path_options.no_schedule: skip the bank scheduling of the sliced layout (measurement)
    bool no_prepass = false;        // ai_path_options.no_prepass: corrected single frames take the general kernel (testing)
    bool no_stream = false;         // ai_path_options.no_stream: single frames take the general pipelined kernel too (testing)
    bool force_fl = false;          // ai_path_options.force_fl: every batch of plain 32-bit frames takes the frame-lane kernel (testing)
    bool no_fl = false;             // ai_path_options.no_fl: large batches stay on the slice-per-lane batched kernel (testing)
    bool profile = false, profile_valid = false;
    bool stage1_only = false;       // ai_profile_enable(ctx, 2): launch only the dominant kernel
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
};

// events around the dominant kernel when profiling is on (no-ops otherwise)
inline void ai_prof_begin(ai_ctx *ctx, cudaStream_t st) { if (ctx->profile) cudaEventRecord(ctx->ev0, st); }
inline void ai_prof_end(ai_ctx *ctx, cudaStream_t st)
{
    if (ctx->profile) { cudaEventRecord(ctx->ev1, st); ctx->profile_valid = true; }
}

// error plumbing -------------------------------------------------------------------------------------------------
int ai_fail(ai_ctx *ctx, int code, const char *fmt, ...);
#define AI_CUDA(ctx, call)                                                                              \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess)                                                                          \
            return ai_fail((ctx), e_ == cudaErrorMemoryAllocation ? AI_ENOMEM : AI_ECUDA, "%s: %s (%s:%d)", #call, \
                           cudaGetErrorString(e_), __FILE__, __LINE__);                                 \
    } while (0)

// builders (build_csr.cu, build_tiled.cu) --------------------------------------------------------------------------
struct PixelSpans {              // per-pixel result of the bounds pass, kept only during the build
    double *fmin = nullptr;      // lower bound in bin units, (u_min - u0) / delta
    double *fmax = nullptr;
    int *first = nullptr;        // first bin with a positive overlap
    int *nb = nullptr;           // number of bins with a positive overlap (0 = pixel outside the range)
};
int ai_build_canonical(ai_ctx *ctx, PixelSpans *spans, cudaStream_t st);
int ai_build_tiled(ai_ctx *ctx, const PixelSpans &spans, cudaStream_t st);
int ai_build_2d(ai_ctx *ctx, cudaStream_t st);
int ai_build_full(ai_ctx *ctx, cudaStream_t st);    // build_2d.cu: full pixel splitting, 1D      // build_2d.cu: canonical CSR + tiled layout of the 2D matrix
int ai_build_lut(ai_ctx *ctx, cudaStream_t st);
void ai_free_spans(PixelSpans *s);
int ai_build_spans(ai_ctx *ctx, PixelSpans *sp, int npt, cudaStream_t st);

// per-frame launches (integrate_*.cu) -------------------------------------------------------------------------------
struct FrameArgs {
    const void *image;
    ai_dtype dtype;
    const float *dark, *flat, *solidangle, *polarization;
    const uint8_t *mask;
    float *radial, *intensity, *sum_signal, *count;
    int nframes;
    int64_t frame_stride;
    int64_t row_pitch = 0;       // elements between rows of `image`; 0 = width (only the library's own corrected frame differs)
    bool held = false;           // the call uses the context's held corrections (dark / flat point at their derived arrays)
};
int ai_launch_tiled(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st);
int ai_launch_tiled_split(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st);
int ai_launch_csr(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st);
int ai_launch_lut(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st);
int ai_launch_scatter(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st);
int ai_build_fl(ai_ctx *ctx, int nframes, cudaStream_t st);                          // build_fl.cu: frame-lane layout from the canonical CSR
void ai_free_fl(FlLayout &fl);
int ai_prepare_fl(ai_ctx *ctx, int max_frames, cudaStream_t st);                         // integrate_fl.cu
int ai_launch_fl(ai_ctx *ctx, const FrameArgs &a, int vec_ok, cudaStream_t st, int *taken);   // integrate_fl.cu
int ai_launch_corr_prep(ai_ctx *ctx, const float *dark, const float *flat, const float *solidangle, const float *polarization,
                        const uint8_t *mask, uint8_t *gone, float *scale, float *dark_out, uint32_t *keep, float *den_out,
                        cudaStream_t st);                                                    // hold.cu
void ai_release_held(ai_ctx *ctx);                                                     // hold.cu
int ai_hold_build(ai_ctx *ctx, const float *dark, const float *flat, const float *solidangle, const float *polarization,
                  const uint8_t *mask, cudaStream_t st);
int ai_launch_correct(ai_ctx *ctx, const FrameArgs &a, int vec_ok, int overlap, int mode, cudaStream_t st, float **out);   // integrate_prep.cu
int ai_stream_full_grid(const ai_ctx *ctx);   // integrate_stream.cu: 1 if the single-frame kernel puts one block on every SM
int ai_stream_stages(const ai_ctx *ctx);      // integrate_stream.cu: (tile + blob) stages of the single-frame kernel, 0 = n/a
