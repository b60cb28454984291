// Internal state of an ai_ctx and the declarations shared by the translation units of libazint.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/azint.h"

// Tile of the detector staged in shared memory by the TILED layout.
constexpr int kTileH = 64;
constexpr int kTileW = 64;
constexpr int kTilePix = kTileH * kTileW;
constexpr int kSegPad = 4;   // segments are padded to a multiple of 4 entries (one 128-bit coefficient load)

struct TiledLayout {
    int tiles_y = 0, tiles_x = 0, ntiles = 0;
    int nseg = 0;                  // number of (tile, bin) segments
    int64_t tnnz = 0;              // padded number of entries
    int *tile_seg_ptr = nullptr;   // [ntiles+1] first segment of each tile
    int *seg_ptr = nullptr;        // [nseg+1]   first entry of each segment (multiple of kSegPad)
    int *seg_slot = nullptr;       // [nseg]     slot of the segment's partial in the bin-major partial buffer
    int4 *seg_meta = nullptr;      // [nseg]     {first entry, padded end, partial slot, float bits of the coefficient sum}
    int4 *tile_desc = nullptr;     // [ntiles]   {first entry, number of entries, first segment, number of segments}
    int *tile_order = nullptr;     // [ntiles]   tiles by descending number of entries (longest first scheduling)
    int max_tile_entries = 0, max_tile_segs = 0;
    double *seg_csum = nullptr;    // [nseg]     sum of the segment's coefficients (count when every pixel is valid)
    float *tcoef = nullptr;        // [tnnz]     coefficient
    uint16_t *tidx = nullptr;      // [tnnz]     pixel index inside the tile (ly * kTileW + lx)
    int *bin_slot_ptr = nullptr;   // [npt+1]    partial slots of bin b are [bin_slot_ptr[b], bin_slot_ptr[b+1])
    int nslot = 0;                 // == nseg
};

struct ai_ctx {
    ai_geometry geo{};
    int height = 0, width = 0, npt = 0;
    ai_unit unit = AI_R_MM;
    bool user_range = false;
    double range_host[2] = {0.0, 0.0};   // valid after build
    ai_layout layout = AI_LAYOUT_TILED;
    ai_accum accum = AI_ACC_F32_KAHAN;
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

    // padded LUT, transposed: entry j of bin b at [j * npt + b]
    int lut_width = 0;
    float *lut_coef = nullptr;
    int32_t *lut_idx = nullptr;

    TiledLayout tl;

    // per-call scratch
    void *partials = nullptr;       // tiled stage-1 output, bin-major
    size_t partials_bytes = 0;
    void *staging = nullptr;        // device copy of a host frame (ai_integrate1d_host)
    size_t staging_bytes = 0;
    float *out_dev = nullptr;       // [3*npt] device outputs of ai_integrate1d_host

    // measurement hook (ai_profile_enable): events around the dominant kernel of the last call
    bool profile = false, profile_valid = false;
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
int ai_build_lut(ai_ctx *ctx, cudaStream_t st);
void ai_free_spans(PixelSpans *s);

// per-frame launches (integrate_*.cu) -------------------------------------------------------------------------------
struct FrameArgs {
    const void *image;
    ai_dtype dtype;
    const float *dark, *flat, *solidangle, *polarization;
    const uint8_t *mask;
    float *radial, *intensity, *sum_signal, *count;
    int nframes;
    int64_t frame_stride;
};
int ai_launch_tiled(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st);
int ai_launch_csr(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st);
int ai_launch_lut(ai_ctx *ctx, const FrameArgs &a, cudaStream_t st);
