/*
 * azint.h -- C ABI of libazint: the 1D azimuthal-integration hot path of arxiv 1412.6367 (pyFAI) on one B200.
 *
 * What the library computes (citations are PAPER.md lines; DESIGN.md section 3 holds the exact definition O1-O7):
 *   - per-pixel radial bounds of the pixel's bounding box in r, 2theta or q   (PAPER.md:32-41 section 3, :50, :120)
 *   - the bounding-box pixel-splitting matrix "bin <- (pixel, weight)" in CSR form: data / indices / indptr,
 *     scipy.sparse.csr_matrix compatible                                      (PAPER.md:122 section 4.1, :159-180)
 *   - per frame: cast + dark / flat / solid-angle / polarisation / mask correction in one pass over the pixels
 *     (PAPER.md:240), the sparse matrix x dense vector product with compensated accumulation and the
 *     three outputs weighted histogram, unweighted histogram and their ratio
 *
 * Conventions
 *   - Every function returns AI_OK (0) or a negative ai_status; nothing throws or aborts across this boundary.
 *   - "DEVICE pointer" = CUDA global memory on the current device; "HOST pointer" = ordinary host memory.
 *     The caller owns every buffer it passes in; the library never frees, keeps or modifies them beyond the
 *     documented outputs.  The library owns the context, the matrix and its scratch buffers.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream).  ai_integrate1d* only ENQUEUE work on that
 *     stream and return without synchronising.  ai_build_csr synchronises the stream (it reads nnz back to size the
 *     matrix).  One context must not be used from two streams at once (it owns per-call scratch).
 *   - Image layout: height x width, row-major, linear pixel index p = i*width + j (i = slow / y, j = fast / x).  Pixel
 *     (i, j) covers [j, j+1] x [i, i+1] in pixel units; the beam centre is given in the same units.
 *   - Frames and correction arrays need only their natural alignment (4 bytes for 32-bit, 2 bytes for 16-bit types).
 */
#ifndef AZINT_H
#define AZINT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ai_ctx ai_ctx; /* opaque, library-owned */

typedef enum {
    AI_OK = 0,
    AI_EINVAL = -1,    /* bad shape, npt < 1, non-positive distance / pixel / wavelength, NULL required pointer, u1 <= u0 */
    AI_ENOTBUILT = -2, /* integrate or get_csr before ai_build_csr */
    AI_ECUDA = -3,     /* a CUDA call failed; text kept for ai_last_error */
    AI_ENOMEM = -4,    /* host or device allocation failed */
    AI_EUNSUPPORTED = -5 /* e.g. a matrix with more than 2^31-1 entries or a LUT that would exceed device memory */
} ai_status;

/* radial unit u(r): r in mm; 2theta = atan(r/d) in degrees or radians;
 * q = 4 pi sin(2theta / 2) / lambda in nm^-1 or A^-1 */
typedef enum { AI_R_MM = 0, AI_TTH_DEG = 1, AI_TTH_RAD = 2, AI_Q_NM = 3, AI_Q_A = 4 } ai_unit;

/* dtype of the raw frame: "16 or 32 bits (int or uint)" or float32 */
typedef enum { AI_F32 = 0, AI_I32 = 1, AI_U16 = 2, AI_I16 = 3, AI_U32 = 4 } ai_dtype;

/* execution layout of the matrix.
 *   AI_LAYOUT_TILED  B200 design: the CSR re-ordered by image tile, tiles staged in shared memory
 *   AI_LAYOUT_CSR    the canonical CSR, one warp per row segment, 128-bit loads
 *   AI_LAYOUT_LUT    padded look-up table, one warp per bin
 *   AI_LAYOUT_TILED_DIRECT  the tiled layout with one thread block per tile and plain loads of the matrix: the
 *                    fallback AI_LAYOUT_TILED takes when a tile's slice of the matrix exceeds its shared-memory ring
 *   AI_LAYOUT_SCATTER  no matrix at all: the forward scatter of PAPER.md:122 with fp32 atomics ("linear read / random
 *                    write") -- a measured comparison, NOT compensated and NOT bit-reproducible  */
typedef enum { AI_LAYOUT_TILED = 0, AI_LAYOUT_CSR = 1, AI_LAYOUT_LUT = 2, AI_LAYOUT_TILED_DIRECT = 3,
               AI_LAYOUT_SCATTER = 4 } ai_layout;

/* accumulator arithmetic: fp32 with Kahan compensation, plain fp32, or fp64 */
typedef enum { AI_ACC_F32_KAHAN = 0, AI_ACC_F32_PLAIN = 1, AI_ACC_F64 = 2 } ai_accum;

/* where the division by the normalisation happens (the paper lists the corrections, not this):
 *   AI_NORM_PIXEL  every pixel is corrected, v = (I - dark) / (flat * solidangle * polarization), then averaged with the
 *                  split weights: intensity = sum c v / sum c                                    (default)
 *   AI_NORM_SPLIT  signal and normalisation are summed separately with the same weights and the sums divided:
 *                  sum_signal = sum c (I - dark), count = sum c (flat * solidangle * polarization), intensity = their
 *                  ratio (`count` then carries the summed normalisation).  One 1D frame per call, AI_LAYOUT_TILED. */
typedef enum { AI_NORM_PIXEL = 0, AI_NORM_SPLIT = 1 } ai_norm;

/* pixel-splitting scheme of the matrix (section 4):
 *   AI_SPLIT_BBOX  bounding box: the pixel's extent along the radial axis, split by overlap / width
 *   AI_SPLIT_FULL  full pixel splitting: the quadrilateral of the pixel's four corners in the (radial
 *                  unit, chi) plane with straight sides; weight = area between the bin's edges / area of the whole.  A
 *                  pixel that holds the beam centre strictly inside, or has no area in that plane, keeps its bounding box.
 *                  1D only.  The automatic range is the bounding-box one in both schemes. */
typedef enum { AI_SPLIT_BBOX = 0, AI_SPLIT_FULL = 1 } ai_split;

/* planar detector orthogonal to the beam; lengths in metres, centre in pixels */
typedef struct {
    double distance_m;
    double pixel_y_m, pixel_x_m;
    double center_y_px, center_x_px;
    double wavelength_m;
} ai_geometry;

/* Create a context (host work only, no device allocation yet).
 *   out             receives the context; destroy with ai_destroy
 *   g               geometry; distance, pixel sizes > 0; wavelength > 0 (only used by the q units)
 *   height, width   detector shape in pixels, >= 1
 *   npt             number of radial bins, >= 1
 *   range_or_null   HOST pointer to {u0, u1} in `unit`, u1 > u0; NULL = [min u_min, max u_max] over all pixels
 * Errors: AI_EINVAL, AI_ENOMEM. */
int ai_setup(ai_ctx **out, const ai_geometry *g, int height, int width, int npt, ai_unit unit,
             const double *range_or_null);

/* Bidimensional ("cake") integration ("mono- and bidimensional integration"; Fig. 3): bins
 * = npt_azim azimuthal x npt_rad radial.  The azimuthal coordinate is chi = atan2(y, x), y along the image
 * rows and x along the columns, both from the beam centre; the axis is periodic (a pixel across the negative x axis is
 * split over the seam).  The weight of a pixel in a bin is the bounding box of PAPER.md:120 taken on both axes: its
 * overlap / width along the radial unit times its overlap / width along chi.
 *   npt_rad, npt_azim    >= 1, npt_rad * npt_azim < 2^28
 *   range_or_null        HOST {u0, u1} in `unit`, NULL = automatic (as ai_setup)
 *   azim_range_or_null   HOST {chi0, chi1} in RADIANS, 0 < chi1 - chi0 <= 2 pi, -2 pi <= chi0, chi1 <= 3 pi; NULL = the
 *                        full circle [-pi, pi]
 * Then ai_build_csr, ai_get_csr (rows = bins, row index a * npt_rad + r) and ai_integrate2d; ai_set_options applies
 * (AI_LAYOUT_LUT is not offered in 2D).  Errors: AI_EINVAL, AI_ENOMEM. */
int ai_setup2d(ai_ctx **out, const ai_geometry *g, int height, int width, int npt_rad, int npt_azim, ai_unit unit,
               const double *range_or_null, const double *azim_range_or_null);

/* Choose the pixel-splitting scheme; between ai_setup and ai_build_csr.  Errors: AI_EINVAL (unknown value, or the matrix
 * is already built), AI_EUNSUPPORTED (AI_SPLIT_FULL on a bidimensional context). */
int ai_set_splitting(ai_ctx *ctx, ai_split split);

/* Which kernels a context may use, for tests and measurements (every switch 0 = the library's own choice, which is what
 * production code wants).  The library reads no environment variable: this call is the only way to re-route frames.
 *   no_tma       frames are staged through registers even where a TMA tensor map applies
 *   no_schedule  the sliced layout is built without its shared-memory bank scheduling
 *   no_prepass   corrected single frames are corrected inside the general pipelined kernel, not by a pre-pass
 *   no_stream    single frames take the general pipelined kernel instead of the single-frame kernel chain
 *   no_fl        batches never take the frame-lane kernel         force_fl   batches of 32-bit frames always take it
 *   no_overlap   every kernel of the single-frame chain waits for the kernel before it (no early reads of the frame)
 *   fl_chunk     frame-lane layout: tiles per chunk (0 = chosen from the first batch's size)
 *   fl_stages    frame-lane kernel: cap on its shared-memory stages (0 = none)
 *   fl_owner     frame-lane layout: 1 = bins dealt to the warps longest first instead of round-robin
 * Between ai_setup / ai_setup2d and ai_build_csr (some switches shape the layouts); NULL = all defaults.
 * Errors: AI_EINVAL (matrix already built, negative sizes, no_fl with force_fl, a non-zero reserved field). */
typedef struct {
    int no_tma, no_schedule, no_prepass, no_stream, no_fl, force_fl, no_overlap;
    int fl_chunk, fl_stages, fl_owner;
    int reserved[6]; /* zero */
} ai_path_options;
int ai_set_path_options(ai_ctx *ctx, const ai_path_options *opt);

/* Build the matrix on the device: bounds -> range -> count -> exclusive scan -> ordered fill (PAPER.md:120-122 for
 * the coefficients, :150 scan, :180 CSR), then the tiled execution layout.  Idempotent.  Synchronises `cuda_stream`.
 * Errors: AI_ECUDA, AI_ENOMEM, AI_EUNSUPPORTED. */
int ai_build_csr(ai_ctx *ctx, void *cuda_stream);

/* Borrow the canonical CSR (DEVICE pointers, valid until ai_destroy): indptr[npt+1], indices[nnz] ascending within
 * each row, data[nnz] float32.  Any output pointer may be NULL.  u0/u1 = the range in use.
 * Errors: AI_ENOTBUILT. */
int ai_get_csr(const ai_ctx *ctx, const int32_t **indptr, const int32_t **indices, const float **data,
               int64_t *nnz, double *u0, double *u1);

/* Copy the canonical CSR into HOST buffers of indptr[npt+1], indices[nnz], data[nnz] elements (sizes from ai_get_csr);
 * any pointer may be NULL.  Synchronous.  Errors: AI_ENOTBUILT, AI_ECUDA. */
int ai_copy_csr_to_host(const ai_ctx *ctx, int32_t *indptr_host, int32_t *indices_host, float *data_host);

/* Choose execution layout, accumulator and the intensity written to bins with count == 0 (default: TILED, KAHAN, 0).
 * AI_LAYOUT_LUT builds the padded table on first use (inside the next integrate call's stream).
 * Errors: AI_EINVAL. */
int ai_set_options(ai_ctx *ctx, ai_layout layout, ai_accum accum, float empty_value);

/* Choose the estimator (see ai_norm).  Errors: AI_EINVAL; an integrate call that cannot honour AI_NORM_SPLIT (batches,
 * bidimensional contexts, other layouts) returns AI_EUNSUPPORTED. */
int ai_set_normalization(ai_ctx *ctx, ai_norm norm);

/* Integrate one frame.  All pointers are DEVICE pointers.
 *   image                      height*width elements of `dtype`
 *   dark, flat, solidangle,
 *   polarization               float32[height*width] or NULL (absent = 0 for dark, 1 for the others)
 *   mask                       uint8[height*width] or NULL; mask != 0 => pixel ignored
 *   radial                     float32[npt] bin centres u0 + (b + 1/2) delta, may be NULL
 *   intensity, sum_signal,
 *   count                      float32[npt] each, required:  sum_signal_b = sum_k c_k v_k, count_b = sum_k c_k valid_k,
 *                              intensity_b = sum_signal_b / count_b (empty_value where count_b == 0), with
 *                              v = (I - dark) / (flat * solidangle * polarization); a pixel is invalid if masked or if
 *                              its denominator is 0 / non-finite or its numerator non-finite.
 * Enqueues on `cuda_stream`; does not synchronise.  Errors: AI_EINVAL, AI_ENOTBUILT, AI_ECUDA.
 * With the default layout a plain 32-bit frame is two kernel launches (the streaming product and a small finish
 * kernel); correction arrays, a mask, 16-bit pixels or rows off 16-byte boundaries add one streaming pre-pass.  The
 * kernels are launched with programmatic stream serialisation so that consecutive calls overlap:
 *   - everything a call WRITES (outputs, the context's scratch) is written in stream order, after all earlier work;
 *   - what a call READS -- the frame and the correction arrays -- may be read as soon as the kernel enqueued right
 *     before it on the stream has completed OR has executed griddepcontrol.launch_dependents
 *     (cudaTriggerProgrammaticLaunchCompletion).  Memory copies, memsets and kernels that never trigger early -- every
 *     ordinary kernel -- give plain stream ordering.  A producer kernel that does trigger early must be followed by
 *     any ordinary stream operation before the call (or build the context with ai_path_options.no_overlap = 1).
 * Between calls the context keeps corrected copies of the frame, partial sums and ticket counters: one context is used
 * by one host thread and on one stream at a time (different contexts are independent), on the device it was built on
 * (AI_EINVAL otherwise). */
int ai_integrate1d(ai_ctx *ctx, const void *image, ai_dtype dtype, const float *dark, const float *flat,
                   const float *solidangle, const float *polarization, const uint8_t *mask, float *radial,
                   float *intensity, float *sum_signal, float *count, void *cuda_stream);

/* ai_integrate1d for callers that must not allocate device memory once they are running.
 *
 * Why it exists: every other integrate entry may call cudaMalloc (and cudaFree, which waits for the whole device) the
 * first time a call needs a library-owned buffer -- partial sums sized by the batch, a corrected copy of the frame, the
 * padded table, the frame-lane layout.  That is no good for (a) a process where something else already owns all device
 * memory (a framework's caching allocator, a fixed memory budget per tenant on a shared GPU): the library's own
 * cudaMalloc fails there; (b) a real-time loop behind a detector: an allocation or a free in the middle of the run
 * stalls every stream of the device, other people's too; (c) code that has to prove "nothing is allocated after
 * start-up".  This entry calls no cudaMalloc, no cudaFree and no library routine that allocates, ever: its only scratch
 * memory, the partial sums (16 bytes per record, `partial records per frame` of ai_get_layout_info), lives in a fixed
 * array of AI_NOALLOC_SCRATCH_BYTES (8 MiB = 524 288 records) that is part of the library's device image -- every GPU
 * that loads the library holds those 8 MiB until the process exits.  ai_setup / ai_build_csr still allocate the matrix:
 * do them at start-up.
 *
 * Arguments, outputs and arithmetic as ai_integrate1d (all DEVICE pointers; AI_NORM_PIXEL; any ai_dtype; the accumulator
 * of ai_set_options).  The layout option is ignored: the frame always takes the block-per-tile kernel pair of
 * AI_LAYOUT_TILED_DIRECT (a memset of the records + 2 launches, plain stream ordering, no overlap between calls) and
 * the profiles are bit-identical to that layout's -- slower than the default path (27.7 against 11.8 us per 2048 x 2048
 * frame in a train of calls on a B200), which is the price of owning no per-context buffers.
 *
 * Limits and rules
 *   - a matrix with more than AI_NOALLOC_SCRATCH_BYTES / 16 partial records is refused with AI_EUNSUPPORTED and a text
 *     that names both sizes; nothing is launched.  For scale: 2048 x 2048 pixels with 1000 bins has 103 132 records, with
 *     3000 bins in q 361 792 (both fit); 4096 x 4096 with 5000 bins has 851 154 (refused).  Bidimensional contexts,
 *     AI_NORM_SPLIT and held corrections (pass the arrays instead) are refused likewise.
 *   - the FIRST call made with a given device current asks the CUDA runtime where the array lives on that device (one
 *     cudaGetSymbolAddress; the runtime may load the library's device code at that moment).  Make that first call during
 *     start-up, outside any stream capture; later calls only enqueue.
 *   - the array is shared by every context, stream and thread of the process on that device and keeps the last call's
 *     records; each call clears what it needs first.  Two calls whose kernels can run on the GPU at the same time (two
 *     streams, two host threads) therefore race on it and both results are garbage: keep all ai_integrate1d_noalloc
 *     calls of a device on one stream, or order them with events.  Calls of the other entry points are not affected.
 * Enqueues on `cuda_stream`; does not synchronise.  Errors: AI_EINVAL, AI_ENOTBUILT, AI_EUNSUPPORTED, AI_ECUDA. */
#define AI_NOALLOC_SCRATCH_BYTES (8u << 20)
int ai_integrate1d_noalloc(ai_ctx *ctx, const void *image, ai_dtype dtype, const float *dark, const float *flat,
                           const float *solidangle, const float *polarization, const uint8_t *mask, float *radial,
                           float *intensity, float *sum_signal, float *count, void *cuda_stream);

/* Integrate one frame into azimuthal x radial bins (a context made by ai_setup2d).  As ai_integrate1d, with
 *   radial       float32[npt_rad] bin centres, may be NULL        azimuthal   float32[npt_azim] bin centres in radians, may be NULL
 *   intensity, sum_signal, count   float32[npt_azim][npt_rad], row-major, required
 * Errors as ai_integrate1d; AI_EINVAL on a 1D context, AI_EUNSUPPORTED with AI_LAYOUT_LUT. */
int ai_integrate2d(ai_ctx *ctx, const void *image, ai_dtype dtype, const float *dark, const float *flat,
                   const float *solidangle, const float *polarization, const uint8_t *mask, float *radial,
                   float *azimuthal, float *intensity, float *sum_signal, float *count, void *cuda_stream);

/* Integrate `nframes` frames that share one matrix and one set of correction arrays (a detector streaming frames,
 * PAPER.md:11); the matrix is read once per group of frames.  All pointers are DEVICE pointers.
 *   frames                     frame f starts at element f * frame_stride_elems (>= height*width)
 *   intensity, sum_signal,
 *   count                      float32[nframes][npt], row-major
 * Enqueues on `cuda_stream`; does not synchronise -- with one exception: the first batch that sends 32 or more 32-bit
 * frames to the frame-lane kernel (1D context, Kahan accumulation, every array on a 16-byte boundary)
 * builds the frame-lane layout of the matrix (one-time, synchronises `cuda_stream`; see ai_get_batch_layout_info), and a
 * larger batch than any before re-allocates scratch (cudaFree synchronises the device).  ai_prepare_batch does both ahead
 * of time: after it, batches of up to its max_frames only enqueue.
 * Which kernels a batch takes is decided by measured cost: the frame-lane kernel takes the leading groups
 * of 64 frames and the remaining frames if they are many enough (plain frames 44 or 60, frames with per-call correction
 * arrays 14, with held corrections 24); the rest goes to the slice-per-lane batch kernel (plain 32-bit frames) or frame
 * by frame through the single-frame kernels (correction arrays, a mask, held corrections, 16-bit pixels: 2 or 3 launches
 * per frame, measured faster than correcting inside a batched kernel).  In the frame-lane kernel and with held
 * corrections a corrected value is (I - dark) times the rounded reciprocal of flat * solidangle * polarization (one
 * rounding more than the division of the other paths).  A frame's profiles do not depend on where it sits among the
 * frames one kernel takes, but they are not bit-identical between the kernels (different fixed summation orders).
 * Errors as ai_integrate1d. */
int ai_integrate1d_batch(ai_ctx *ctx, const void *frames, ai_dtype dtype, int nframes, int64_t frame_stride_elems,
                         const float *dark, const float *flat, const float *solidangle, const float *polarization,
                         const uint8_t *mask, float *intensity, float *sum_signal, float *count, void *cuda_stream);

/* Does now, at start-up, what ai_integrate1d_batch (and ai_integrate1d with correction arrays) would otherwise do inside the
 * first call that needs it: builds the frame-lane layout for batches of up to `max_frames` frames (where it applies) and
 * allocates the library-owned scratch of every kernel a batch of that size can take -- partial sums, the per-call arrays of
 * corrected batches, the corrected frames of the pre-pass, the scaled blobs of a held set (call it after
 * ai_hold_corrections then).  After it, calls with at most `max_frames` frames only enqueue: no cudaMalloc, no cudaFree,
 * no host synchronisation (tests/test_gpu_parity_fl.py checks the device's free memory across such calls).  Optional: without
 * it, or for a larger batch later, the lazy behaviour described above remains.  ai_set_options / ai_set_path_options should
 * be final before the call.  Synchronises `cuda_stream`.  Errors: AI_EINVAL, AI_ENOTBUILT, AI_ENOMEM, AI_ECUDA. */
int ai_prepare_batch(ai_ctx *ctx, int max_frames, void *cuda_stream);

/* End-to-end variant: `image_host` and the three outputs are HOST pointers (pinned memory makes the copies
 * asynchronous); correction arrays and mask stay DEVICE pointers (they are per-detector constants, uploaded once, as in
 * PAPER.md:240-254 where only the image crosses the bus per frame).  Copies the frame host->device, integrates, copies
 * the 3*npt results device->host and synchronises `cuda_stream` before returning.
 * Errors as ai_integrate1d. */
int ai_integrate1d_host(ai_ctx *ctx, const void *image_host, ai_dtype dtype, const float *dark, const float *flat,
                        const float *solidangle, const float *polarization, const uint8_t *mask,
                        float *intensity_host, float *sum_signal_host, float *count_host, void *cuda_stream);

/* A stream of frames that live in HOST memory (the transfer is more than
 * half of the paper's per-frame time).  The frames travel in chunks of up to 8: one upload per chunk into one of two
 * device staging buffers on a library-owned copy stream (the upload of chunk k+1 overlaps the kernels of chunk k), one
 * batched launch per chunk (as ai_integrate1d_batch: the matrix is read once per chunk), three downloads per chunk.
 *   frames_host         HOST pointer (pinned memory for the overlap to happen), frame k at k * frame_stride_elems elements
 *   dark ... mask       DEVICE pointers or NULL, shared by all frames
 *   *_host outputs      HOST pointers, [nframes][npt] row-major
 * Synchronises `cuda_stream` before returning.  Errors as ai_integrate1d. */
int ai_integrate1d_host_frames(ai_ctx *ctx, const void *frames_host, ai_dtype dtype, int nframes,
                               int64_t frame_stride_elems, const float *dark, const float *flat,
                               const float *solidangle, const float *polarization, const uint8_t *mask,
                               float *intensity_host, float *sum_signal_host, float *count_host, void *cuda_stream);

/* Sizes of the TILED execution layout, for byte accounting in benchmarks.  info (HOST pointer)
 * receives 8 values: {tile height in rows, number of tiles, number of (tile, bin) segments, padded number of entries,
 * total bytes of the sliced matrix (all blobs), largest blob in bytes, partial records per frame, (tile + blob) stages
 * the single-frame kernel would use (0 = it does not apply)}.  Errors: AI_EINVAL, AI_ENOTBUILT. */
int ai_get_layout_info(const ai_ctx *ctx, int64_t info[8]);

/* Sizes of the frame-lane layout used by large batches.  info (HOST pointer) receives 8 values:
 * {1 if the layout is built (0: not yet, or it does not apply -- the rest is 0 then), tile height in rows (tiles are 32
 * pixels wide), tiles that hold entries, chunks of tiles (a work item = chunk x group of 64 frames), partial sums per
 * frame (one per chunk and bin of the chunk's window), total bytes of the blobs, largest blob in bytes, frames per
 * group}.  Errors: AI_EINVAL, AI_ENOTBUILT. */
int ai_get_batch_layout_info(const ai_ctx *ctx, int64_t info[8]);

/* Holds a set of correction arrays for the calls that follow (dark current, flat field, solid angle and
 * polarisation are per-experiment constants; in PAPER.md:248-254 only the image crosses the bus per frame).  DEVICE
 * pointers to height*width elements each, any of them NULL; all five NULL drops the held set.  The arrays are read by
 * kernels this call enqueues on `cuda_stream` and not referenced afterwards: they may be freed or changed once the
 * stream has passed this point (changing them has no effect until they are held again).  Every later ai_integrate1d /
 * ai_integrate1d_batch / ai_integrate1d_host* / ai_integrate2d call on this context that passes NO correction array and
 * no mask of its own integrates frames corrected with the held set; a call that passes any array uses its own
 * arguments only, as before.  ai_build_csr drops the held set.
 *
 * What holding buys: sum c (I - dark) / den = sum (c / den) (I - dark), so the division and the mask are
 * folded into a copy of the matrix once -- a pixel that is invalid for every frame (masked, zero or non-finite
 * denominator or reciprocal, non-finite dark current) gets zero coefficients and leaves the counts -- and a frame is
 * corrected inside the integration kernel: AI_LAYOUT_TILED with AI_ACC_F32_KAHAN, one 32-bit frame per call, takes the
 * single-frame kernel with the dark tile loaded beside the frame tile (2 launches instead of 3, one pass over frame,
 * dark current and matrix), and corrected frame-lane batches skip their per-call preparation.  Everywhere else the held
 * set acts as a (dark, flat = product of the three, 0 where invalid) pair.  A corrected value is (I - dark) times the
 * rounded reciprocal of the denominator here (one rounding more than the division of the per-call path).
 * Costs 17 bytes per pixel plus a copy of the layout's blobs.  Call it with the context idle or on the stream the
 * integrate calls use (the derived arrays are rewritten in place).
 * Errors: AI_EINVAL, AI_ENOTBUILT, AI_ENOMEM, AI_ECUDA. */
int ai_hold_corrections(ai_ctx *ctx, const float *dark, const float *flat, const float *solidangle,
                        const float *polarization, const uint8_t *mask, void *cuda_stream);

/* Number of kernels the last ai_integrate1d* call launched (for accounting in benchmarks). */
int ai_last_launch_count(const ai_ctx *ctx);

/* Measurement hook.  on = 1: every ai_integrate1d* call records CUDA events on its stream around its dominant
 * kernel (TILED: stage 1, the SpMV; CSR / LUT: the single kernel); ai_profile_last synchronises on the last of those
 * events and returns the device time of that kernel launch in milliseconds through *kernel_ms.
 * on = 2 (TILED layouts): ai_integrate1d* launches ONLY the dominant kernel -- no events, no second stage, the outputs
 * are not written -- so that a benchmark can time a train of back-to-back launches of that kernel with its own events.
 * on = 0: normal operation.
 * Errors: AI_EINVAL (NULL, or nothing recorded yet), AI_ECUDA. */
int ai_profile_enable(ai_ctx *ctx, int on);
int ai_profile_last(ai_ctx *ctx, float *kernel_ms);

/* Release the context, the matrix and all scratch memory.  NULL is allowed. */
void ai_destroy(ai_ctx *ctx);

/* Static description of a status code. */
const char *ai_strerror(int code);
/* Text of the last error on this context ("" if none); valid until the next call on the context. */
const char *ai_last_error(const ai_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* AZINT_H */
