// Device code shared by the two matrix builders (canonical CSR and tiled layout): the coefficient of PAPER.md:122 and
// the ordered "marching" fill that places entries in ascending pixel order without a sort and without atomics.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/azint.h"

constexpr double kBuildPi = 3.14159265358979323846;

// B1 (map): radial coordinate of a radius r in the requested unit, fp64, every operation
// rounded once.
__device__ __forceinline__ double unit_of_r(double r, double dist, double lambda, int unit)
{
    switch (unit) {
    case AI_R_MM: return __dmul_rn(1e3, r);
    case AI_TTH_RAD: return atan(__ddiv_rn(r, dist));
    case AI_TTH_DEG: return __ddiv_rn(__dmul_rn(atan(__ddiv_rn(r, dist)), 180.0), kBuildPi);
    case AI_Q_NM:
        return __dmul_rn(1e-9, __ddiv_rn(__dmul_rn(4.0 * kBuildPi, sin(__ddiv_rn(atan(__ddiv_rn(r, dist)), 2.0))), lambda));
    default:
        return __dmul_rn(1e-10, __ddiv_rn(__dmul_rn(4.0 * kBuildPi, sin(__ddiv_rn(atan(__ddiv_rn(r, dist)), 2.0))), lambda));
    }
}

// Overlap of pixel [f_lo, f_hi] (bin units) with bin b, over the pixel's width ("proportional to the
// area of the pixel segment that falls into that bin"; PAPER.md:122 outermost bins first, the rest evenly).
// Plain fp64 operations, each rounded once (no FMA contraction).
__device__ __forceinline__ double split_overlap(double f_lo, double f_hi, int b, int npt)
{
    double a = fmax(f_lo, 0.0);
    double z = fmin(f_hi, (double)npt);
    return __dsub_rn(fmin(z, (double)(b + 1)), fmax(a, (double)b));
}
__device__ __forceinline__ double split_coefficient(double f_lo, double f_hi, int b, int npt)
{
    double w = __dsub_rn(f_hi, f_lo);
    if (!(w > 0.0)) return 1.0;     // zero-width pixel: everything in one bin
    return __ddiv_rn(split_overlap(f_lo, f_hi, b, npt), w);
}

// first bin and number of bins with a positive overlap for a pixel with bounds [f_lo, f_hi] in bin units
__device__ __forceinline__ void split_span(double f_lo, double f_hi, int npt, int *first, int *nb)
{
    *first = 0;
    *nb = 0;
    if (!(f_hi > 0.0) || !(f_lo < (double)npt)) return;      // outside the range (also NaN)
    double w = __dsub_rn(f_hi, f_lo);
    if (!(w > 0.0)) {
        int b = (int)floor(f_lo);
        *first = min(max(b, 0), npt - 1);
        *nb = 1;
        return;
    }
    double a = fmax(f_lo, 0.0);
    double z = fmin(f_hi, (double)npt);
    int b0 = (int)floor(a);
    int b1 = min((int)floor(z), npt - 1);
    // only the last bin can have a zero overlap (upper bound exactly on its lower edge)
    if (b1 > b0 && !(split_overlap(f_lo, f_hi, b1, npt) > 0.0)) --b1;
    *first = b0;
    *nb = b1 - b0 + 1;
}

// Ordered fill of one chunk of pixels by one warp.
//
// A chunk is an ordered list of pixels (an image line for the canonical CSR, a tile for the tiled layout).  The warp
// walks it 32 pixels at a time; for every bin b touched by the group, a ballot tells which lanes' pixels cover b, and
// the entry of lane l goes to   base(b) + cursor(b) + popc(ballot & lanes_below_l).   cursor(b) then advances by
// popc(ballot).  Entries of a bin therefore appear in chunk order, i.e. ascending pixel index -- deterministic, stable,
// no atomics, no sort.  Cursors live in global memory (one int per (chunk, bin)) and are only touched by this warp.
//
// Chunk concept:
//   int  npix()                       number of pixel slots in the chunk
//   bool pixel(int k, int64_t *p)     global pixel index of slot k (false: slot outside the image)
//   int  base(int b)                  start of bin b's destination range
//   volatile int *cursor(int b)       running offset of this chunk inside that range
//   int64_t place(int b, int64_t pos) final position of the entry whose position in ascending pixel order is pos
//   void emit(int64_t pos, int k, int64_t p, float coef)
template <class Chunk>
__device__ __forceinline__ void marching_fill(Chunk &ch, const double *__restrict__ fmin_a,
                                              const double *__restrict__ fmax_a, const int *__restrict__ first_a,
                                              const int *__restrict__ nb_a, int npt)
{
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const int n = ch.npix();
    for (int k0 = 0; k0 < n; k0 += 32) {
        int k = k0 + lane;
        int64_t p = 0;
        bool in = k < n && ch.pixel(k, &p);
        int first = 0, nb = 0;
        double f_lo = 0.0, f_hi = 0.0;
        if (in) {
            first = first_a[p];
            nb = nb_a[p];
            f_lo = fmin_a[p];
            f_hi = fmax_a[p];
        }
        int lo = nb > 0 ? first : 0x7fffffff;
        int hi = nb > 0 ? first + nb - 1 : -1;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
            hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        for (int b0 = lo; b0 <= hi; b0 += 32) {
            int myb = b0 + lane;
            volatile int *cur = myb <= hi ? ch.cursor(myb) : nullptr;
            int start = cur ? ch.base(myb) + *cur : 0;
            int mine = 0;
            int span = min(32, hi - b0 + 1);
            for (int bb = 0; bb < span; ++bb) {
                int b = b0 + bb;
                bool covers = nb > 0 && b >= first && b < first + nb;
                unsigned m = __ballot_sync(0xffffffffu, covers);
                int s = __shfl_sync(0xffffffffu, start, bb);
                if (covers)
                    ch.emit(ch.place(b, (int64_t)s + __popc(m & lt)), k, p, (float)split_coefficient(f_lo, f_hi, b, npt));
                if (lane == bb) mine = __popc(m);
            }
            if (cur) *cur = *cur + mine;
            __syncwarp();
        }
    }
}
