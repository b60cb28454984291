// Pieces shared by the two TILED stage-1 kernels (integrate_tiled.cu: one block per tile; integrate_pipe.cu: persistent,
// warp-specialised, bulk-copy pipelined): the per-lane accumulators (PAPER.md:186-188 compensated sums), the merge
// inside a group of lanes, the partial record, and tile staging with fused cast + corrections.
#pragma once
#include "common.cuh"

constexpr int kLanes = 8;            // lanes cooperating on one (tile, bin) segment
constexpr int kStep = kLanes * 4;    // entries consumed per group per 128-bit coefficient load

// four interleaved accumulators per lane, one per entry of a 128-bit coefficient load: the four compensated
// recurrences of a step are independent, so their latencies overlap
template <int ACC> struct AccumQ {
    Accum<ACC> a, b, c, d;
    __device__ __forceinline__ Accum<ACC> total() const
    {
        Accum<ACC> r = a, q = c;
        r.absorb(b);
        q.absorb(d);
        r.absorb(q);
        return r;
    }
};

template <int ACC>
__device__ __forceinline__ void group_reduce(Accum<ACC> &a)
{
#pragma unroll
    for (int o = kLanes / 2; o > 0; o >>= 1) {
        if constexpr (ACC == AI_ACC_F32_KAHAN) {
            float s2 = __shfl_xor_sync(AI_FULL_MASK, a.s, o);
            float c2 = __shfl_xor_sync(AI_FULL_MASK, a.c, o);
            a.merge(s2, c2);
        } else if constexpr (ACC == AI_ACC_F32_PLAIN) {
            a.s = __fadd_rn(a.s, __shfl_xor_sync(AI_FULL_MASK, a.s, o));
        } else {
            a.s += __shfl_xor_sync(AI_FULL_MASK, a.s, o);
        }
    }
}

// one 16-byte record per segment: fp32 modes (S_hi, S_lo, C_hi, C_lo), fp64 mode (S, C)
template <int ACC>
__device__ __forceinline__ void store_partial(void *partials, int64_t slot, const Accum<ACC> &S, const Accum<ACC> &C,
                                              bool tracked, double csum)
{
    if constexpr (ACC == AI_ACC_F64) {
        reinterpret_cast<double2 *>(partials)[slot] = make_double2(S.s, tracked ? C.s : csum);
    } else if constexpr (ACC == AI_ACC_F32_KAHAN) {
        float c_hi = tracked ? C.s : (float)csum;
        float c_lo = tracked ? -C.c : (float)(csum - (double)c_hi);
        reinterpret_cast<float4 *>(partials)[slot] = make_float4(S.s, -S.c, c_hi, c_lo);
    } else {
        reinterpret_cast<float4 *>(partials)[slot] = make_float4(S.s, 0.0f, tracked ? C.s : (float)csum, 0.0f);
    }
}

// ---- H5: one warp adds the partials of a bin in a fixed order (lane-strided, then a shuffle tree) and writes the
// three outputs (ratio, unweighted histogram, weighted histogram).  `part_f` = the frame's partial
// records; loads bypass L1 (the records were written by other SMs).  Two bins are summed side by side so that their
// loads overlap (the records may have to come from HBM); results do not depend on the pairing.
constexpr int kFinishUnroll = 4;      // 128-bit loads in flight per lane and bin

// one partial record as (signal, count) in the arithmetic the final sum is carried in
template <int ACC> struct FinishT { using T = double; };
template <> struct FinishT<AI_ACC_F32_PLAIN> { using T = float; };

template <int ACC>
__device__ __forceinline__ void finish_load(const void *part_f, int k, bool on, typename FinishT<ACC>::T &s,
                                            typename FinishT<ACC>::T &c)
{
    if constexpr (ACC == AI_ACC_F64) {
        const double2 v = on ? __ldcg(reinterpret_cast<const double2 *>(part_f) + k) : make_double2(0, 0);
        s = v.x; c = v.y;
    } else {
        const float4 v = on ? __ldcg(reinterpret_cast<const float4 *>(part_f) + k) : make_float4(0, 0, 0, 0);
        if constexpr (ACC == AI_ACC_F32_PLAIN) { s = v.x; c = v.z; }
        else { s = (double)v.x + (double)v.y; c = (double)v.z + (double)v.w; }
    }
}

template <int ACC>
__device__ __forceinline__ void finish_write(typename FinishT<ACC>::T S, typename FinishT<ACC>::T C, int lane,
                                             float empty, float *intensity, float *sum_signal, float *count)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        S += __shfl_xor_sync(AI_FULL_MASK, S, d);
        C += __shfl_xor_sync(AI_FULL_MASK, C, d);
    }
    if (lane == 0) {
        if constexpr (ACC == AI_ACC_F32_PLAIN) write_bin_f32(0, S, C, empty, intensity, sum_signal, count);
        else write_bin(0, S, C, empty, intensity, sum_signal, count);
    }
}

// bins b0 (slots [beg0, end0)) and, if two, b1 (slots [beg1, end1)); out_* point at element 0 of the frame's outputs
template <int ACC>
__device__ __forceinline__ void finish_bins(const void *part_f, int b0, int beg0, int end0, bool two, int b1, int beg1,
                                            int end1, int lane, float empty, float *intensity, float *sum_signal,
                                            float *count)
{
    using T = typename FinishT<ACC>::T;
    T S0 = 0, C0 = 0, S1 = 0, C1 = 0;
    if (!two) beg1 = end1 = 0;
    const int n0 = end0 - beg0, n1 = end1 - beg1;
    for (int k0 = lane; k0 < n0 || k0 < n1; k0 += 32 * kFinishUnroll) {
        T s0[kFinishUnroll], c0[kFinishUnroll], s1[kFinishUnroll], c1[kFinishUnroll];
#pragma unroll
        for (int i = 0; i < kFinishUnroll; ++i) {
            finish_load<ACC>(part_f, beg0 + k0 + 32 * i, k0 + 32 * i < n0, s0[i], c0[i]);
            finish_load<ACC>(part_f, beg1 + k0 + 32 * i, k0 + 32 * i < n1, s1[i], c1[i]);
        }
#pragma unroll
        for (int i = 0; i < kFinishUnroll; ++i) { S0 += s0[i]; C0 += c0[i]; S1 += s1[i]; C1 += c1[i]; }
    }
    finish_write<ACC>(S0, C0, lane, empty, intensity + b0, sum_signal + b0, count + b0);
    if (two) finish_write<ACC>(S1, C1, lane, empty, intensity + b1, sum_signal + b1, count + b1);
}

template <int ACC>
__device__ __forceinline__ void finish_bin(const void *part_f, int beg, int end, int lane, float empty, float *intensity,
                                           float *sum_signal, float *count)
{
    finish_bins<ACC>(part_f, 0, beg, end, false, 0, 0, 0, lane, empty, intensity, sum_signal, count);
}

// one THREAD adds the partials of a bin, in slot order: for matrices with many bins of a few partials each (2D)
template <int ACC>
__device__ __forceinline__ void finish_bin_serial(const void *part_f, int beg, int end, float empty, float *intensity,
                                                  float *sum_signal, float *count)
{
    using T = typename FinishT<ACC>::T;
    T S = 0, C = 0;
    for (int k = beg; k < end; ++k) {
        T s, c;
        finish_load<ACC>(part_f, k, true, s, c);
        S += s;
        C += c;
    }
    if constexpr (ACC == AI_ACC_F32_PLAIN) write_bin_f32(0, S, C, empty, intensity, sum_signal, count);
    else write_bin(0, S, C, empty, intensity, sum_signal, count);
}

// value of the pixel whose position in the tile buffer is stored as a byte offset
__device__ __forceinline__ float tile_at(const float *tile, unsigned off)
{
    return *reinterpret_cast<const float *>(reinterpret_cast<const char *>(tile) + off);
}
__device__ __forceinline__ float4 gather4(const float *tile, const ushort4 &x)
{
    return make_float4(tile_at(tile, x.x), tile_at(tile, x.y), tile_at(tile, x.z), tile_at(tile, x.w));
}

// four matrix entries against four gathered pixel values; TRACK: the tile holds invalid (non-finite) pixels, so they
// are skipped and count is accumulated too
template <int ACC, bool TRACK>
__device__ __forceinline__ void accumulate4(const float4 &c4, const float4 &v, AccumQ<ACC> &S, AccumQ<ACC> &C)
{
    if constexpr (TRACK) {
        const bool k0 = finite_f(v.x), k1 = finite_f(v.y), k2 = finite_f(v.z), k3 = finite_f(v.w);
        S.a.add(c4.x, k0 ? v.x : 0.0f);
        S.b.add(c4.y, k1 ? v.y : 0.0f);
        S.c.add(c4.z, k2 ? v.z : 0.0f);
        S.d.add(c4.w, k3 ? v.w : 0.0f);
        C.a.add1(k0 ? c4.x : 0.0f);
        C.b.add1(k1 ? c4.y : 0.0f);
        C.c.add1(k2 ? c4.z : 0.0f);
        C.d.add1(k3 ? c4.w : 0.0f);
    } else {
        S.a.add(c4.x, v.x);
        S.b.add(c4.y, v.y);
        S.c.add(c4.z, v.z);
        S.d.add(c4.w, v.w);
    }
}
template <int ACC, bool TRACK>
__device__ __forceinline__ void consume4(const float *tile, const float4 &c4, const ushort4 &i4, AccumQ<ACC> &S,
                                         AccumQ<ACC> &C)
{
    accumulate4<ACC, TRACK>(c4, gather4(tile, i4), S, C);
}

// ---- H1 + H2: tile staging ---------------------------------------------------------------------------------------------
// Loads tile (ty, tx) of one frame, casts, corrects, and parks it in shared memory at ai_tile_pos; NT threads cooperate
// (`tid` in [0, NT)).  All loads of a batch are issued before the first is used, so a thread keeps BATCH 128-bit loads
// per array in flight; `acquire()` is called once, after the first batch's loads were issued and before the first
// store (the pipelined kernel waits for its shared-memory stage there, so the wait overlaps the load latency).
// Returns true if this thread met an invalid pixel (masked, zero / non-finite denominator, non-finite value).
template <int DT, int NT, int BP, int BC, class Acquire>   // BP / BC: batch size without / with correction arrays
__device__ __forceinline__ bool stage_tile(float *tile, const void *img, const Corrections &cor, int ty, int tx,
                                           int th, int height, int width, int vec_ok, int tid, Acquire acquire)
{
    const bool has_den = cor.flat || cor.solidangle || cor.polarization;
    const bool plain = !cor.dark && !has_den && !cor.mask;
    const int nchunk = th * (kTileW / 4);
    const int y0 = ty * th, x0 = tx * kTileW;
    bool bad = false, acquired = false;
    if (vec_ok && plain) {
        constexpr int B = BP;
        for (int q0 = tid; q0 < nchunk; q0 += NT * B) {
            float4 v[B];
#pragma unroll
            for (int i = 0; i < B; ++i) {
                const int q = q0 + i * NT, y = y0 + (q >> 4), x = x0 + (q & 15) * 4;
                v[i] = (q < nchunk && y < height && x < width) ? load_raw4<DT>(img, (int64_t)y * width + x)
                                                               : make_float4(0, 0, 0, 0);
            }
            if (!acquired) { acquire(); acquired = true; }
#pragma unroll
            for (int i = 0; i < B; ++i) {
                const int q = q0 + i * NT;
                if constexpr (DT == AI_F32) {
                    if (!finite_f(v[i].x) || !finite_f(v[i].y) || !finite_f(v[i].z) || !finite_f(v[i].w)) {
                        v[i].x = finite_f(v[i].x) ? v[i].x : quiet_nan();
                        v[i].y = finite_f(v[i].y) ? v[i].y : quiet_nan();
                        v[i].z = finite_f(v[i].z) ? v[i].z : quiet_nan();
                        v[i].w = finite_f(v[i].w) ? v[i].w : quiet_nan();
                        bad = true;
                    }
                }
                if (q < nchunk) *reinterpret_cast<float4 *>(tile + ai_tile_pos(q >> 4, (q & 15) * 4, th)) = v[i];
            }
        }
    } else if (vec_ok) {
        constexpr int B = BC;
        const float4 one4 = make_float4(1, 1, 1, 1), zero4 = make_float4(0, 0, 0, 0);
        for (int q0 = tid; q0 < nchunk; q0 += NT * B) {
            float4 raw[B], dk[B], fl[B], sa[B], po[B];
            uchar4 mk[B];
            bool in[B];
#pragma unroll
            for (int i = 0; i < B; ++i) {
                const int q = q0 + i * NT, y = y0 + (q >> 4), x = x0 + (q & 15) * 4;
                const int64_t p = (int64_t)y * width + x;
                in[i] = q < nchunk && y < height && x < width;
                raw[i] = in[i] ? load_raw4<DT>(img, p) : zero4;
                dk[i] = (in[i] && cor.dark) ? __ldg(reinterpret_cast<const float4 *>(cor.dark + p)) : zero4;
                fl[i] = (in[i] && cor.flat) ? __ldg(reinterpret_cast<const float4 *>(cor.flat + p)) : one4;
                sa[i] = (in[i] && cor.solidangle) ? __ldg(reinterpret_cast<const float4 *>(cor.solidangle + p)) : one4;
                po[i] = (in[i] && cor.polarization) ? __ldg(reinterpret_cast<const float4 *>(cor.polarization + p)) : one4;
                mk[i] = (in[i] && cor.mask) ? __ldg(reinterpret_cast<const uchar4 *>(cor.mask + p)) : make_uchar4(0, 0, 0, 0);
            }
            if (!acquired) { acquire(); acquired = true; }
#pragma unroll
            for (int i = 0; i < B; ++i) {
                const int q = q0 + i * NT;
                float4 v = zero4;
                if (in[i]) {
                    v.x = correct_value(raw[i].x, dk[i].x, fl[i].x, sa[i].x, po[i].x, mk[i].x != 0, has_den);
                    v.y = correct_value(raw[i].y, dk[i].y, fl[i].y, sa[i].y, po[i].y, mk[i].y != 0, has_den);
                    v.z = correct_value(raw[i].z, dk[i].z, fl[i].z, sa[i].z, po[i].z, mk[i].z != 0, has_den);
                    v.w = correct_value(raw[i].w, dk[i].w, fl[i].w, sa[i].w, po[i].w, mk[i].w != 0, has_den);
                    bad = bad || v.x != v.x || v.y != v.y || v.z != v.z || v.w != v.w;
                }
                if (q < nchunk) *reinterpret_cast<float4 *>(tile + ai_tile_pos(q >> 4, (q & 15) * 4, th)) = v;
            }
        }
    } else {
        acquire();
        for (int k = tid; k < th * kTileW; k += NT) {
            const int ly = k / kTileW, lx = k % kTileW, y = y0 + ly, x = x0 + lx;
            float v = 0.f;
            if (y < height && x < width) {
                v = corrected_pixel<DT>(img, (int64_t)y * width + x, cor);
                bad = bad || v != v;
            }
            tile[ai_tile_pos(ly, lx, th)] = v;
        }
    }
    if (!acquired) acquire();
    return bad;
}
