// Pieces shared by the two TILED stage-1 kernels (integrate_tiled.cu: one block per tile; integrate_pipe.cu: persistent,
// warp-specialised, bulk-copy pipelined): tile staging with fused cast + corrections, the per-lane
// accumulate step, the merge inside a group of lanes (PAPER.md:186-188 compensated sums) and the partial record.
#pragma once
#include "common.cuh"

constexpr int kLanes = 8;            // lanes cooperating on one (tile, bin) segment
constexpr int kStep = kLanes * 4;    // entries consumed per group per 128-bit coefficient load

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

// four matrix entries against the staged tile; TRACK: the tile holds invalid (NaN) pixels, so count is accumulated too
template <int ACC, bool TRACK>
__device__ __forceinline__ void consume4(const float *tile, const float4 &c4, const ushort4 &i4, Accum<ACC> &S,
                                         Accum<ACC> &C)
{
    const float c[4] = {c4.x, c4.y, c4.z, c4.w};
    const float v[4] = {tile[i4.x], tile[i4.y], tile[i4.z], tile[i4.w]};
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        if constexpr (TRACK) {
            bool ok = v[e] == v[e];
            S.add(c[e], ok ? v[e] : 0.0f);
            C.add1(ok ? c[e] : 0.0f);
        } else {
            S.add(c[e], v[e]);
        }
    }
}

// H1 + H2: load tile (ty, tx) of one frame, cast, correct, park in shared memory; NT threads cooperate, `tid` in [0, NT).
// Returns true if this thread met an invalid pixel (masked, zero / non-finite denominator, non-finite value).
template <int DT, int NT>
__device__ __forceinline__ bool stage_tile(float *tile, const void *img, const Corrections &cor, int ty, int tx,
                                           int height, int width, int vec_ok, int tid)
{
    const bool has_den = cor.flat || cor.solidangle || cor.polarization;
    const bool plain = !cor.dark && !has_den && !cor.mask;
    bool bad = false;
    if (vec_ok && plain) {
        // no correction arrays: all of the thread's 128-bit loads are in flight together
        constexpr int kPer = kTilePix / 4 / NT;
        float4 v[kPer];
#pragma unroll
        for (int i = 0; i < kPer; ++i) {
            int q = tid + i * NT;
            int y = ty * kTileH + q / (kTileW / 4), x = tx * kTileW + (q % (kTileW / 4)) * 4;
            v[i] = (y < height && x < width) ? load_raw4<DT>(img, (int64_t)y * width + x) : make_float4(0, 0, 0, 0);
        }
#pragma unroll
        for (int i = 0; i < kPer; ++i) {
            if constexpr (DT == AI_F32) {
                bool b = !finite_f(v[i].x) || !finite_f(v[i].y) || !finite_f(v[i].z) || !finite_f(v[i].w);
                if (b) {
                    v[i].x = finite_f(v[i].x) ? v[i].x : quiet_nan();
                    v[i].y = finite_f(v[i].y) ? v[i].y : quiet_nan();
                    v[i].z = finite_f(v[i].z) ? v[i].z : quiet_nan();
                    v[i].w = finite_f(v[i].w) ? v[i].w : quiet_nan();
                    bad = true;
                }
            }
            reinterpret_cast<float4 *>(tile)[tid + i * NT] = v[i];
        }
    } else if (vec_ok) {
        for (int q = tid; q < kTilePix / 4; q += NT) {
            int ly = q / (kTileW / 4), lx = (q % (kTileW / 4)) * 4;
            int y = ty * kTileH + ly, x = tx * kTileW + lx;
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (y < height && x < width) {
                int64_t p = (int64_t)y * width + x;
                float4 raw = load_raw4<DT>(img, p);
                float4 dk = cor.dark ? __ldg(reinterpret_cast<const float4 *>(cor.dark + p)) : make_float4(0, 0, 0, 0);
                float4 fl = cor.flat ? __ldg(reinterpret_cast<const float4 *>(cor.flat + p)) : make_float4(1, 1, 1, 1);
                float4 sa = cor.solidangle ? __ldg(reinterpret_cast<const float4 *>(cor.solidangle + p))
                                           : make_float4(1, 1, 1, 1);
                float4 po = cor.polarization ? __ldg(reinterpret_cast<const float4 *>(cor.polarization + p))
                                             : make_float4(1, 1, 1, 1);
                uchar4 mk = cor.mask ? __ldg(reinterpret_cast<const uchar4 *>(cor.mask + p)) : make_uchar4(0, 0, 0, 0);
                v.x = correct_value(raw.x, dk.x, fl.x, sa.x, po.x, mk.x != 0, has_den);
                v.y = correct_value(raw.y, dk.y, fl.y, sa.y, po.y, mk.y != 0, has_den);
                v.z = correct_value(raw.z, dk.z, fl.z, sa.z, po.z, mk.z != 0, has_den);
                v.w = correct_value(raw.w, dk.w, fl.w, sa.w, po.w, mk.w != 0, has_den);
                bad = bad || v.x != v.x || v.y != v.y || v.z != v.z || v.w != v.w;
            }
            reinterpret_cast<float4 *>(tile)[q] = v;
        }
    } else {
        for (int k = tid; k < kTilePix; k += NT) {
            int y = ty * kTileH + k / kTileW, x = tx * kTileW + k % kTileW;
            float v = 0.f;
            if (y < height && x < width) {
                v = corrected_pixel<DT>(img, (int64_t)y * width + x, cor);
                bad = bad || v != v;
            }
            tile[k] = v;
        }
    }
    return bad;
}
