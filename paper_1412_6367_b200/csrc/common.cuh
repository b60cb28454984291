// Device helpers shared by the per-frame kernels: raw-pixel load + cast ("casted from integer to float"),
// the one-pass pixel corrections, and the three accumulator arithmetics.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ctx.h"

#define AI_FULL_MASK 0xffffffffu

struct Corrections {
    const float *dark, *flat, *solidangle, *polarization;
    const uint8_t *mask;
};

// ---- raw pixel load + cast ------------------------------------------------------------------------------------------
template <int DT> struct RawType;
template <> struct RawType<AI_F32> { using T = float; };
template <> struct RawType<AI_I32> { using T = int32_t; };
template <> struct RawType<AI_U16> { using T = uint16_t; };
template <> struct RawType<AI_I16> { using T = int16_t; };
template <> struct RawType<AI_U32> { using T = uint32_t; };

template <int DT>
__device__ __forceinline__ float load_raw(const void *img, int64_t p)
{
    using T = typename RawType<DT>::T;
    return static_cast<float>(__ldg(reinterpret_cast<const T *>(img) + p));
}

// four consecutive pixels, p a multiple of 4 and the array 16-byte (32-bit types) / 8-byte (16-bit types) aligned
template <int DT>
__device__ __forceinline__ float4 load_raw4(const void *img, int64_t p)
{
    if constexpr (DT == AI_F32) {
        return __ldg(reinterpret_cast<const float4 *>(reinterpret_cast<const float *>(img) + p));
    } else if constexpr (DT == AI_I32) {
        int4 v = __ldg(reinterpret_cast<const int4 *>(reinterpret_cast<const int32_t *>(img) + p));
        return make_float4((float)v.x, (float)v.y, (float)v.z, (float)v.w);
    } else if constexpr (DT == AI_U32) {
        uint4 v = __ldg(reinterpret_cast<const uint4 *>(reinterpret_cast<const uint32_t *>(img) + p));
        return make_float4((float)v.x, (float)v.y, (float)v.z, (float)v.w);
    } else if constexpr (DT == AI_U16) {
        ushort4 v = __ldg(reinterpret_cast<const ushort4 *>(reinterpret_cast<const uint16_t *>(img) + p));
        return make_float4((float)v.x, (float)v.y, (float)v.z, (float)v.w);
    } else {
        short4 v = __ldg(reinterpret_cast<const short4 *>(reinterpret_cast<const int16_t *>(img) + p));
        return make_float4((float)v.x, (float)v.y, (float)v.z, (float)v.w);
    }
}

// ---- corrections: v = (I - dark) / (flat * solidangle * polarization); invalid pixels become NaN ---------------------
__device__ __forceinline__ float quiet_nan() { return __int_as_float(0x7fc00000); }
__device__ __forceinline__ bool finite_f(float x) { return fabsf(x) <= 3.402823466e38f; }   // false for NaN / Inf

// mode 0: the corrected value; 1: its numerator I - dark; 2: its denominator flat * solid * pol (the two sums of the
// split-normalisation estimator, ai_set_normalization) -- the validity test is the same in all three
__device__ __forceinline__ float correct_value(float raw, float dark, float flat, float solid, float pol, bool masked,
                                               bool has_den, int mode = 0)
{
    float num = raw - dark;
    bool ok = !masked && finite_f(num);
    float v = num, den = 1.0f;
    if (has_den) {
        den = flat * solid * pol;
        ok = ok && den != 0.0f && finite_f(den);
        v = num / den;              // IEEE division (no fast-math): parity with the oracle within fp32 rounding
    }
    if (mode == 1) v = num;
    if (mode == 2) v = den;
    return ok ? v : quiet_nan();
}

template <int DT>
__device__ __forceinline__ float corrected_pixel(const void *img, int64_t p, const Corrections &c, int mode = 0)
{
    float raw = load_raw<DT>(img, p);
    float dark = c.dark ? __ldg(c.dark + p) : 0.0f;
    float flat = c.flat ? __ldg(c.flat + p) : 1.0f;
    float sol = c.solidangle ? __ldg(c.solidangle + p) : 1.0f;
    float pol = c.polarization ? __ldg(c.polarization + p) : 1.0f;
    bool masked = c.mask ? (__ldg(c.mask + p) != 0) : false;
    return correct_value(raw, dark, flat, sol, pol, masked, c.flat || c.solidangle || c.polarization, mode);
}

// ---- accumulators -----------------------------------------------------------------------------------------------------
// All three expose: add(float c, float v)  [accumulate the product c*v], merge over the warp, and a (hi, lo) pair whose
// exact sum hi + lo is the accumulated value as far as the mode carries it.
template <int ACC> struct Accum;

// fp32 Kahan ("compensated arithmetics (or [Kahan] summation)"): s carries the sum, c the running error
// (what was added in excess), so the carried value is s - c.
template <> struct Accum<AI_ACC_F32_KAHAN> {
    float s = 0.0f, c = 0.0f;
    __device__ __forceinline__ void add(float coef, float v)
    {
        float y = __fmaf_rn(coef, v, -c);
        float t = __fadd_rn(s, y);
        c = __fsub_rn(__fsub_rn(t, s), y);
        s = t;
    }
    __device__ __forceinline__ void add1(float x)
    {
        float y = __fsub_rn(x, c);
        float t = __fadd_rn(s, y);
        c = __fsub_rn(__fsub_rn(t, s), y);
        s = t;
    }
    // merge another lane's (s, c): error-free two-sum of the two sums, errors collected in c (reading 10)
    __device__ __forceinline__ void merge(float s2, float c2)
    {
        float t = __fadd_rn(s, s2);
        float bb = __fsub_rn(t, s);
        float e = __fadd_rn(__fsub_rn(s, __fsub_rn(t, bb)), __fsub_rn(s2, bb));   // s + s2 == t + e exactly
        c = __fsub_rn(__fadd_rn(c, c2), e);
        s = t;
    }
    __device__ __forceinline__ void absorb(const Accum &o) { merge(o.s, o.c); }
    __device__ __forceinline__ void shfl_down(int d)
    {
        s = __shfl_down_sync(AI_FULL_MASK, s, d);
        c = __shfl_down_sync(AI_FULL_MASK, c, d);
    }
    __device__ __forceinline__ void warp_reduce()
    {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            float s2 = __shfl_xor_sync(AI_FULL_MASK, s, o);
            float c2 = __shfl_xor_sync(AI_FULL_MASK, c, o);
            merge(s2, c2);
        }
    }
    __device__ __forceinline__ double value() const { return (double)s - (double)c; }
    __device__ __forceinline__ float value_f() const { return __fsub_rn(s, c); }
};

template <> struct Accum<AI_ACC_F32_PLAIN> {
    float s = 0.0f;
    __device__ __forceinline__ void add(float coef, float v) { s = __fmaf_rn(coef, v, s); }
    __device__ __forceinline__ void add1(float x) { s = __fadd_rn(s, x); }
    __device__ __forceinline__ void absorb(const Accum &o) { s = __fadd_rn(s, o.s); }
    __device__ __forceinline__ void shfl_down(int d) { s = __shfl_down_sync(AI_FULL_MASK, s, d); }
    __device__ __forceinline__ void warp_reduce()
    {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s = __fadd_rn(s, __shfl_xor_sync(AI_FULL_MASK, s, o));
    }
    __device__ __forceinline__ double value() const { return (double)s; }
    __device__ __forceinline__ float value_f() const { return s; }
};

template <> struct Accum<AI_ACC_F64> {
    double s = 0.0;
    __device__ __forceinline__ void add(float coef, float v) { s = fma((double)coef, (double)v, s); }
    __device__ __forceinline__ void add1(float x) { s += (double)x; }
    __device__ __forceinline__ void absorb(const Accum &o) { s += o.s; }
    __device__ __forceinline__ void shfl_down(int d) { s = __shfl_down_sync(AI_FULL_MASK, s, d); }
    __device__ __forceinline__ void warp_reduce()
    {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(AI_FULL_MASK, s, o);
    }
    __device__ __forceinline__ double value() const { return s; }
    __device__ __forceinline__ float value_f() const { return (float)s; }
};

// final step H5 / O7: intensity = S / C, empty_value where the bin received nothing
__device__ __forceinline__ void write_bin(int b, double S, double C, float empty, float *intensity, float *sum_signal,
                                          float *count)
{
    sum_signal[b] = (float)S;
    count[b] = (float)C;
    intensity[b] = C > 0.0 ? (float)(S / C) : empty;
}
__device__ __forceinline__ void write_bin_f32(int b, float S, float C, float empty, float *intensity,
                                              float *sum_signal, float *count)
{
    sum_signal[b] = S;
    count[b] = C;
    intensity[b] = C > 0.0f ? __fdiv_rn(S, C) : empty;
}
