/*
 * cs_device.cuh -- device-side arithmetic of the Count-Sketch pass (sm_100a): quantise, sampling hash,
 * affine hashes mod 2^61-1 (cs_hash.h: 32x32->64 multiplies, word-aligned Mersenne folds), median of d.
 * Restates the arithmetic contract of include/cs.h; shares nothing with oracle/.
 */
#ifndef CS_DEVICE_CUH_
#define CS_DEVICE_CUH_

#include "cs_internal.h"

namespace cs {

__device__ __forceinline__ uint64_t mix64(uint64_t z) {
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

/* Sampling (R13): keep iff mix64(K + (i+1)*gamma) < floor(p * 2^64). */
__device__ __forceinline__ bool keep_particle(uint64_t K, uint64_t index, uint64_t Tp) {
    return mix64(K + (index + 1) * GAMMA) < Tp;
}

/* Stage 1 "compute cell ID from XYZ": one binary32 multiply (no FMA), floor, saturate. */
__device__ __forceinline__ uint32_t quantise_axis(float x, float qscale, float top) {
    float f = floorf(__fmul_rn(x, qscale));
    f = fminf(fmaxf(f, 0.0f), top);          // fmaxf(NaN, 0) = 0
    return __float2uint_rz(f);
}

__device__ __forceinline__ uint64_t cell_of(float x, float y, float z, const ScaleParams& sp) {
    uint32_t ix = quantise_axis(x, sp.qscale, sp.top);
    uint32_t iy = quantise_axis(y, sp.qscale, sp.top);
    uint32_t iz = quantise_axis(z, sp.qscale, sp.top);
    return (uint64_t)ix + (uint64_t)sp.G * ((uint64_t)iy + (uint64_t)sp.G * (uint64_t)iz);
}

__device__ __forceinline__ uint64_t mad_wide(uint32_t a, uint32_t b, uint64_t c) {
    return (uint64_t)a * (uint64_t)b + c;     // IMAD.WIDE.U32
}

/* General form for any 64-bit c (used when a caller-supplied cell id is >= 2^60): 128-bit product through
 * __umul64hi, 2^64 == 8 (mod p). */
__device__ __forceinline__ uint64_t affine_mod_p_wide(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t lo = a * c;
    uint64_t hi = __umul64hi(a, c);           // < 2^61
    uint64_t r = (lo & P61) + (lo >> 61) + ((hi << 3) & P61) + (hi >> 58) + b;   // < 3*2^61 + 16
    r = (r & P61) + (r >> 61);
    r = (r + ((r + 1) >> 61)) & P61;
    return r;
}

/* Bucket index and sign of row `rc` for cell c. */
template <bool BIG, bool POW2>
__device__ __forceinline__ void bucket_sign(const RowCoef& rc, uint32_t c0, uint32_t c1, uint64_t w,
                                            uint32_t& bucket, int32_t& sign) {
    if (POW2) bucket = affine_low32<BIG>(rc.h, c0, c1) & (uint32_t)(w - 1);     // w <= 2^31
    else      bucket = (uint32_t)(affine_mod_p<BIG>(rc.h, c0, c1) % w);
    sign = 1 - 2 * (int32_t)(affine_low32<BIG>(rc.s, c0, c1) & 1u);
}

__device__ __forceinline__ int32_t mul_sign(int32_t t, int32_t sign) {
    return sign > 0 ? t : (int32_t)(0u - (uint32_t)t);      // two's-complement wrap (R16)
}

__device__ __forceinline__ void cswap(int32_t& a, int32_t& b) {
    int32_t lo = min(a, b), hi = max(a, b);
    a = lo; b = hi;
}

/* rank-th smallest (0-based) of v[0..D-1] -- rank = (D-1)/2 is the (lower) median, rank = 0 the Count-Min minimum:
 * odd-even transposition network, fully unrolled for D <= 8. */
template <int D>
__device__ __forceinline__ int32_t select_of(int32_t (&v)[D], int rank) {
#pragma unroll
    for (int r = 0; r < D; ++r) {
#pragma unroll
        for (int i = (r & 1); i + 1 < D; i += 2) cswap(v[i], v[i + 1]);
    }
    if (rank == (D - 1) / 2) return v[(D - 1) / 2];
    return v[rank];
}

__device__ __forceinline__ int32_t select_rt(int32_t* v, int d, int rank) {
    for (int i = 1; i < d; ++i) {
        int32_t x = v[i];
        int j = i - 1;
        while (j >= 0 && v[j] > x) { v[j + 1] = v[j]; --j; }
        v[j + 1] = x;
    }
    return v[rank];
}

__host__ __device__ __forceinline__ uint32_t est_to_key(int32_t est) { return 0x7FFFFFFFu - (uint32_t)est; }
__host__ __device__ __forceinline__ int32_t key_to_est(uint32_t ek) { return (int32_t)(0x7FFFFFFFu - ek); }

constexpr int PASS_THREADS = 256;

/* 16-byte streaming load of positions: read once, do not keep in L1, first to leave L2 (the sketch lives there). */
__device__ __forceinline__ float4 ld_stream16(const float4* p) {
    float4 v;
    asm volatile("ld.global.cs.v4.f32 {%0, %1, %2, %3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ float ld_stream4(const float* p) {
    float v;
    asm volatile("ld.global.cs.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}

/* T[j][h] += s without a return value: RED.E.ADD at L2. */
__device__ __forceinline__ void red_add(int32_t* addr, int32_t v) {
    asm volatile("red.global.add.s32 [%0], %1;" :: "l"(addr), "r"(v) : "memory");
}

}  // namespace cs
#endif
