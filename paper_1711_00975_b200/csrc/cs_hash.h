/*
 * cs_hash.h -- the affine hash x -> (a*x + b) mod (2^61 - 1) (R1) in 32-bit limbs, written once
 * for device and host (the host instance is exported as cs_hash_cell so that the CPU test suite can check
 * this limb arithmetic against big-integer arithmetic without a GPU).  Nothing in oracle/ includes this file;
 * the oracle computes the same function with unsigned __int128 and the % operator.
 *
 * p = 2^61 - 1, so 2^61 == 1 (mod p).  Cell id c = c1*2^31 + c0 with c0 < 2^31, c1 < 2^29 (c < 2^60).
 *   a = ah*2^32 + al            al < 2^32, ah < 2^29
 *   A = a*2^31 mod p = Ah*2^32 + Al                     (so a*c == a*c0 + A*c1 mod p)
 *   b = bh*2^32 + bl            bh < 2^29
 * Chained multiply-adds (IMAD.WIDE.U32: 32 x 32 + 64 -> 64), the second pair riding on the high word of the first:
 *   D = al*c0 + Al*c1 + b       < 2^63 + 2^61 + 2^61 < 2^64
 *   E = ah*c0 + Ah*c1 + (D>>32) < 2^60 + 2^58 + 2^32 < 2^61
 *   x = E*2^32 + low32(D)  ==  a*c + b  (mod p),   x < 2^93
 * One fold: x = xh*2^61 + xl with xh = E >> 29 (< 2^32), xl = (E mod 2^29)*2^32 + low32(D) (< 2^61):
 *   t = xl + xh < 2^61 + 2^32 < 2p,   t == x (mod p)
 * Canonical residue without a compare: u = t + 1, q = u >> 61 (0 or 1; q = 1 exactly when t >= p), r = t - q*p
 *   = (u - 1 + q) mod 2^61.  So low32(r) = low32(u) - 1 + q: the bucket (w a power of two <= 2^31) and the sign bit need
 * nothing else.  8 SASS instructions per hash for one-limb cell ids, 10 for two limbs (the first version of this file
 * folded the two products separately: ~21).
 */
#ifndef CS_HASH_H_
#define CS_HASH_H_

#include <stdint.h>

#if defined(__CUDACC__)
#define CS_HD __host__ __device__ __forceinline__
#else
#define CS_HD inline
#endif

namespace cs {

constexpr uint64_t P61 = (1ULL << 61) - 1;            // Mersenne prime 2^61 - 1

struct HashCoef {
    uint32_t al, ah;   // a
    uint32_t Al, Ah;   // a * 2^31 mod p
    uint32_t bl, bh;   // b
};

/* host: split one (a, b) pair, a in [1, p-1], b in [0, p-1] */
inline HashCoef split_coef(uint64_t a, uint64_t b) {
    HashCoef k;
    k.al = (uint32_t)a;
    k.ah = (uint32_t)(a >> 32);
    /* a = x*2^30 + y (y < 2^30)  =>  a*2^31 = x*2^61 + y*2^31 == x + y*2^31 < 2^31 + 2^61 */
    uint64_t A = (a >> 30) + ((a & 0x3FFFFFFFULL) << 31);
    if (A >= P61) A -= P61;
    k.Al = (uint32_t)A;
    k.Ah = (uint32_t)(A >> 32);
    k.bl = (uint32_t)b;
    k.bh = (uint32_t)(b >> 32);
    return k;
}

CS_HD uint32_t cell_c0(uint64_t c) { return (uint32_t)c & 0x7FFFFFFFu; }
CS_HD uint32_t cell_c1(uint64_t c) { return (uint32_t)(c >> 31); }

/* 32 x 32 + 64 -> 64.  On the device this is spelled as the PTX mad.wide.u32 (one IMAD.WIDE): written as C, NVVM
 * widens the operands to 64 bits and ptxas no longer sees that their high words are zero. */
CS_HD uint64_t mad_wide_u32(uint32_t a, uint32_t b, uint64_t c) {
#if defined(__CUDA_ARCH__)
    uint64_t d;
    asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(d) : "r"(a), "r"(b), "l"(c));
    return d;
#else
    return (uint64_t)a * b + c;
#endif
}

/* u = t + 1 of the header comment for the pair (E, low32(D)) */
CS_HD uint64_t fold_u(uint64_t E, uint32_t Dl) {
    const uint32_t xh = (uint32_t)(E >> 29);
    const uint64_t xl = ((uint64_t)((uint32_t)E & 0x1FFFFFFFu) << 32) | Dl;
    return xl + (uint64_t)xh + 1u;
}

/* u for cell (c0, c1); BIG = false when c < 2^31 (c1 == 0). */
template <bool BIG>
CS_HD uint64_t affine_u(const HashCoef& k, uint32_t c0, uint32_t c1) {
    uint64_t D = mad_wide_u32(k.al, c0, ((uint64_t)k.bh << 32) | k.bl);
    if (BIG) D = mad_wide_u32(k.Al, c1, D);
    uint64_t E = mad_wide_u32(k.ah, c0, (uint64_t)(uint32_t)(D >> 32));
    if (BIG) E = mad_wide_u32(k.Ah, c1, E);
    return fold_u(E, (uint32_t)D);
}

/* low 32 bits of the canonical residue (a*c + b) mod p */
template <bool BIG>
CS_HD uint32_t affine_low32(const HashCoef& k, uint32_t c0, uint32_t c1) {
    const uint64_t u = affine_u<BIG>(k, c0, c1);
    return (uint32_t)u + (uint32_t)(u >> 61) - 1u;
}

/* the canonical residue itself (needed when w is not a power of two) */
template <bool BIG>
CS_HD uint64_t affine_mod_p(const HashCoef& k, uint32_t c0, uint32_t c1) {
    const uint64_t u = affine_u<BIG>(k, c0, c1);
    return (u - 1u + (u >> 61)) & P61;
}

/* Table form for cell ids with a small high limb (c1 < HASH_TB): tb = (A*c1 + b) mod p is looked up (a kernel would keep
 * tb[c1][hash] in shared memory), so that only the two c0 products remain: D = al*c0 + tb (< 2^63 + 2^61),
 * E = ah*c0 + (D >> 32).  Kept as a checked alternative (cs_hash_cell big = 2); the kernels use the table-free forms:
 * two more multiply-adds cost less than a 16-byte shared-memory load at a random address per row. */
constexpr uint32_t HASH_TB = 64;     /* table entries per hash: c1 = 0 .. 63 */
CS_HD uint32_t affine_low32_tb(const HashCoef& k, uint32_t c0, uint64_t tb) {
    const uint64_t D = mad_wide_u32(k.al, c0, tb);
    const uint64_t E = mad_wide_u32(k.ah, c0, (uint64_t)(uint32_t)(D >> 32));
    const uint64_t u = fold_u(E, (uint32_t)D);
    return (uint32_t)u + (uint32_t)(u >> 61) - 1u;
}
CS_HD uint64_t affine_mod_p_tb(const HashCoef& k, uint32_t c0, uint64_t tb) {
    const uint64_t D = mad_wide_u32(k.al, c0, tb);
    const uint64_t E = mad_wide_u32(k.ah, c0, (uint64_t)(uint32_t)(D >> 32));
    const uint64_t u = fold_u(E, (uint32_t)D);
    return (u - 1u + (u >> 61)) & P61;
}

CS_HD uint64_t coef_a(const HashCoef& k) { return ((uint64_t)k.ah << 32) | k.al; }
CS_HD uint64_t coef_b(const HashCoef& k) { return ((uint64_t)k.bh << 32) | k.bl; }

}  // namespace cs
#endif
