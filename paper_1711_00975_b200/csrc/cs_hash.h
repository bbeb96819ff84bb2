/*
 * cs_hash.h -- the affine hash x -> (a*x + b) mod (2^61 - 1) (R1) in 32-bit limbs, written once
 * for device and host (the host instance is exported as cs_hash_cell so that the CPU test suite can check
 * this limb arithmetic against big-integer arithmetic without a GPU).  Nothing in oracle/ includes this file;
 * the oracle computes the same function with unsigned __int128 and the % operator.
 *
 * Limbs (p = 2^61 - 1, so 2^61 == 1 mod p), cell id c = c1*2^31 + c0 with c0 < 2^31, c1 < 2^29 (c < 2^60):
 *   a = ah*2^32 + al            al < 2^32, ah < 2^29
 *   A = a*2^31 mod p = Ah*2^32 + Al
 *   b = bh*2^32 + bl            bh < 2^29
 *   a*c + b == lo + m*2^32 + b (mod p)
 *     lo = al*c0 + Al*c1        < 2^63 + 2^61                   (fits 64 bits; two IMAD.WIDE)
 *     m  = ah*c0 + Ah*c1        < 2^60 + 2^58 < 2^61            (two IMAD.WIDE)
 *   m*2^32 = (m >> 29)*2^61 + (m & (2^29-1))*2^32 == mh + ml*2^32      (word-aligned: no 64-bit shifts)
 *   lo     = (lo >> 61)*2^61 + (lo & p)           == lh + ll
 *   s = ll + ml*2^32 + mh + lh + b  < 3*2^61 + 2^32 + 8 < 2^63
 *   with sh = s >> 61 (0..3):  q = floor(s / p) = (s + sh + 1) >> 61,   r = s - q*p = (s + q) mod 2^61
 *   (s = sh*p + (sh + sl) with sl = s mod 2^61, and sh + sl < p + 4 < 2p, so q = sh + [sh + sl >= p])
 * so the low 32 bits of the canonical residue are low32(s) + q: the bucket (w a power of two <= 2^31) and the
 * sign bit need nothing else.
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

/* s of the header comment; BIG = false when c < 2^31 (c1 == 0). */
template <bool BIG>
CS_HD uint64_t affine_partial(const HashCoef& k, uint32_t c0, uint32_t c1) {
    uint64_t lo = mad_wide_u32(k.al, c0, 0);
    uint64_t m = mad_wide_u32(k.ah, c0, 0);
    if (BIG) {
        lo = mad_wide_u32(k.Al, c1, lo);
        m = mad_wide_u32(k.Ah, c1, m);
    }
    const uint32_t mh = (uint32_t)(m >> 29);
    const uint32_t ml = (uint32_t)m & 0x1FFFFFFFu;
    const uint32_t lo_h = (uint32_t)(lo >> 32);
    const uint32_t hi = (lo_h & 0x1FFFFFFFu) + ml + k.bh;          // < 3 * 2^29: b rides in free 3-input adder slots
    return (((uint64_t)hi << 32) | (uint32_t)lo) + (uint64_t)mh + (uint64_t)(lo_h >> 29) + (uint64_t)k.bl;
}

/* low 32 bits of the canonical residue (a*c + b) mod p */
template <bool BIG>
CS_HD uint32_t affine_low32(const HashCoef& k, uint32_t c0, uint32_t c1) {
    const uint64_t s = affine_partial<BIG>(k, c0, c1);
    const uint32_t sh = (uint32_t)(s >> 61);
    const uint32_t q = (uint32_t)((s + (uint64_t)(sh + 1u)) >> 61);
    return (uint32_t)s + q;
}

/* the canonical residue itself (needed when w is not a power of two) */
template <bool BIG>
CS_HD uint64_t affine_mod_p(const HashCoef& k, uint32_t c0, uint32_t c1) {
    const uint64_t s = affine_partial<BIG>(k, c0, c1);
    const uint32_t sh = (uint32_t)(s >> 61);
    const uint64_t q = (s + (uint64_t)(sh + 1u)) >> 61;
    return (s + q) & P61;
}

CS_HD uint64_t coef_a(const HashCoef& k) { return ((uint64_t)k.ah << 32) | k.al; }
CS_HD uint64_t coef_b(const HashCoef& k) { return ((uint64_t)k.bh << 32) | k.bl; }

}  // namespace cs
#endif
