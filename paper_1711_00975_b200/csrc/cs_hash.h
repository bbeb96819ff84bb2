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

/* Table form for cell ids with a small high limb (c1 < 64, i.e. G^3 <= 2^37): tb = (A*c1 + b) mod p is looked up
 * (kernels keep tb[c1][hash] in shared memory), so that only the two c0 products remain:
 *   s = ll + ml*2^32 + mh + lh + tb,  same bounds as above with tb < 2^61 in the place of b. */
CS_HD uint64_t affine_partial_tb(const HashCoef& k, uint32_t c0, uint64_t tb) {
    const uint64_t lo = mad_wide_u32(k.al, c0, 0);
    const uint64_t m = mad_wide_u32(k.ah, c0, 0);
    const uint32_t mh = (uint32_t)(m >> 29);
    const uint32_t ml = (uint32_t)m & 0x1FFFFFFFu;
    const uint32_t lo_h = (uint32_t)(lo >> 32);
    const uint32_t hi = (lo_h & 0x1FFFFFFFu) + ml + (uint32_t)(tb >> 32);
    return (((uint64_t)hi << 32) | (uint32_t)lo) + (uint64_t)mh + (uint64_t)(lo_h >> 29) + (uint64_t)(uint32_t)tb;
}

/* low 32 bits of the canonical residue from s (see the header comment) */
CS_HD uint32_t fold_low32(uint64_t s) {
    const uint32_t sh = (uint32_t)(s >> 61);
    const uint32_t q = (uint32_t)((s + (uint64_t)(sh + 1u)) >> 61);
    return (uint32_t)s + q;
}

/* The same value as fold_low32(affine_partial_tb(k, c0, tb1 - 1)) for tb1 = tb + 1 (the kernels' tables hold
 * tb + 1).  On the device the 64-bit adds, the shifts by 29 and the 29-bit masks are spelled as multiply-adds
 * (x*8 as a 32x32->64 product yields x >> 29 in its high word; x - (x >> 29)*2^29 is x & (2^29-1)), because the
 * kernels are bound by the integer ALU pipe while the multiply-add pipe idles:
 *   lo = al*c0 + tb1 = lh*2^61 + ll,   s1 = ll + lh + mh + ml*2^32 = s + 1  (< 2^62 + 2^33),
 *   q = floor(s / p) = (s1 + (s1 >> 61)) >> 61   (holds also when s1 is a multiple of 2^61),  low32(r) = low32(s1) + q - 1. */
CS_HD uint32_t affine_low32_tb(const HashCoef& k, uint32_t c0, uint64_t tb1) {
#if defined(__CUDA_ARCH__)
    const uint64_t m = mad_wide_u32(k.ah, c0, 0);
    const uint32_t m_l = (uint32_t)m, m_h = (uint32_t)(m >> 32);
    const uint32_t t_h = (uint32_t)(mad_wide_u32(m_l, 8u, 0) >> 32);            // m_l >> 29
    const uint32_t mh = m_h * 8u + t_h;                                          // m >> 29
    const uint32_t ml = m_l & 0x1FFFFFFFu;
    const uint64_t lo = mad_wide_u32(k.al, c0, tb1);
    const uint32_t lo_l = (uint32_t)lo, lo_h = (uint32_t)(lo >> 32);
    const uint32_t lh = (uint32_t)(mad_wide_u32(lo_h, 8u, 0) >> 32);            // lo >> 61
    const uint32_t hi = (lo_h & 0x1FFFFFFFu) + ml;
    uint64_t s1 = ((uint64_t)hi << 32) | lo_l;
    s1 = mad_wide_u32(mh, 1u, s1);
    s1 = mad_wide_u32(lh, 1u, s1);
    const uint32_t sh = (uint32_t)(mad_wide_u32((uint32_t)(s1 >> 32), 8u, 0) >> 32);
    const uint64_t w = mad_wide_u32(sh, 1u, s1);
    const uint32_t q = (uint32_t)(mad_wide_u32((uint32_t)(w >> 32), 8u, 0) >> 32);
    return (uint32_t)s1 + q - 1u;
#else
    return fold_low32(affine_partial_tb(k, c0, tb1 - 1));
#endif
}

constexpr uint32_t HASH_TB = 64;     /* table entries per hash: c1 = 0 .. 63 */

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
