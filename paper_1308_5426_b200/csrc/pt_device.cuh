// pt_device.cuh -- device helpers shared by the libpt kernels (sm_100a).
// Philox-4x32-10 counter-based generator (Salmon et al., SC'11), the 53-bit
// uniform, the 4-bit spin packing and the SWAR nibble match.  Citations are
// PAPER.md:<line>; readings A1-A16 are listed in DESIGN.md.
#pragma once
#include <cstdint>

namespace ptdev {

enum : uint32_t { TAG_INIT = 0u, TAG_SWEEP = 1u, TAG_SWAP = 2u };

struct Philox4 { uint32_t w0, w1, w2, w3; };

// Ten rounds of Philox-4x32; counter (c0..c3), key (k0,k1).
__device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                 uint32_t k0, uint32_t k1) {
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    constexpr uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t h0 = __umulhi(M0, c0), l0 = M0 * c0;
        const uint32_t h1 = __umulhi(M1, c2), l1 = M1 * c2;
        c0 = h1 ^ c1 ^ k0;
        c1 = l1;
        c2 = h0 ^ c3 ^ k1;
        c3 = l0;
        k0 += W0;
        k1 += W1;
    }
    return Philox4{c0, c1, c2, c3};
}

// u in [0,1) with 53 random bits: ((w1>>5) 2^26 + (w2>>6)) 2^-53 (exact in fp64).
__device__ __forceinline__ double uniform53(uint32_t w1, uint32_t w2) {
    const unsigned long long m = ((unsigned long long)(w1 >> 5) << 26) | (unsigned long long)(w2 >> 6);
    return (double)m * (1.0 / 9007199254740992.0);
}

// Integer acceptance threshold (reading A9): Eq. 8 accepts a
// change of energy dE (fixed point 2^-24) iff dE <= 0 or u < exp(-beta dE 2^-24),
// i.e. iff dE < -ln(u) 2^24/beta =: t, i.e. iff dE <= ceil(t) - 1.
// scale = 2^24/beta (+inf for beta = 0: always accept).
__device__ __forceinline__ int accept_threshold(double u, double scale) {
    const double t = -log(u) * scale;
    return (t < 2147483647.0) ? (int)ceil(t) - 1 : 2147483647;
}

// 8 spins per 32-bit word, colour c in 0..15 of site i in nibble i%8 of word i/8.
__device__ __forceinline__ int get_nibble(const uint32_t* words, int i) {
    return (int)((words[i >> 3] >> ((i & 7) << 2)) & 15u);
}

// Bit 4n+3 of the result is set iff nibble n of w equals colour k (exact per
// nibble: no borrow crosses a nibble).
__device__ __forceinline__ uint32_t match_nibbles(uint32_t w, uint32_t k) {
    const uint32_t z = w ^ (k * 0x11111111u);                 // nibble == 0 where equal
    const uint32_t nz = ((z & 0x77777777u) + 0x77777777u) | z; // bit 3 of a nibble set iff nibble != 0
    return ~nz & 0x88888888u;
}

// Wide packing (q > 16): 4 spins per 32-bit word, colour c in 0..255 of site i in byte i%4 of word i/4.  The
// generic kernels take the width (4 or 8 bits per spin) at run time; the direct kernels are 4-bit only.
__device__ __forceinline__ int get_colour(const uint32_t* words, int i, int bits) {
    return bits == 4 ? get_nibble(words, i) : (int)((words[i >> 2] >> ((i & 3) << 3)) & 255u);
}

// Top bit of every field of w (nibble or byte) that equals colour k; the n-th site of the word answers at bit
// bits*(n+1)-1, so site = bit / bits.
__device__ __forceinline__ uint32_t match_colours(uint32_t w, uint32_t k, int bits) {
    if (bits == 4) return match_nibbles(w, k);
    const uint32_t z = w ^ (k * 0x01010101u);
    const uint32_t nz = ((z & 0x7f7f7f7fu) + 0x7f7f7f7fu) | z;
    return ~nz & 0x80808080u;
}

// Adds x*x to the 128-bit accumulator (lo, hi).
__device__ __forceinline__ void add_square_128(unsigned long long& lo, long long& hi, long long x) {
    const unsigned long long ax = (unsigned long long)(x < 0 ? -x : x);
    const unsigned long long plo = ax * ax;
    const unsigned long long phi = __umul64hi(ax, ax);
    const unsigned long long nlo = lo + plo;
    hi = (long long)((unsigned long long)hi + phi + (nlo < lo ? 1ull : 0ull));
    lo = nlo;
}

// Adds x^4 to the 256-bit accumulator a[0..3] (little-endian limbs): x^2 = hi 2^64 + lo, x^4 = lo^2 + 2 lo hi 2^64
// + hi^2 2^128, schoolbook in base 2^64.
__device__ __forceinline__ void add_fourth_256(unsigned long long a[4], long long x) {
    const unsigned long long ax = (unsigned long long)(x < 0 ? -x : x);
    const unsigned long long lo = ax * ax, hi = __umul64hi(ax, ax);
    const unsigned long long ll_lo = lo * lo, ll_hi = __umul64hi(lo, lo);
    const unsigned long long lh_lo = lo * hi, lh_hi = __umul64hi(lo, hi);
    const unsigned long long hh_lo = hi * hi, hh_hi = __umul64hi(hi, hi);
    unsigned long long add[4];
    add[0] = ll_lo;
    // limb 1 = ll_hi + 2 lh_lo (three 64-bit terms: carry in 0..2)
    unsigned long long s1 = ll_hi + lh_lo;
    unsigned long long c1 = s1 < ll_hi ? 1ull : 0ull;
    unsigned long long s1b = s1 + lh_lo;
    c1 += s1b < s1 ? 1ull : 0ull;
    add[1] = s1b;
    // limb 2 = c1 + 2 lh_hi + hh_lo
    unsigned long long s2 = c1 + lh_hi;
    unsigned long long c2 = s2 < lh_hi ? 1ull : 0ull;
    unsigned long long s2b = s2 + lh_hi;
    c2 += s2b < s2 ? 1ull : 0ull;
    unsigned long long s2c = s2b + hh_lo;
    c2 += s2c < s2b ? 1ull : 0ull;
    add[2] = s2c;
    add[3] = c2 + hh_hi;
    unsigned long long carry = 0ull;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const unsigned long long t = a[k] + carry;
        const unsigned long long c0 = t < carry ? 1ull : 0ull;
        const unsigned long long u = t + add[k];
        carry = c0 + (u < t ? 1ull : 0ull);
        a[k] = u;
    }
}

}  // namespace ptdev
