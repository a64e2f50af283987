// Counter-based RNG and the bit-defined samplers of the GA operators (device side).
//
// PAPER.md:101 generates random chromosomes on the GPU in bulk ("una tantum") and consumes the pool
// when needed; here every draw is a pure function of (seed, index, chromosome, generation, tag), so there
// is no pool and no state (BASELINE.json north_star).
//
//   Philox4x32-10: Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3", SC'11.
//   key = (seed lo, seed hi); counter = (index, chromosome, generation, tag)      [SURVEY 8(c) R4]
//
// The Gaussian sampler uses only IEEE binary32 + - * / sqrt, each rounded once (the __f*_rn intrinsics
// are never contracted into FMAs), so a CPU can reproduce it bit for bit               [SURVEY 8(c) R5]
#pragma once
#include <cstdint>

namespace game {

enum : uint32_t { kTagInit = 0u, kTagSelect = 1u, kTagCross = 2u, kTagMutate = 3u, kTagImmigrant = 4u };

struct PhiloxKey {
    uint32_t k0, k1;
};

__host__ __device__ inline PhiloxKey make_key(uint64_t seed) {
    PhiloxKey k;
    k.k0 = static_cast<uint32_t>(seed);
    k.k1 = static_cast<uint32_t>(seed >> 32);
    return k;
}

// One Philox4x32-10 block: ten rounds of two 32x32->64 multiplies and a word permutation, the key
// bumped by the Weyl constants between rounds.
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, PhiloxKey key) {
    constexpr uint32_t kMul0 = 0xD2511F53u, kMul1 = 0xCD9E8D57u;
    constexpr uint32_t kWeyl0 = 0x9E3779B9u, kWeyl1 = 0xBB67AE85u;
    uint32_t k0 = key.k0, k1 = key.k1;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t lo0 = kMul0 * c0, hi0 = __umulhi(kMul0, c0);
        const uint32_t lo1 = kMul1 * c2, hi1 = __umulhi(kMul1, c2);
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += kWeyl0;
        k1 += kWeyl1;
    }
    return make_uint4(c0, c1, c2, c3);
}

__device__ __forceinline__ uint32_t word_of(const uint4& v, uint32_t i) {
    return i == 0 ? v.x : (i == 1 ? v.y : (i == 2 ? v.z : v.w));
}

// uniform index in [0, n): high word of w * n
__device__ __forceinline__ uint32_t index_below(uint32_t w, uint32_t n) { return __umulhi(w, n); }

// Bernoulli threshold T = floor(p * 2^32), hit iff w < T; p <= 0 never, p >= 1 always (T = 2^32).
__host__ inline uint64_t bernoulli_threshold(double p) {
    if (!(p > 0.0)) return 0ull;
    if (p >= 1.0) return 1ull << 32;
    return static_cast<uint64_t>(p * 4294967296.0);  // truncation == floor for p > 0
}

// gene in [-1, 1): 23 random bits scaled by 2^-23, minus one (both exact)          [SURVEY 8(c) R6]
__device__ __forceinline__ float gene_from_word(uint32_t w) {
    return __fsub_rn(__fmul_rn(__uint2float_rn(w >> 8), 0x1p-23f), 1.0f);
}

// -2 ln(u1), u1 = ((a >> 9) + 1) * 2^-23 in (0, 1]: exponent/mantissa split, f folded into
// (sqrt(1/2), sqrt(2)], ln f = 2 atanh(s), s = (f-1)/(f+1), odd Taylor series to s^9.
__device__ __forceinline__ float neg2_log_u1(uint32_t a) {
    const float u1 = __fmul_rn(__uint2float_rn((a >> 9) + 1u), 0x1p-23f);
    const uint32_t bits = __float_as_uint(u1);
    int e = static_cast<int>(bits >> 23) - 127;
    float f = __uint_as_float((bits & 0x007FFFFFu) | 0x3F800000u);
    if (f > 0x1.6a09e6p+0f) {  // 0x1.6a09e6p+0
        f = __fmul_rn(f, 0.5f);
        e += 1;
    }
    const float s = __fdiv_rn(__fsub_rn(f, 1.0f), __fadd_rn(f, 1.0f));
    const float s2 = __fmul_rn(s, s);
    float p = 0x1.c71c72p-4f;                          // 1/9
    p = __fadd_rn(__fmul_rn(p, s2), 0x1.24924ap-3f);    // 1/7
    p = __fadd_rn(__fmul_rn(p, s2), 0x1.99999ap-3f);    // 1/5
    p = __fadd_rn(__fmul_rn(p, s2), 0x1.555556p-2f);     // 1/3
    p = __fadd_rn(__fmul_rn(p, s2), 1.0f);
    const float e_ln2 = __fmul_rn(__int2float_rn(e), 0x1.62e430p-1f);  // 0x1.62e430p-1
    const float ln_f = __fmul_rn(__fmul_rn(2.0f, s), p);
    return __fmul_rn(-2.0f, __fadd_rn(e_ln2, ln_f));
}

// cos((q + frac) * pi/2), q = b >> 30, frac = ((b >> 6) & 0xFFFFFF) * 2^-24: Taylor series of cos and
// sin on [0, pi/2) in Horner form, quadrant by symmetry.
__device__ __forceinline__ float cos_quarter_turns(uint32_t b) {
    const uint32_t q = b >> 30;
    const float frac = __fmul_rn(__uint2float_rn((b >> 6) & 0xFFFFFFu), 0x1p-24f);
    const float x = __fmul_rn(frac, 0x1.921fb6p+0f);  // 0x1.921fb6p+0
    const float x2 = __fmul_rn(x, x);
    float c = -0x1.93974ap-37f;
    c = __fadd_rn(__fmul_rn(c, x2), 0x1.1eed8ep-29f);
    c = __fsub_rn(__fmul_rn(c, x2), 0x1.27e4fcp-22f);
    c = __fadd_rn(__fmul_rn(c, x2), 0x1.a01a02p-16f);
    c = __fsub_rn(__fmul_rn(c, x2), 0x1.6c16c2p-10f);
    c = __fadd_rn(__fmul_rn(c, x2), 0x1.555556p-5f);
    c = __fsub_rn(__fmul_rn(c, x2), 0.5f);
    c = __fadd_rn(__fmul_rn(c, x2), 1.0f);
    float s = 0x1.612462p-33f;
    s = __fsub_rn(__fmul_rn(s, x2), 0x1.ae6456p-26f);
    s = __fadd_rn(__fmul_rn(s, x2), 0x1.71de3ap-19f);
    s = __fsub_rn(__fmul_rn(s, x2), 0x1.a01a02p-13f);
    s = __fadd_rn(__fmul_rn(s, x2), 0x1.111112p-7f);
    s = __fsub_rn(__fmul_rn(s, x2), 0x1.555556p-3f);
    s = __fadd_rn(__fmul_rn(s, x2), 1.0f);
    s = __fmul_rn(x, s);
    return q == 0 ? c : (q == 1 ? -s : (q == 2 ? -c : s));
}

// Box-Muller: z = sqrt(-2 ln u1) * cos(angle)
__device__ __forceinline__ float gauss_from_words(uint32_t a, uint32_t b) {
    return __fmul_rn(__fsqrt_rn(neg2_log_u1(a)), cos_quarter_turns(b));
}

}  // namespace game
