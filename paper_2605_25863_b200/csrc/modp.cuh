// modp.cuh -- device arithmetic in F_p, 2 <= p < 2^31 (run-time p, host-precomputed constants).
//
// The paper makes p a compile-time constant through JIT so that `%` becomes shifts and
// multiplies.  This build is ahead-of-time compiled, so the same
// effect comes from Barrett constants computed once per call on the host.
#pragma once
#include <cstdint>

namespace linac {

struct ModP {
    uint32_t p;        // the modulus
    uint32_t c32;      // 2^32 mod p
    uint64_t m64;      // floor(2^64 / p)   (p >= 2, so it fits)
    uint32_t w[7];     // 2^(8k) mod p, k = 0..6  (limb recombination weights of the tensor path)
    uint32_t ninv;     // -p^-1 mod 2^32 (Montgomery constant; 0 when p is even, i.e. p = 2)
    uint32_t wm[7];    // 2^(8k) * 2^32 mod p: the same weights in Montgomery form
};

#ifdef __CUDACC__
// x mod p for any x < 2^64.  q = floor(x*m64 / 2^64) is floor(x/p) or one less, so one
// conditional subtraction finishes the job; r < 2p < 2^32 so 32-bit arithmetic suffices for it.
__device__ __forceinline__ uint32_t reduce64(uint64_t x, const ModP& f) {
    uint64_t q = __umul64hi(x, f.m64);
    uint32_t r = (uint32_t)x - (uint32_t)q * f.p;
    return r >= f.p ? r - f.p : r;
}

__device__ __forceinline__ uint32_t mulmod(uint32_t a, uint32_t b, const ModP& f) {
    return reduce64((uint64_t)a * b, f);
}

__device__ __forceinline__ uint32_t addmod(uint32_t a, uint32_t b, const ModP& f) {
    uint32_t s = a + b;   // < 2^32 because p < 2^31
    return s >= f.p ? s - f.p : s;
}

__device__ __forceinline__ uint32_t submod(uint32_t a, uint32_t b, const ModP& f) {
    return a >= b ? a - b : a + f.p - b;
}

// a - b*c mod p
__device__ __forceinline__ uint32_t submulmod(uint32_t a, uint32_t b, uint32_t c, const ModP& f) {
    return submod(a, mulmod(b, c, f), f);
}

// Montgomery reduction (R = 2^32, p odd): t * 2^-32 mod p for t < p * 2^32.  Four instructions against
// Barrett's fourteen; used where a constant factor 2^-32 can be absorbed (the fast panel's
// division-free elimination, where it only rescales rows, and the tensor epilogue, whose weights
// carry the compensating 2^32).
__device__ __forceinline__ uint32_t redc(uint64_t t, const ModP& f) {
    const uint32_t m = (uint32_t)t * f.ninv;
    const uint32_t u = (uint32_t)((t + (uint64_t)m * f.p) >> 32);     // t + m*p < 2^64, low word is zero
    return u >= f.p ? u - f.p : u;
}
__device__ __forceinline__ uint32_t mulredc(uint32_t a, uint32_t b, const ModP& f) { return redc((uint64_t)a * b, f); }

// a^-1 = a^(p-2) mod p (Fermat; p an odd prime) by square-and-multiply on Montgomery products: a chain of
// about 45 four-instruction multiplications, several times shorter than extended Euclid's divisions.
__device__ __forceinline__ uint32_t invmod_fermat(uint32_t a, const ModP& f) {
    const uint32_t one = f.c32;                              // 1 in Montgomery form (2^32 mod p)
    uint32_t base = reduce64((uint64_t)a * f.c32, f);        // a in Montgomery form
    uint32_t acc = one;
    for (uint32_t e = f.p - 2; e; e >>= 1) {
        if (e & 1u) acc = mulredc(acc, base, f);
        base = mulredc(base, base, f);
    }
    return redc(acc, f);
}

// Keeps a 64-bit accumulator of products below 2^63 + 2^32 without a full reduction:
// x = hi*2^32 + lo  ==  hi*(2^32 mod p) + lo   (mod p).
__device__ __forceinline__ uint64_t fold64(uint64_t x, const ModP& f) {
    return (x >> 32) * (uint64_t)f.c32 + (uint32_t)x;
}

// a^{-1} mod p by the extended Euclidean algorithm (K7's "rescale the head to 1", PAPER.md:243;
// the paper does not say how the device inverts).  a in [1,p).  All lanes of a warp may call it
// with the same argument (no divergence then).
__device__ __forceinline__ uint32_t invmod(uint32_t a, const ModP& f) {
    uint32_t r0 = f.p, r1 = a;
    int64_t t0 = 0, t1 = 1;
    while (r1 != 0) {
        uint32_t q = r0 / r1;
        uint32_t r2 = r0 - q * r1;
        int64_t t2 = t0 - (int64_t)q * t1;
        r0 = r1; r1 = r2;
        t0 = t1; t1 = t2;
    }
    // |t0| < p throughout (standard bound on Bezout coefficients)
    return t0 < 0 ? (uint32_t)(t0 + (int64_t)f.p) : (uint32_t)t0;
}
#endif  // __CUDACC__

}  // namespace linac
