// generators.cuh -- device-side step functions of the four generator families
// (sm_100a).  Product code: shares nothing with oracle/.
//
// Citations: PAPER.md:<line> of /root/reference/PAPER.md; R-<id> = DESIGN.md section 3.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/rng_b200.h"

namespace rngb200 {

// ---------------------------------------------------------------------------------
// splitmix64, random access in k (R-S1; stands in for "seed with another RNG",
// PAPER.md:46, :230).
// ---------------------------------------------------------------------------------
__host__ __device__ __forceinline__ uint64_t splitmix64_at(uint64_t seed, uint64_t k)
{
    uint64_t z = seed + (k + 1ull) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

// ---------------------------------------------------------------------------------
// LCG64 (eq.(1), :46) and its skip-ahead (eq.(2),(3)).
// An affine map x -> A x + C (mod 2^64).
// ---------------------------------------------------------------------------------
struct Affine {
    uint64_t A, C;
};
constexpr uint64_t kLcgA = 2862933555777941757ull;
constexpr uint64_t kLcgC = 1442695040888963407ull;
// multiply-with-carry multiplier (a m - 1 is a safe prime, m = 2^32)
constexpr uint32_t kMwcA = 4294967118u;
// the 32-bit LCG of PAPER.md:46 (a = 1664525, c = 1013904223, m = 2^32; Table 2 "LCG32")
constexpr uint32_t kLcg32A = 1664525u;
constexpr uint32_t kLcg32C = 1013904223u;

__host__ __device__ __forceinline__ uint64_t affine_apply(const Affine &m, uint64_t x) { return m.A * x + m.C; }
// f after g:  f(g(x)) = (A_f A_g) x + (A_f C_g + C_f)
__host__ __device__ __forceinline__ Affine affine_compose(const Affine &f, const Affine &g)
{
    return Affine{f.A * g.A, f.A * g.C + f.C};
}
// base^n by binary exponentiation (square-and-multiply over the bits of n)
__host__ __device__ inline Affine affine_pow(Affine base, uint64_t n)
{
    Affine r{1ull, 0ull};
    while (n) {
        if (n & 1ull) r = affine_compose(base, r);
        base = affine_compose(base, base);
        n >>= 1;
    }
    return r;
}

// ---------------------------------------------------------------------------------
// XORWOW (R-B1).  State words x,y,z,w,v and Weyl counter d; advance, then output.
// ---------------------------------------------------------------------------------
// Pipe steering (sm_100a): LOP3, SHF and IADD3 issue on the alu pipe, IMAD (non-wide) on the
// fma pipe, 64 lanes/clk/SM each.  ptxas decides between IADD3 and IMAD.IADD by its own
// heuristics; where a kernel is bound by one of the two pipes these helpers pin an addition
// to the other one.  `one` / `zero` are the kernel parameters Gen::k_one / Gen::k_zero (1 and 0,
// which neither nvvm nor ptxas can fold), so  a*one + b  must stay an IMAD and the
// three-input  a + b + zero  an IADD3.
__device__ __forceinline__ uint32_t add_on_fma_pipe(uint32_t a, uint32_t b, uint32_t one) { return a * one + b; }
__device__ __forceinline__ uint32_t add_on_alu_pipe(uint32_t a, uint32_t b, uint32_t zero) { return a + b + zero; }

struct Xorwow {
    uint32_t x, y, z, w, v, d;
    __device__ __forceinline__ uint32_t next()
    {
        uint32_t t = x ^ (x >> 2);
        x = y; y = z; z = w; w = v;
        v = (v ^ (v << 4)) ^ (t ^ (t << 1));
        d += 362437u;
        return d + v;
    }
    // same draw with the two additions pinned to the fma pipe (for alu-pipe-bound consumers)
    __device__ __forceinline__ uint32_t next_fma_adds(uint32_t one)
    {
        uint32_t t = x ^ (x >> 2);
        x = y; y = z; z = w; w = v;
        v = (v ^ (v << 4)) ^ (t ^ (t << 1));
        d = add_on_fma_pipe(d, 362437u, one);
        return add_on_fma_pipe(d, v, one);
    }
};

// ---------------------------------------------------------------------------------
// Philox4x32-R (R-C1).  One round: two mulhi/mullo S-boxes with
// multipliers M0 (on c0) and M1 (on c2), xor with the key words and the other
// halves, words permuted; the key is bumped by (W0, W1) after every round.
// ---------------------------------------------------------------------------------
constexpr uint32_t kPhM0 = 0xD2511F53u, kPhM1 = 0xCD9E8D57u;
constexpr uint32_t kPhW0 = 0x9E3779B9u, kPhW1 = 0xBB67AE85u;

// kinds that are Philox4x32-R (counter-based, stateless) and their number of rounds
// (the 7-round variant is the paper's fastest Crush-resistant choice)
__host__ __device__ constexpr bool kind_is_philox(int kind) { return kind == RNG_PHILOX4X32_10 || kind == RNG_PHILOX4X32_7; }
__host__ __device__ constexpr int philox_rounds(int kind) { return kind == RNG_PHILOX4X32_7 ? 7 : 10; }

template <int R = 10>
__device__ __forceinline__ uint4 philox4x32(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                            uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < R; r++) {
        const uint64_t p0 = (uint64_t)kPhM0 * c0; // hi/lo of M0*c0 (one IMAD.WIDE)
        const uint64_t p1 = (uint64_t)kPhM1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += kPhW0;
        k1 += kPhW1;
    }
    return make_uint4(c0, c1, c2, c3);
}

// ---------------------------------------------------------------------------------
// XORShift1024 (eq.(8); (a,b,c) = (329,347,344)),
// cooperative form of Listing 1: lane i of a warp holds word i,
// lane 0 the most significant (R-D1).  329 = 10*32+9, 347 = 10*32+27, 344 = 10*32+24:
//   phase A (<<329): s_i ^= (s_{i+10} << 9)  | (s_{i+11} >> 23)
//   phase B (>>347): s_i ^= (s_{i-10} >> 27) | (s_{i-11} << 5)
//   phase C (<<344): s_i ^= (s_{i+10} << 24) | (s_{i+11} >> 8)
// with s_j = 0 outside [0,31] (the paper's zero padding).  The paper
// exchanges words through a padded `volatile` shared array and implicit warp synchrony;
// here the exchange is a warp shuffle (the paper's footnote 3, anticipates
// it), which also carries the needed synchronisation on sm_70+.  All 32 lanes must call.
// ---------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t xs1024_update_coop(uint32_t s, int lane)
{
    constexpr unsigned FULL = 0xffffffffu;
    uint32_t hi, lo;
    // phase A
    hi = __shfl_down_sync(FULL, s, 10);
    lo = __shfl_down_sync(FULL, s, 11);
    hi = (lane + 10 < 32) ? hi : 0u;
    lo = (lane + 11 < 32) ? lo : 0u;
    s ^= __funnelshift_l(lo, hi, 9);
    // phase B
    lo = __shfl_up_sync(FULL, s, 10);
    hi = __shfl_up_sync(FULL, s, 11);
    lo = (lane >= 10) ? lo : 0u;
    hi = (lane >= 11) ? hi : 0u;
    s ^= __funnelshift_r(lo, hi, 27);
    // phase C
    hi = __shfl_down_sync(FULL, s, 10);
    lo = __shfl_down_sync(FULL, s, 11);
    hi = (lane + 10 < 32) ? hi : 0u;
    lo = (lane + 11 < 32) ? lo : 0u;
    s ^= __funnelshift_l(lo, hi, 24);
    return s;
}
// Weyl term of the n-th update (eq.(9), R-D6): y = n c, y ^ (y >> 16)
__host__ __device__ __forceinline__ uint32_t xs1024_weyl_term(uint64_t n_updates)
{
    const uint32_t y = (uint32_t)n_updates * 362437u;
    return y ^ (y >> 16);
}

// fixed output map (BASELINE.json): (u >> 8) * 2^-24, exact (24-bit integer -> float).
// Evaluated WITHOUT an integer->float conversion: the bit pattern x = u >> 8 < 2^24, read as a float, IS the number
// x 2^-149 -- below 2^23 a denormal (no implicit one), from 2^23 on the first normal binade, whose exponent bit
// contributes exactly the 2^23 at which the denormals stop.  One multiplication by 2^125 (exact: x has 24 bits and
// the product is a normal number) gives x 2^-24.  That is ONE integer-side instruction (the shift) and one FMUL,
// which the fma-lite pipe takes; the kernels here are bound by integer-side issue, where the
// conversion instruction I2FP (alu pipe) or two PRMT cost twice as much.  mul.rn.f32 without .ftz: denormal inputs
// are honoured whatever -ftz the file is compiled with.
__device__ __forceinline__ float u32_to_f32(uint32_t u)
{
    float f;
    asm("mul.rn.f32 %0, %1, 0f7E000000;" : "=f"(f) : "f"(__uint_as_float(u >> 8))); // 0f7E000000 = 2^125
    return f;
}
// The same map in the other exact forms this library went through, kept selectable in the Philox fill (variant
// "cvt") so that the difference stays measurable:
//  1: through the conversion instruction, I2FP(u >> 8) * 2^-24 (I2FP issues on the alu pipe);
//  2: by exponent bias, A = 0x4B00'b3b2 = 2^23 + (u >> 16), B = 0x4B00'00b1 = 2^23 + ((u >> 8) & 255) (one PRMT each),
//     f = fma(B, 2^-24, fma(A, 2^-16, -128.5)): the inner fma is (u>>16) 2^-16 - 1/2, the outer one adds
//     1/2 + b1 2^-24; both results are representable, no rounding occurs;
//  3: "round up" selects the conversion unit's I2F (xu pipe) for u & ~255 (at most 24 significant bits: exact in
//     any rounding mode), scaled by 2^-32.
template <int CVT>
__device__ __forceinline__ float u32_to_f32_form(uint32_t u)
{
    if (CVT == 1) return __uint2float_rn(u >> 8) * 0x1p-24f;
    if (CVT == 2) {
        const float A = __uint_as_float(__byte_perm(u, 0x4B000000u, 0x7432));
        const float B = __uint_as_float(__byte_perm(u, 0x4B000000u, 0x7441));
        return __fmaf_rn(B, 0x1p-24f, __fmaf_rn(A, 0x1p-16f, -128.5f));
    }
    if (CVT == 3) return __uint2float_ru(u & 0xffffff00u) * 0x1p-32f;
    return u32_to_f32(u);
}
// the 32-bit word a fill kernel stores: the draw itself, or the bits of its float image
__device__ __forceinline__ uint32_t out_word(uint32_t u, bool f32)
{
    return f32 ? __float_as_uint(u32_to_f32(u)) : u;
}

} // namespace rngb200
