// streams.cuh -- "thread s owns stream s" generator objects: state in registers, loaded
// from / stored to the handle's interleaved device state with coalesced accesses
// (PAPER.md:19 requirement (b), :58).
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include "internal.h"
#include "lfib.cuh"

namespace rngb200 {

template <int KIND>
struct Stream;

// ---- LCG64 and its leapfrog sub-streams: x, and the handle's step map (pow2[0]) ----
struct StreamLcg {
    uint64_t x;
    Affine step;
    __device__ __forceinline__ void load(const Gen &g, uint64_t s)
    {
        x = ((const uint64_t *)g.state)[s];
        step = g.lcg->pow2[0];
    }
    __device__ __forceinline__ uint32_t next()
    {
        const uint32_t r = (uint32_t)(x >> 32); // 32 most significant bits
        x = step.A * x + step.C;                // eq.(1) / eq.(2)
        return r;
    }
    __device__ __forceinline__ void store(const Gen &g, uint64_t s) { ((uint64_t *)g.state)[s] = x; }
};
template <>
struct Stream<RNG_LCG64> : StreamLcg {
};
template <>
struct Stream<RNG_LCG64_LEAPFROG> : StreamLcg {
};

// ---- LCG64, both halves of the state as output (R-F2): high word, low word, advance ----
template <>
struct Stream<RNG_LCG64_BOTH> {
    uint64_t x;
    uint32_t half; // 0: the high word of x comes next, 1: the low word
    __device__ __forceinline__ void load(const Gen &g, uint64_t s)
    {
        x = ((const uint64_t *)g.state)[s];
        half = (uint32_t)g.draws_done & 1u; // all streams advance in lockstep
    }
    __device__ __forceinline__ uint32_t next()
    {
        const uint32_t r = half ? (uint32_t)x : (uint32_t)(x >> 32);
        if (half) x = kLcgA * x + kLcgC; // eq.(1)
        half ^= 1u;
        return r;
    }
    __device__ __forceinline__ void store(const Gen &g, uint64_t s) { ((uint64_t *)g.state)[s] = x; }
};

// ---- XORWOW: six words, interleaved w[k*S + s] ----
template <>
struct Stream<RNG_XORWOW> {
    Xorwow st;
    __device__ __forceinline__ void load(const Gen &g, uint64_t s)
    {
        const uint32_t *w = (const uint32_t *)g.state;
        st.x = w[0 * g.S + s];
        st.y = w[1 * g.S + s];
        st.z = w[2 * g.S + s];
        st.w = w[3 * g.S + s];
        st.v = w[4 * g.S + s];
        st.d = w[5 * g.S + s];
    }
    __device__ __forceinline__ uint32_t next() { return st.next(); }
    __device__ __forceinline__ void store(const Gen &g, uint64_t s)
    {
        uint32_t *w = (uint32_t *)g.state;
        w[0 * g.S + s] = st.x;
        w[1 * g.S + s] = st.y;
        w[2 * g.S + s] = st.z;
        w[3 * g.S + s] = st.w;
        w[4 * g.S + s] = st.v;
        w[5 * g.S + s] = st.d;
    }
};

// ---- the 32-bit LCG (eq.(1), :46): the whole word is the draw ----
template <>
struct Stream<RNG_LCG32> {
    uint32_t x;
    __device__ __forceinline__ void load(const Gen &g, uint64_t s) { x = ((const uint32_t *)g.state)[s]; }
    __device__ __forceinline__ uint32_t next()
    {
        const uint32_t r = x;      // u_n = x_n / m, PAPER.md:35 (output, then advance: R-A3)
        x = kLcg32A * x + kLcg32C; // eq.(1), m = 2^32
        return r;
    }
    __device__ __forceinline__ void store(const Gen &g, uint64_t s) { ((uint32_t *)g.state)[s] = x; }
};

// ---- multiply-with-carry: one 32x32+32 -> 64 multiply-add per draw ----
template <>
struct Stream<RNG_MWC> {
    uint32_t x, c;
    __device__ __forceinline__ void load(const Gen &g, uint64_t s)
    {
        const uint64_t v = ((const uint64_t *)g.state)[s];
        x = (uint32_t)v;
        c = (uint32_t)(v >> 32);
    }
    __device__ __forceinline__ uint32_t next()
    {
        const uint32_t r = x;
        const uint64_t t = (uint64_t)kMwcA * x + c; // a x_n + c_n
        x = (uint32_t)t;                            // mod m
        c = (uint32_t)(t >> 32);                    // the carry
        return r;
    }
    __device__ __forceinline__ void store(const Gen &g, uint64_t s) { ((uint64_t *)g.state)[s] = ((uint64_t)c << 32) | x; }
};

// ---- multiply-with-carry with the stream's own multiplier ----
template <>
struct Stream<RNG_MWC_MULTI> {
    uint32_t x, c, a;
    __device__ __forceinline__ void load(const Gen &g, uint64_t s)
    {
        const uint32_t *w = (const uint32_t *)g.state;
        x = w[s];
        c = w[g.S + s];
        a = w[2 * g.S + s];
    }
    __device__ __forceinline__ uint32_t next()
    {
        const uint32_t r = x;
        const uint64_t t = (uint64_t)a * x + c;
        x = (uint32_t)t;
        c = (uint32_t)(t >> 32);
        return r;
    }
    __device__ __forceinline__ void store(const Gen &g, uint64_t s)
    {
        uint32_t *w = (uint32_t *)g.state;
        w[s] = x;
        w[g.S + s] = c; // the multiplier never changes
    }
};

// ---- sub-streams of ONE 32-bit LCG sequence: x <- A x + C with (A, C) = (a, c)^n_total mod 2^32 ----
template <>
struct Stream<RNG_LCG32_LEAPFROG> {
    uint32_t x, A, Cc;
    __device__ __forceinline__ void load(const Gen &g, uint64_t s)
    {
        x = ((const uint32_t *)g.state)[s];
        A = (uint32_t)g.lcg->pow2[0].A; // built by the seeding kernel (eq.(2))
        Cc = (uint32_t)g.lcg->pow2[0].C;
    }
    __device__ __forceinline__ uint32_t next()
    {
        const uint32_t r = x;
        x = A * x + Cc;
        return r;
    }
    __device__ __forceinline__ void store(const Gen &g, uint64_t s) { ((uint32_t *)g.state)[s] = x; }
};

// ---- Philox4x32-R: key = global stream id ^ seed; position = draws_done (R-C2) ----
template <int R>
struct StreamPhilox {
    uint32_t k0, k1;
    uint64_t j; // next draw index
    uint4 buf;
    __device__ __forceinline__ void refill()
    {
        const uint64_t b = j >> 2;
        buf = philox4x32<R>((uint32_t)b, (uint32_t)(b >> 32), 0u, 0u, k0, k1);
    }
    __device__ __forceinline__ void load(const Gen &g, uint64_t s)
    {
        const uint64_t key = (g.first + s) ^ g.seed;
        k0 = (uint32_t)key;
        k1 = (uint32_t)(key >> 32);
        j = g.draws_done;
        if (j & 3ull) refill();
    }
    __device__ __forceinline__ uint32_t next()
    {
        const uint32_t p = (uint32_t)j & 3u;
        if (p == 0u) refill();
        j++;
        return p == 0u ? buf.x : p == 1u ? buf.y : p == 2u ? buf.z : buf.w;
    }
    __device__ __forceinline__ void store(const Gen &, uint64_t) {}
};
template <>
struct Stream<RNG_PHILOX4X32_10> : StreamPhilox<10> {
};
template <>
struct Stream<RNG_PHILOX4X32_7> : StreamPhilox<7> {
};

// ---- float lagged Fibonacci, ring shared by the 256 threads of the CTA (lfib.cuh) ----
template <>
struct Stream<RNG_LFIB521> : LfibStream<RNG_LFIB521> {
};
template <>
struct Stream<RNG_LFIB1279> : LfibStream<RNG_LFIB1279> {
};

// ---- XORShift1024/Weyl, cooperative: lane = word index; whole warps only ----
template <>
struct Stream<RNG_XS1024W> {
    uint32_t s_word;
    uint32_t n; // low 32 bits of the update count (the Weyl term only needs n mod 2^32)
    int lane;
    __device__ __forceinline__ void load(const Gen &g, uint64_t s)
    {
        s_word = ((const uint32_t *)g.state)[s];
        n = (uint32_t)g.draws_done;
        lane = (int)(threadIdx.x & 31u); // blockDim.x % 32 == 0 and (first + s) % 32 == lane
    }
    __device__ __forceinline__ uint32_t next()
    {
        s_word = xs1024_update_coop(s_word, lane);
        n++;
        return xs1024_weyl_term(n) + s_word;
    }
    __device__ __forceinline__ void store(const Gen &g, uint64_t s) { ((uint32_t *)g.state)[s] = s_word; }
};

} // namespace rngb200
