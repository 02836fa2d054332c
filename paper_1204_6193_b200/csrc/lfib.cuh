// lfib.cuh -- the paper's second state-sharing generator: additive lagged Fibonacci on floats,
//     u_n = u_{n-r} + u_{n-s} (mod 1)                     (eq.(5))
// with (r,s) = (521,353) and (1279,861), "the ring buffer ... shared among the
// threads of a block".  Readings R-G1..G3: single precision, seeds
// are 23-bit fractions so every sum is exact; an instance serves the T = 256 threads of a CTA
// (T <= s, so the T numbers of a batch only need older ones) and deals its numbers round-robin:
// thread t's draw j is v_{jT+t}.  The ring lives in shared memory (RB = 1024 / 2048 words >= r + T,
// so a batch never overwrites what the same batch still reads); ONE block barrier per draw.
// Requirements on a kernel that uses Stream<RNG_LFIB*>: blockDim.x == 256, thread <-> stream
// s = blockIdx.x*256 + threadIdx.x, and every thread of the CTA calls load / next / store the same
// number of times (they contain __syncthreads()).
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include "internal.h"

namespace rngb200 {

constexpr int LFIB_T = 256;
__host__ __device__ constexpr int lfib_r(int kind) { return kind == RNG_LFIB1279 ? 1279 : 521; }
__host__ __device__ constexpr int lfib_s(int kind) { return kind == RNG_LFIB1279 ? 861 : 353; }
__host__ __device__ constexpr int lfib_rb(int kind) { return kind == RNG_LFIB1279 ? 2048 : 1024; }
__host__ __device__ constexpr bool kind_is_lfib(int kind) { return kind == RNG_LFIB521 || kind == RNG_LFIB1279; }

// eq.(5): one single-precision addition mod 1 (exact for 23-bit fractions, R-G1)
__device__ __forceinline__ float lfib_add(float a, float b)
{
    const float t = __fadd_rn(a, b);
    return t >= 1.0f ? __fsub_rn(t, 1.0f) : t;
}
// the draw as a 32-bit integer: (v 2^23) << 9, so that (u >> 8) 2^-24 == v.  v is a 23-bit fraction, so
// 1 + v is exact and its mantissa field IS v 2^23: shifting the bit pattern left by 9 drops sign and
// exponent (one FADD + one shift instead of a float -> int conversion on the slow conversion unit).
__device__ __forceinline__ uint32_t lfib_u32(float v) { return __float_as_uint(__fadd_rn(v, 1.0f)) << 9; }

template <int KIND>
struct LfibStream {
    static constexpr int R = lfib_r(KIND), S = lfib_s(KIND), RB = lfib_rb(KIND);
    float *ring;  // shared, RB words
    uint32_t pos; // ring index of v_{next batch, thread 0}
    float *st;    // this instance's r words in global memory (the last r numbers, oldest first)
    __device__ __forceinline__ static float *ring_storage()
    {
        __shared__ float ring_words[RB];
        return ring_words;
    }
    __device__ __forceinline__ void load(const Gen &g, uint64_t s)
    {
        ring = ring_storage();
        st = (float *)g.state + (s / LFIB_T) * (uint64_t)R;
        for (int i = threadIdx.x; i < R; i += LFIB_T) ring[i] = st[i];
        pos = (uint32_t)R;
        __syncthreads();
    }
    __device__ __forceinline__ float next_float()
    {
        const uint32_t n = pos + threadIdx.x;
        const float v = lfib_add(ring[(n - R) & (RB - 1)], ring[(n - S) & (RB - 1)]);
        ring[n & (RB - 1)] = v;
        pos = (pos + LFIB_T) & (RB - 1);
        __syncthreads(); // the next batch reads what this one wrote (s < 2T for r = 521)
        return v;
    }
    __device__ __forceinline__ uint32_t next() { return lfib_u32(next_float()); }

    // Batched form for kernels that draw in groups of NB = RB/256 batches: after NB batches the ring index is
    // back where it started, so the three ring addresses of batch q of a group are per-thread constants.
    // A group must start with pos == R (true at load() and after any number of whole groups).
    static constexpr int NB = RB / LFIB_T;
    struct Group {
        const float *a[NB], *b[NB];
        float *w[NB];
    };
    __device__ __forceinline__ void group_init(Group &gr) const
    {
#pragma unroll
        for (int q = 0; q < NB; q++) {
            const uint32_t n = (uint32_t)R + threadIdx.x + (uint32_t)(LFIB_T * q);
            gr.a[q] = ring + ((n - R) & (RB - 1));
            gr.b[q] = ring + ((n - S) & (RB - 1));
            gr.w[q] = ring + (n & (RB - 1));
        }
    }
    // batch q of a group (q is a compile-time constant after unrolling)
    __device__ __forceinline__ float group_step(const Group &gr, int q)
    {
        const float v = lfib_add(*gr.a[q], *gr.b[q]);
        *gr.w[q] = v;
        __syncthreads();
        return v;
    }
    __device__ __forceinline__ void store(const Gen &, uint64_t)
    {
        for (int i = threadIdx.x; i < R; i += LFIB_T) st[i] = ring[(pos - R + i) & (RB - 1)];
    }
};

} // namespace rngb200
