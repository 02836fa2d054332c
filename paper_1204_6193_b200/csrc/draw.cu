// draw.cu -- in-register draw mode: every stream draws n numbers
// that never leave the register file and reduces them to {XOR, SUM mod 2^32}.  This is the
// regime of the paper's peak numbers ("compute-bound"): the only memory
// traffic is one state load and one state store per stream plus 8 bytes out.
#include "internal.h"
#include "streams.cuh"

namespace rngb200 {

// UNROLL draws per trip of the main loop.  XORWOW rotates its five words every draw, so a
// multiple of 5 lets the compiler rename registers instead of moving them.
template <int KIND>
__global__ void __launch_bounds__(256) draw_reduce_kernel(Gen g, uint2 *__restrict__ out, uint64_t n)
{
    constexpr int UNROLL = (KIND == RNG_XORWOW) ? 20 : 8;
    const uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.S) return; // xs1024: S % 32 == 0, whole warps leave together
    Stream<KIND> gen;
    gen.load(g, s);
    uint32_t x = 0u, sum = 0u;
    // XORWOW's draw is 4-5 alu-pipe operations (xors, the right shift) and as many additions /
    // left shifts; with the additions pinned to the fma pipe the two pipes carry equal loads.
    const uint32_t one = g.k_one;
    auto draw = [&]() -> uint32_t {
        if constexpr (KIND == RNG_XORWOW) return gen.st.next_fma_adds(one);
        else return gen.next();
    };
    auto accumulate = [&](uint32_t u) {
        x ^= u;
        if constexpr (KIND == RNG_XORWOW) sum = add_on_fma_pipe(sum, u, one);
        else sum += u;
    };
    uint64_t trips = n / UNROLL;
    const uint32_t rest = (uint32_t)(n - trips * UNROLL);
    while (trips) { // 32-bit inner counter: the 64-bit one costs three uniform instructions per trip
        const uint32_t t32 = trips > 0x40000000ull ? 0x40000000u : (uint32_t)trips;
        trips -= t32;
#pragma unroll 1
        for (uint32_t t = 0; t < t32; t++) {
#pragma unroll
            for (int q = 0; q < UNROLL; q++) accumulate(draw());
        }
    }
    for (uint32_t j = 0; j < rest; j++) accumulate(draw());
    gen.store(g, s);
    out[s] = make_uint2(x, sum);
}

// Philox: counter-based, so the n draws of a stream are the words of consecutive blocks;
// whole blocks are reduced four words at a time with the round keys' base hoisted.
template <int R>
__global__ void __launch_bounds__(256) philox_draw_reduce_kernel(Gen g, uint2 *__restrict__ out, uint64_t n)
{
    const uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.S) return;
    const uint64_t key = (g.first + s) ^ g.seed;
    const uint32_t k0 = (uint32_t)key, k1 = (uint32_t)(key >> 32);
    uint64_t j = g.draws_done;
    const uint64_t end = j + n;
    uint32_t x = 0u, sum = 0u;
    // head: words of a partially consumed block
    if ((j & 3ull) && j < end) {
        const uint64_t b = j >> 2;
        const uint4 r = philox4x32<R>((uint32_t)b, (uint32_t)(b >> 32), 0u, 0u, k0, k1);
        const uint32_t w[4] = {r.x, r.y, r.z, r.w};
        for (; (j & 3ull) && j < end; j++) {
            x ^= w[j & 3ull];
            sum += w[j & 3ull];
        }
    }
    for (; j + 4 <= end; j += 4) {
        const uint64_t b = j >> 2;
        const uint4 r = philox4x32<R>((uint32_t)b, (uint32_t)(b >> 32), 0u, 0u, k0, k1);
        x ^= r.x ^ r.y ^ r.z ^ r.w;
        sum += r.x + r.y + r.z + r.w;
    }
    if (j < end) { // tail
        const uint64_t b = j >> 2;
        const uint4 r = philox4x32<R>((uint32_t)b, (uint32_t)(b >> 32), 0u, 0u, k0, k1);
        const uint32_t w[4] = {r.x, r.y, r.z, r.w};
        for (; j < end; j++) {
            x ^= w[j & 3ull];
            sum += w[j & 3ull];
        }
    }
    out[s] = make_uint2(x, sum);
}

cudaError_t launch_draw_reduce(const rng_handle &h, uint32_t *d_out, uint64_t n, cudaStream_t st)
{
    const Gen &g = h.g;
    if (g.kind == RNG_XS1024W && h.var_xs1024 != 64) return launch_xs1024_draw(h, d_out, n, st);
    const uint64_t grid = (g.S + 255) / 256;
    if (grid > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    uint2 *o = (uint2 *)d_out;
    switch (g.kind) {
    case RNG_LCG64: draw_reduce_kernel<RNG_LCG64><<<(unsigned)grid, 256, 0, st>>>(g, o, n); break;
    case RNG_LCG64_LEAPFROG: draw_reduce_kernel<RNG_LCG64_LEAPFROG><<<(unsigned)grid, 256, 0, st>>>(g, o, n); break;
    case RNG_XORWOW: draw_reduce_kernel<RNG_XORWOW><<<(unsigned)grid, 256, 0, st>>>(g, o, n); break;
    case RNG_XS1024W: draw_reduce_kernel<RNG_XS1024W><<<(unsigned)grid, 256, 0, st>>>(g, o, n); break;
    case RNG_PHILOX4X32_10: philox_draw_reduce_kernel<10><<<(unsigned)grid, 256, 0, st>>>(g, o, n); break;
    case RNG_PHILOX4X32_7: philox_draw_reduce_kernel<7><<<(unsigned)grid, 256, 0, st>>>(g, o, n); break;
    case RNG_LCG32: draw_reduce_kernel<RNG_LCG32><<<(unsigned)grid, 256, 0, st>>>(g, o, n); break;
    default: return cudaErrorInvalidValue;
    }
    count_launch();
    return cudaGetLastError();
}

} // namespace rngb200
