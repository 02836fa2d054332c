// draw.cu -- in-register draw mode: every stream draws n numbers
// that never leave the register file and reduces them to {XOR, SUM mod 2^32}.  This is the
// regime of the paper's peak numbers ("compute-bound"): the only memory
// traffic is one state load and one state store per stream plus 8 bytes out.
#include <type_traits>

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
    if constexpr (KIND == RNG_LCG64_BOTH) {
        // both words of every state: finish a half-used state, then whole states (one
        // multiply-add per TWO draws, no per-draw parity test), then at most one leading high word
        uint64_t left = n;
        if (left && gen.half) {
            accumulate(gen.next());
            left--;
        }
        uint64_t pairs = left >> 1;
        uint64_t y = gen.x;
        while (pairs) {
            const uint32_t t32 = pairs > 0x40000000ull ? 0x40000000u : (uint32_t)pairs;
            pairs -= t32;
#pragma unroll 8
            for (uint32_t t = 0; t < t32; t++) {
                accumulate((uint32_t)(y >> 32));
                accumulate((uint32_t)y);
                y = kLcgA * y + kLcgC;
            }
        }
        gen.x = y;
        if (left & 1ull) accumulate(gen.next());
        gen.store(g, s);
        out[s] = make_uint2(x, sum);
        return;
    }
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
    // whole blocks.  The counter is (lo32(b), hi32(b), 0, 0) (R-C2) and b advances by one: round 1's
    // only non-zero product M0 * lo32(b) grows by M0 per block (a 64-bit add instead of a multiply) and
    // round 2's first product M0 * (hi32(b) ^ k0) is constant while hi32(b) is (see philox_group_fast in
    // fill.cu); both are re-derived whenever lo32(b) wraps.  2R - 2 multiplies per block instead of 2R.
    if (j + 4 <= end) {
        uint64_t b = j >> 2;
        const uint64_t b_end = end >> 2; // first block that is not whole
        uint32_t rk0[R], rk1[R];
#pragma unroll
        for (int r = 0; r < R; r++) rk0[r] = k0 + (uint32_t)r * kPhW0, rk1[r] = k1 + (uint32_t)r * kPhW1;
        while (b < b_end) {
            const uint32_t bhi = (uint32_t)(b >> 32);
            uint64_t seg = (((uint64_t)bhi + 1ull) << 32) - b; // blocks left with this high word
            if (seg > b_end - b) seg = b_end - b;
            uint64_t p0 = (uint64_t)kPhM0 * (uint32_t)b;
            const uint64_t q = (uint64_t)kPhM0 * (bhi ^ rk0[0]);
            b += seg;
            // U blocks interleaved per trip: the ten rounds of one block are a dependent chain
            constexpr int U = 2;
            auto blocks = [&](auto nblk) {
                constexpr int NB = decltype(nblk)::value;
                uint32_t c0[NB], c1[NB], c2[NB], c3[NB];
#pragma unroll
                for (int u = 0; u < NB; u++) {
                    const uint64_t pu = p0 + (uint64_t)u * (uint64_t)kPhM0; // = M0 * lo32(b + u)
                    // after round 1: (c0,c1,c2,c3) = (bhi ^ k0, 0, hi(pu) ^ k1, lo(pu)); round 2:
                    const uint32_t a2 = (uint32_t)(pu >> 32) ^ rk1[0];
                    const uint64_t p1 = (uint64_t)kPhM1 * a2;
                    c0[u] = (uint32_t)(p1 >> 32) ^ rk0[1];
                    c2[u] = (uint32_t)(q >> 32) ^ (uint32_t)pu ^ rk1[1];
                    c1[u] = (uint32_t)p1, c3[u] = (uint32_t)q;
                }
#pragma unroll
                for (int r = 2; r < R; r++) {
#pragma unroll
                    for (int u = 0; u < NB; u++) {
                        const uint64_t m0 = (uint64_t)kPhM0 * c0[u];
                        const uint64_t m1 = (uint64_t)kPhM1 * c2[u];
                        const uint32_t n0 = (uint32_t)(m1 >> 32) ^ c1[u] ^ rk0[r];
                        const uint32_t n2 = (uint32_t)(m0 >> 32) ^ c3[u] ^ rk1[r];
                        c1[u] = (uint32_t)m1, c3[u] = (uint32_t)m0, c0[u] = n0, c2[u] = n2;
                    }
                }
#pragma unroll
                for (int u = 0; u < NB; u++) {
                    x ^= c0[u] ^ c1[u] ^ c2[u] ^ c3[u];
                    sum += c0[u] + c1[u] + c2[u] + c3[u];
                }
                p0 += (uint64_t)NB * (uint64_t)kPhM0;
            };
            while (seg) { // 32-bit trip counts
                const uint32_t s32 = seg > 0x40000000ull ? 0x40000000u : (uint32_t)seg;
                seg -= s32;
#pragma unroll 1
                for (uint32_t t = 0; t < s32 / U; t++) blocks(std::integral_constant<int, U>{});
                if (s32 % U) blocks(std::integral_constant<int, 1>{});
            }
        }
        j = b_end << 2;
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
    case RNG_LCG64_BOTH: draw_reduce_kernel<RNG_LCG64_BOTH><<<(unsigned)grid, 256, 0, st>>>(g, o, n); break;
    case RNG_MWC: draw_reduce_kernel<RNG_MWC><<<(unsigned)grid, 256, 0, st>>>(g, o, n); break;
    case RNG_MWC_MULTI: draw_reduce_kernel<RNG_MWC_MULTI><<<(unsigned)grid, 256, 0, st>>>(g, o, n); break;
    case RNG_LCG32_LEAPFROG: draw_reduce_kernel<RNG_LCG32_LEAPFROG><<<(unsigned)grid, 256, 0, st>>>(g, o, n); break;
    case RNG_LFIB521:
    case RNG_LFIB1279: return launch_lfib_draw(g, d_out, n, st); // CTA = instance (lfib.cu)
    default: return cudaErrorInvalidValue;
    }
    count_launch();
    return cudaGetLastError();
}

} // namespace rngb200
