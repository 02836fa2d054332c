// ising.cu -- a8: the consumer.  Checkerboard Metropolis half-sweeps of the zero-field
// nearest-neighbour 2D Ising ferromagnet on a periodic L x L lattice of int8 +1/-1 spins
// (BASELINE.json config 5; readings R-E1..E8), drawing in-register from
// the per-thread streams: random numbers never touch HBM.
//
// Stream -> site assignment (geometry independent): sites of colour c are numbered
// q = y*(L/2) + xh, x = 2*xh + ((y+c)&1); stream s owns q in [sK, (s+1)K) and spends one
// draw per site in increasing q.  Acceptance: flip iff (r>>8) < T[(h+4)/2] with
// T[i] = min(2^24, ceil(P[i] 2^24)), which is EXACTLY (float)(r>>8)*2^-24 < P[i].
#include "internal.h"
#include "streams.cuh"

namespace rngb200 {

// ------------------------------------------------------------------------------------
// generic half-sweep: any kind, any L (even, >= 4), any K.  One thread per stream.
// ------------------------------------------------------------------------------------
template <int KIND>
__global__ void __launch_bounds__(256) ising_half_sweep_generic_kernel(Gen g, int8_t *__restrict__ sp, uint32_t L,
                                                                       IsingTable tab, uint64_t K, int colour)
{
    const uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.S) return; // xs1024: whole warps leave together
    Stream<KIND> gen;
    gen.load(g, s);
    const uint32_t hw = L >> 1;
    const uint64_t q0 = s * K;
    uint32_t y = (uint32_t)(q0 / hw), xh = (uint32_t)(q0 % hw);
    for (uint64_t k = 0; k < K; k++) {
        const uint32_t x = 2u * xh + ((y + (uint32_t)colour) & 1u);
        const uint32_t xl = x ? x - 1 : L - 1, xr = (x + 1 == L) ? 0 : x + 1;
        const uint32_t yu = y ? y - 1 : L - 1, yd = (y + 1 == L) ? 0 : y + 1;
        int8_t *row = sp + (uint64_t)y * L;
        const int sc = row[x];
        const int nn = row[xl] + row[xr] + sp[(uint64_t)yu * L + x] + sp[(uint64_t)yd * L + x];
        const int h = sc * nn;                  // in {-4,-2,0,2,4}; Delta E = 2h (R-E2)
        const uint32_t r = gen.next();          // a draw is always consumed (R-E3)
        if ((r >> 8) < tab.T[(h + 4) >> 1]) row[x] = (int8_t)(-sc);
        if (++xh == hw) {
            xh = 0;
            y++;
        }
    }
    gen.store(g, s);
}

// spin i = +1 if bit (i & 63) of SM_seed[i >> 6] is set, else -1.  One thread per 16 spins.
__global__ void __launch_bounds__(256) ising_init_random_kernel(int8_t *__restrict__ sp, uint64_t N, uint64_t seed)
{
    const uint64_t v = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; // group of 16 spins
    const uint64_t i0 = v * 16ull;
    if (i0 >= N) return;
    const uint64_t z = splitmix64_at(seed, i0 >> 6);
    const uint32_t bits = (uint32_t)(z >> (i0 & 63ull)) & 0xffffu;
    if (i0 + 16 <= N) {
        uint32_t w[4];
#pragma unroll
        for (int k = 0; k < 4; k++) {
            uint32_t word = 0;
#pragma unroll
            for (int b = 0; b < 4; b++) {
                const uint32_t up = (bits >> (4 * k + b)) & 1u;
                word |= (up ? 0x01u : 0xffu) << (8 * b);
            }
            w[k] = word;
        }
        *reinterpret_cast<uint4 *>(sp + i0) = make_uint4(w[0], w[1], w[2], w[3]); // N % 4 == 0, sp 16-byte aligned
    } else {
        for (uint64_t i = i0; i < N; i++) sp[i] = ((bits >> (i - i0)) & 1u) ? 1 : -1;
    }
}

// E = - sum over bonds, each bond once (right and down neighbour of every site)
__global__ void __launch_bounds__(256) ising_energy_kernel(const int8_t *__restrict__ sp, uint32_t L,
                                                          unsigned long long *__restrict__ out)
{
    const uint64_t N = (uint64_t)L * L;
    long long acc = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t y = (uint32_t)(i / L), x = (uint32_t)(i % L);
        const uint32_t xr = (x + 1 == L) ? 0 : x + 1, yd = (y + 1 == L) ? 0 : y + 1;
        acc -= (int)sp[i] * ((int)sp[(uint64_t)y * L + xr] + (int)sp[(uint64_t)yd * L + x]);
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    __shared__ long long part[8];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        long long t = 0;
        for (int w = 0; w < 8; w++) t += part[w];
        atomicAdd(out, (unsigned long long)t); // two's complement: wraps to the signed sum
    }
}

cudaError_t launch_ising_half_sweep(const rng_handle &h, int8_t *d_spins, uint32_t L, const IsingTable &tab, uint64_t K,
                                    uint64_t draws_done, int colour, cudaStream_t st)
{
    Gen g = h.g;
    g.draws_done = draws_done;
    const uint64_t grid = (g.S + 255) / 256;
    if (grid > 0x7fffffffull) return cudaErrorInvalidConfiguration;
#define GENERIC(KIND) \
    ising_half_sweep_generic_kernel<KIND><<<(unsigned)grid, 256, 0, st>>>(g, d_spins, L, tab, K, colour)
    switch (g.kind) {
    case RNG_LCG64: GENERIC(RNG_LCG64); break;
    case RNG_LCG64_LEAPFROG: GENERIC(RNG_LCG64_LEAPFROG); break;
    case RNG_XORWOW: GENERIC(RNG_XORWOW); break;
    case RNG_XS1024W: GENERIC(RNG_XS1024W); break;
    case RNG_PHILOX4X32_10: GENERIC(RNG_PHILOX4X32_10); break;
    default: return cudaErrorInvalidValue;
    }
#undef GENERIC
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_ising_init_random(int8_t *d_spins, uint32_t L, uint64_t seed, cudaStream_t st)
{
    const uint64_t N = (uint64_t)L * L, groups = (N + 15) / 16;
    const uint64_t grid = (groups + 255) / 256;
    if (grid > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    ising_init_random_kernel<<<(unsigned)grid, 256, 0, st>>>(d_spins, N, seed);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_ising_energy(const int8_t *d_spins, uint32_t L, int64_t *d_out, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(d_out, 0, sizeof(int64_t), st);
    if (e != cudaSuccess) return e;
    const uint64_t N = (uint64_t)L * L;
    uint64_t grid = (N + 255) / 256;
    if (grid > 148ull * 16) grid = 148ull * 16;
    ising_energy_kernel<<<(unsigned)grid, 256, 0, st>>>(d_spins, L, (unsigned long long *)d_out);
    count_launch();
    return cudaGetLastError();
}

} // namespace rngb200
