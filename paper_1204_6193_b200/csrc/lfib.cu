// lfib.cu -- seeding and fill kernels of the float lagged Fibonacci generators (lfib.cuh;
// PAPER.md:105-124, eq.(5); R-G1..G3).  Draw mode and the Ising consumer use Stream<RNG_LFIB*>
// through the generic kernels of draw.cu / ising.cu (256-thread CTAs = whole instances).
#include "lfib.cuh"

namespace rngb200 {

// R-G3: u_i of instance g = (w >> 9) 2^-23, w = 32-bit word g r + i of the splitmix64 word sequence
// (word 2k = lo32, 2k+1 = hi32 of SM_seed[k]); if no u_i is an odd multiple of 2^-23, u_0 gets that bit.
// One CTA per instance.
template <int KIND>
__global__ void __launch_bounds__(LFIB_T) lfib_seed_kernel(float *__restrict__ state, uint64_t first_inst, uint64_t seed)
{
    constexpr int R = lfib_r(KIND);
    const uint64_t gg = first_inst + blockIdx.x;
    float *st = state + (uint64_t)blockIdx.x * R;
    int odd = 0;
    uint32_t k0 = 0u;
    for (int i = threadIdx.x; i < R; i += LFIB_T) {
        const uint64_t w = gg * (uint64_t)R + (uint64_t)i;
        const uint64_t z = splitmix64_at(seed, w >> 1);
        const uint32_t k = ((w & 1ull) ? (uint32_t)(z >> 32) : (uint32_t)z) >> 9;
        odd |= (int)(k & 1u);
        if (i == 0) k0 = k;
        st[i] = (float)k * 0x1p-23f; // exact: k < 2^23
    }
    const int any_odd = __syncthreads_or(odd);
    if (!any_odd && threadIdx.x == 0) st[0] = (float)(k0 + 1u) * 0x1p-23f;
}

// Fill: the CTA is the instance; a batch yields one number per thread = one draw for each of the
// CTA's 256 rows.  32 batches are staged in a [256 rows][32 draws] tile (row stride 33 words:
// conflict-free both ways), then every warp writes its 32 rows, one whole 128-byte line per store
// instruction.
template <int KIND, bool F32>
__global__ void __launch_bounds__(LFIB_T) lfib_fill_kernel(Gen g, uint32_t *__restrict__ out, uint64_t n)
{
    __shared__ uint32_t tile[LFIB_T * 33];
    const uint64_t s0 = (uint64_t)blockIdx.x * LFIB_T;
    const uint32_t t = threadIdx.x, lane = t & 31u, warp = t >> 5;
    LfibStream<KIND> gen;
    gen.load(g, s0 + t);
    constexpr int NB = LfibStream<KIND>::NB;
    typename LfibStream<KIND>::Group gr;
    gen.group_init(gr);
    for (uint64_t j0 = 0; j0 < n; j0 += 32) {
        const uint32_t kk = (uint32_t)((n - j0 < 32ull) ? (n - j0) : 32ull);
        if (kk == 32u) { // whole groups of NB batches: constant ring addresses (NB divides 32)
#pragma unroll 1
            for (uint32_t q0 = 0; q0 < 32u; q0 += NB) {
#pragma unroll
                for (int q = 0; q < NB; q++) {
                    const float v = gen.group_step(gr, q);
                    tile[t * 33u + q0 + q] = F32 ? __float_as_uint(v) : lfib_u32(v);
                }
            }
        } else {
            for (uint32_t q = 0; q < kk; q++) { // ragged last tile of the call
                const float v = gen.next_float();
                tile[t * 33u + q] = F32 ? __float_as_uint(v) : lfib_u32(v);
            }
        }
        // next_float() ended with a barrier: the tile is complete
        for (uint32_t r = 0; r < 32u; r++) {
            const uint32_t row = warp * 32u + r;
            if (lane < kk) __stcs(out + (s0 + row) * n + j0 + lane, tile[row * 33u + lane]);
        }
        __syncthreads(); // before the tile is overwritten
    }
    gen.store(g, s0 + t);
}

// In-register draw mode: {xor, sum} of the n draws of every stream; whole groups first, then the rest.
template <int KIND>
__global__ void __launch_bounds__(LFIB_T) lfib_draw_kernel(Gen g, uint2 *__restrict__ out, uint64_t n)
{
    const uint64_t s = (uint64_t)blockIdx.x * LFIB_T + threadIdx.x;
    LfibStream<KIND> gen;
    gen.load(g, s);
    constexpr int NB = LfibStream<KIND>::NB;
    typename LfibStream<KIND>::Group gr;
    gen.group_init(gr);
    uint32_t x = 0u, sum = 0u;
    uint64_t groups = n / NB;
    const uint32_t rest = (uint32_t)(n - groups * NB);
    while (groups) {
        const uint32_t g32 = groups > 0x40000000ull ? 0x40000000u : (uint32_t)groups;
        groups -= g32;
#pragma unroll 1
        for (uint32_t i = 0; i < g32; i++) {
#pragma unroll
            for (int q = 0; q < NB; q++) {
                const uint32_t u = lfib_u32(gen.group_step(gr, q));
                x ^= u;
                sum += u;
            }
        }
    }
    for (uint32_t j = 0; j < rest; j++) {
        const uint32_t u = gen.next();
        x ^= u;
        sum += u;
    }
    gen.store(g, s);
    out[s] = make_uint2(x, sum);
}

cudaError_t launch_lfib_draw(const Gen &g, uint32_t *d_out, uint64_t n, cudaStream_t st)
{
    const uint64_t inst = g.S / LFIB_T;
    if (inst > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    if (g.kind == RNG_LFIB1279) lfib_draw_kernel<RNG_LFIB1279><<<(unsigned)inst, LFIB_T, 0, st>>>(g, (uint2 *)d_out, n);
    else lfib_draw_kernel<RNG_LFIB521><<<(unsigned)inst, LFIB_T, 0, st>>>(g, (uint2 *)d_out, n);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_seed_lfib(const Gen &g, cudaStream_t st)
{
    const uint64_t inst = g.S / LFIB_T;
    if (inst > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    if (g.kind == RNG_LFIB1279)
        lfib_seed_kernel<RNG_LFIB1279><<<(unsigned)inst, LFIB_T, 0, st>>>((float *)g.state, g.first / LFIB_T, g.seed);
    else
        lfib_seed_kernel<RNG_LFIB521><<<(unsigned)inst, LFIB_T, 0, st>>>((float *)g.state, g.first / LFIB_T, g.seed);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_lfib_fill(const Gen &g, void *d_out, uint64_t n, bool f32, cudaStream_t st)
{
    const uint64_t inst = g.S / LFIB_T;
    if (inst > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    uint32_t *o = (uint32_t *)d_out;
#define LF(KIND)                                                                        \
    do {                                                                                \
        if (f32) lfib_fill_kernel<KIND, true><<<(unsigned)inst, LFIB_T, 0, st>>>(g, o, n);  \
        else lfib_fill_kernel<KIND, false><<<(unsigned)inst, LFIB_T, 0, st>>>(g, o, n);     \
    } while (0)
    if (g.kind == RNG_LFIB1279) LF(RNG_LFIB1279);
    else LF(RNG_LFIB521);
#undef LF
    count_launch();
    return cudaGetLastError();
}

} // namespace rngb200
