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

// Fill: the CTA is the instance; a batch yields one number per thread = one draw for each of the CTA's 256 rows, and a
// row becomes a whole 128-byte line after 32 batches.  Round 2: the ring IS the staging tile.  It holds 32 batches
// (8192 numbers, logical index m at word (m >> 8) * 257 + (m & 255): batch-slot stride 257 makes both the
// generation accesses -- consecutive threads, consecutive words -- and the transposed write-out -- one thread reads
// four consecutive draws of a row, i.e. four consecutive slots -- conflict-free), so a draw costs 2 LDS + 1 STS when it
// is generated and 1 LDS when it is written out, instead of 3 LDS + 2 STS with a separate tile, and the write-out
// is one 128-bit streaming store per four draws.  The state (the last r numbers) is loaded into the last slots, so
// that batch 0 of the first tile finds its lagged numbers where every later tile finds them.
// A lag Lg = 256 k + rem puts number n - Lg of thread t (n = 256 q + t) into slot q - k - w at offset
// t - rem + 256 w, w = (t < rem): two base pointers per lag make every address of the unrolled tile an immediate
// offset.  A barrier is needed only every floor(s / 256) batches (1 for r = 521, 3 for r = 1279): later batches
// read nothing younger.
template <int KIND, int SLOTS_>
struct LfibTile {
    static constexpr int R = lfib_r(KIND), S = lfib_s(KIND);
    static constexpr int SLOTS = SLOTS_, STRIDE = LFIB_T + 1, WORDS = SLOTS * STRIDE;
    static constexpr int PER_BAR = S / LFIB_T; // batches between barriers
    __device__ __forceinline__ static uint32_t addr(uint32_t m) { return (m >> 8) * STRIDE + (m & 255u); } // m < 256 SLOTS
    // pointers for lag LG of thread t: p = slot-relative base, pk = the address for batch q == k
    template <int LG>
    struct Lag {
        static constexpr int k = LG / LFIB_T, rem = LG % LFIB_T;
        const float *p, *pk;
        __device__ __forceinline__ void init(const float *ring, uint32_t t)
        {
            const int w = t < (uint32_t)rem ? 1 : 0;
            p = ring + ((int)t - rem + LFIB_T * w) - w * STRIDE;
            pk = p + w * (SLOTS * STRIDE);
        }
        // number n - LG for batch q (compile-time q after unrolling)
        __device__ __forceinline__ float at(int q) const
        {
            return q > k ? p[(q - k) * STRIDE] : q == k ? *pk : p[(q - k + SLOTS) * STRIDE];
        }
        // the same for a run-time q (ragged last tile)
        __device__ __forceinline__ float at_dyn(const float *ring, uint32_t t, uint32_t q) const
        {
            const uint32_t m = (LFIB_T * q + t - (uint32_t)LG) & (uint32_t)(SLOTS * LFIB_T - 1);
            return ring[addr(m)];
        }
    };
};

// SLOTS = batches per tile = draws per row and visit: 32 (one 128-byte line) or 64 (256 contiguous bytes per row,
// the store pattern that lifts the B200's write ceiling from 5.6 to 6.6 TB/s for 4 KiB rows).
template <int KIND, bool F32, int SLOTS>
__global__ void __launch_bounds__(LFIB_T) lfib_fill_kernel(Gen g, uint32_t *__restrict__ out, uint64_t n)
{
    using TL = LfibTile<KIND, SLOTS>;
    constexpr int R = TL::R, S = TL::S, STRIDE = TL::STRIDE;
    extern __shared__ float lfib_ring[];
    float *ring = lfib_ring;
    const uint64_t s0 = (uint64_t)blockIdx.x * LFIB_T;
    const uint32_t t = threadIdx.x, lane = t & 31u, warp = t >> 5;
    float *st = (float *)g.state + (uint64_t)blockIdx.x * (uint64_t)R;
    if (n == 0ull) return;
    for (uint32_t i = t; i < (uint32_t)R; i += LFIB_T) ring[TL::addr((uint32_t)(SLOTS * LFIB_T - R) + i)] = st[i];
    typename TL::template Lag<R> la;
    typename TL::template Lag<S> lb;
    la.init(ring, t);
    lb.init(ring, t);
    float *wp = ring + t;
    const bool vec_ok = (n & 3ull) == 0ull; // every row start is then 16-byte aligned
    __syncthreads();
    uint32_t kk = (uint32_t)SLOTS;
    for (uint64_t j0 = 0; j0 < n; j0 += SLOTS) {
        kk = (uint32_t)((n - j0 < (uint64_t)SLOTS) ? (n - j0) : (uint64_t)SLOTS);
        if (kk == (uint32_t)SLOTS) {
#pragma unroll
            for (int q = 0; q < SLOTS; q++) {
                wp[q * STRIDE] = lfib_add(la.at(q), lb.at(q));
                if (q % TL::PER_BAR == TL::PER_BAR - 1 || q == SLOTS - 1) __syncthreads();
            }
        } else {
            for (uint32_t q = 0; q < kk; q++) { // ragged last tile of the call
                wp[q * STRIDE] = lfib_add(la.at_dyn(ring, t, q), lb.at_dyn(ring, t, q));
                __syncthreads();
            }
        }
        // ---- write out rows 32 warp .. 32 warp + 31 (this warp's own streams) ----
        if (kk == (uint32_t)SLOTS && vec_ok) {
            const uint32_t c = lane & 7u, rs = lane >> 3;
#pragma unroll
            for (int it = 0; it < 8; it++) {
                const uint32_t row = warp * 32u + 4u * (uint32_t)it + rs;
#pragma unroll
                for (int h = 0; h < SLOTS / 32; h++) { // the 128-byte lines of the row segment, back to back
                    const float *src = ring + (32u * h + 4u * c) * STRIDE + row;
                    uint4 v;
                    v.x = F32 ? __float_as_uint(src[0]) : lfib_u32(src[0]);
                    v.y = F32 ? __float_as_uint(src[STRIDE]) : lfib_u32(src[STRIDE]);
                    v.z = F32 ? __float_as_uint(src[2 * STRIDE]) : lfib_u32(src[2 * STRIDE]);
                    v.w = F32 ? __float_as_uint(src[3 * STRIDE]) : lfib_u32(src[3 * STRIDE]);
                    __stcs(reinterpret_cast<uint4 *>(out + (s0 + row) * n + j0 + 32u * h + 4u * c), v);
                }
            }
        } else {
            for (uint32_t r = 0; r < 32u; r++) {
                const uint32_t row = warp * 32u + r;
                for (uint32_t q = lane; q < kk; q += 32u) {
                    const float v = ring[q * STRIDE + row];
                    __stcs(out + (s0 + row) * n + j0 + q, F32 ? __float_as_uint(v) : lfib_u32(v));
                }
            }
        }
        __syncthreads(); // before the slots are overwritten
    }
    // the state: the last r numbers, oldest first; the last tile ended with batch kk - 1 in slot kk - 1
    for (uint32_t i = t; i < (uint32_t)R; i += LFIB_T)
        st[i] = ring[TL::addr((LFIB_T * kk - (uint32_t)R + i) & (uint32_t)(SLOTS * LFIB_T - 1))];
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

template <int KIND, int SLOTS>
static cudaError_t launch_lfib_fill_t(const Gen &g, uint32_t *o, uint64_t n, bool f32, unsigned inst, cudaStream_t st)
{
    constexpr size_t smem = (size_t)LfibTile<KIND, SLOTS>::WORDS * sizeof(float);
    auto kf = lfib_fill_kernel<KIND, true, SLOTS>;
    auto ku = lfib_fill_kernel<KIND, false, SLOTS>;
    if (smem > 48 * 1024) { // cheap and per device: set on every launch
        const cudaError_t e = cudaFuncSetAttribute(f32 ? kf : ku, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    if (f32) kf<<<inst, LFIB_T, smem, st>>>(g, o, n);
    else ku<<<inst, LFIB_T, smem, st>>>(g, o, n);
    count_launch();
    return cudaGetLastError();
}

// variant "store": 0 = automatic (64-draw tiles for rows of at least 64 draws), 1 = 32-draw tiles, 2 = 64-draw tiles
cudaError_t launch_lfib_fill(const Gen &g, void *d_out, uint64_t n, bool f32, int variant, cudaStream_t st)
{
    const uint64_t inst = g.S / LFIB_T;
    if (inst > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    uint32_t *o = (uint32_t *)d_out;
    const bool wide = variant == 2 || (variant == 0 && n >= 64);
    if (g.kind == RNG_LFIB1279)
        return wide ? launch_lfib_fill_t<RNG_LFIB1279, 64>(g, o, n, f32, (unsigned)inst, st)
                    : launch_lfib_fill_t<RNG_LFIB1279, 32>(g, o, n, f32, (unsigned)inst, st);
    return wide ? launch_lfib_fill_t<RNG_LFIB521, 64>(g, o, n, f32, (unsigned)inst, st)
                : launch_lfib_fill_t<RNG_LFIB521, 32>(g, o, n, f32, (unsigned)inst, st);
}

} // namespace rngb200
