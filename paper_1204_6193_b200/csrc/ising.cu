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

// ------------------------------------------------------------------------------------
// chunk half-sweep (fast path A): one thread per 16-byte chunk of a row = 8 sites of the
// active colour.  Block (32, 8): lanes = 32 consecutive chunks (512 contiguous bytes of a
// row), warps = 8 consecutive rows, so the rows a CTA reads as "up", "centre" and "down"
// overlap in L1 and every global access is a coalesced 128-bit one.
//
//  * spins stay int8 +1/-1 (0x01 / 0xff).  For a word w of the centre row and the words
//    l, r (w shifted by one byte either way across the word boundary), u, d (rows y-1, y+1):
//        A = ((l^w)&m) + ((r^w)&m) + ((u^w)&m) + ((d^w)&m),   m = 0x02020202
//    holds in EVERY byte 2*nbar, nbar = number of neighbours anti-aligned with that spin
//    (0x01^0xff = 0xfe has bit 1 set); only the bytes at active sites are used.  The number
//    of aligned neighbours is (h+4)/2 = 4 - nbar, h = s * (sum of neighbours)  (R-E2).
//  * threshold lookup: byte 4*nbar of (A<<1) is the byte offset into a 5-entry shared
//    table tab[nbar] = 256*T[4-nbar] - 1, and  (r>>8) < T  <=>  r <= 256*T - 1  for
//    1 <= T <= 2^24 (the host takes the generic kernel if some T is 0).
//  * flip = xor 0xfe into the site's byte, predicated on the compare.
//  * the one neighbour byte outside the chunk (left of byte 0 if the sites sit at even x,
//    right of byte 15 if at odd x) comes from the adjacent lane by shuffle, from global
//    memory at the ends of the warp.  It belongs to the other colour, which no thread
//    writes during this half-sweep.
//
// Streams: PHILOX (stateless; needs K % 4 == 0 and draws_done % 4 == 0): the chunk's two
// groups of 4 sites are two whole Philox blocks of the owning stream(s).  Stateful kinds
// need K == 8: the thread owns stream s = chunk index, state in registers for 8 draws.
// ------------------------------------------------------------------------------------
struct IsingFastTable {
    uint32_t thr[5]; // thr[nbar] = 256*T[4-nbar] - 1
};

template <int KIND>
__global__ void __launch_bounds__(256) ising_chunk_kernel(Gen g, int8_t *__restrict__ sp, uint32_t L, IsingFastTable ft,
                                                          uint32_t K, int log2K, int colour)
{
    __shared__ uint32_t tab[8];
    if (threadIdx.y == 0 && threadIdx.x < 5) tab[threadIdx.x] = ft.thr[threadIdx.x];
    __syncthreads();
    constexpr unsigned FULL = 0xffffffffu;
    const uint32_t lane = threadIdx.x;
    const uint32_t cpr = L >> 4; // chunks per row
    const uint32_t cx_raw = blockIdx.x * 32u + lane;
    const bool active = cx_raw < cpr;
    const uint32_t cx = active ? cx_raw : cpr - 1u;
    const uint32_t y = blockIdx.y * 8u + threadIdx.y;
    const uint32_t yu = y ? y - 1u : L - 1u, yd = (y + 1u == L) ? 0u : y + 1u;
    const uint32_t p = (y + (uint32_t)colour) & 1u; // x parity of the active sites of this row (warp-uniform)

    int8_t *rowp = sp + (uint64_t)y * L;
    const uint4 W4 = reinterpret_cast<const uint4 *>(rowp)[cx];
    const uint4 U4 = reinterpret_cast<const uint4 *>(sp + (uint64_t)yu * L)[cx];
    const uint4 D4 = reinterpret_cast<const uint4 *>(sp + (uint64_t)yd * L)[cx];
    uint32_t w[4] = {W4.x, W4.y, W4.z, W4.w};
    const uint32_t u[4] = {U4.x, U4.y, U4.z, U4.w};
    const uint32_t d[4] = {D4.x, D4.y, D4.z, D4.w};

    uint32_t prevw = 0u, nextw = 0u; // word left of w[0] (top byte used) / right of w[3] (low byte used)
    if (p == 0u) {
        prevw = __shfl_up_sync(FULL, w[3], 1);
        if (lane == 0u) {
            const uint32_t xl = cx ? cx * 16u - 1u : L - 1u;
            prevw = (uint32_t)(uint8_t)rowp[xl] << 24;
        }
    } else {
        nextw = __shfl_down_sync(FULL, w[0], 1);
        if (lane == 31u || cx_raw + 1u >= cpr) {
            const uint32_t xr = (cx + 1u == cpr) ? 0u : cx * 16u + 16u;
            nextw = (uint32_t)(uint8_t)rowp[xr];
        }
    }

    // per byte: 4 * (number of anti-aligned neighbours) = byte offset into tab
    constexpr uint32_t M = 0x02020202u;
    uint32_t a4[4];
#pragma unroll
    for (int i = 0; i < 4; i++) {
        const uint32_t l = __funnelshift_l(i ? w[i - 1] : prevw, w[i], 8);
        const uint32_t r = __funnelshift_r(w[i], i < 3 ? w[i + 1] : nextw, 8);
        const uint32_t a = ((l ^ w[i]) & M) + ((r ^ w[i]) & M) + ((u[i] ^ w[i]) & M) + ((d[i] ^ w[i]) & M);
        a4[i] = a << 1;
    }

    // the 8 draws of this chunk, in site order
    uint32_t rnd[8];
    if (kind_is_philox(KIND)) {
        const uint64_t q0 = (uint64_t)y * (L >> 1) + 8ull * cx;
#pragma unroll
        for (int gi = 0; gi < 2; gi++) {
            const uint64_t qg = q0 + 4u * gi;
            const uint64_t s = log2K >= 0 ? (qg >> log2K) : (qg / K);
            const uint64_t k = qg - s * K;
            const uint64_t key = (g.first + s) ^ g.seed;
            const uint64_t b = (g.draws_done + k) >> 2;
            const uint4 o = philox4x32<philox_rounds(KIND)>((uint32_t)b, (uint32_t)(b >> 32), 0u, 0u, (uint32_t)key, (uint32_t)(key >> 32));
            rnd[4 * gi + 0] = o.x;
            rnd[4 * gi + 1] = o.y;
            rnd[4 * gi + 2] = o.z;
            rnd[4 * gi + 3] = o.w;
        }
    } else {
        const uint64_t s = (uint64_t)y * cpr + cx; // K == 8: stream = chunk
        Stream<KIND> gen;
        gen.load(g, s);
#pragma unroll
        for (int t = 0; t < 8; t++) rnd[t] = gen.next();
        if (active) gen.store(g, s);
    }

    const uint32_t sel0 = 0x4440u | p, sel1 = 0x4442u | p;        // byte p / byte 2+p of a word -> low byte
    const uint32_t fm0 = 0xfeu << (8u * p), fm1 = 0xfe0000u << (8u * p);
    const char *tabb = reinterpret_cast<const char *>(tab);
#pragma unroll
    for (int t = 0; t < 8; t++) {
        const int i = t >> 1;
        const uint32_t off = __byte_perm(a4[i], 0u, (t & 1) ? sel1 : sel0);
        const uint32_t thr = *reinterpret_cast<const uint32_t *>(tabb + off);
        if (rnd[t] <= thr) w[i] ^= (t & 1) ? fm1 : fm0;
    }
    if (active) reinterpret_cast<uint4 *>(rowp)[cx] = make_uint4(w[0], w[1], w[2], w[3]);
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
    // fast path A (chunk kernel): see ising_chunk_kernel
    {
        bool thr_ok = true;
        IsingFastTable ft;
        for (int nb = 0; nb < 5; nb++) {
            const uint32_t T = tab.T[4 - nb];
            if (T < 1u || T > (1u << 24)) thr_ok = false;
            ft.thr[nb] = (uint32_t)(((uint64_t)T << 8) - 1ull);
        }
        const uint32_t cpr = L >> 4;
        const bool geom_ok = (L % 16u) == 0u && L >= 16u && L <= 65536u && h.var_ising != 1;
        bool kind_ok;
        if (kind_is_philox(g.kind)) kind_ok = (K % 4ull) == 0ull && (draws_done % 4ull) == 0ull;
        else if (kind_is_lfib(g.kind)) kind_ok = false; // CTA-shared state: the generic kernel's thread <-> stream map only
        else if (g.kind == RNG_XS1024W) kind_ok = K == 8ull && (cpr % 32u) == 0u;
        else kind_ok = K == 8ull;
        if (thr_ok && geom_ok && kind_ok) {
            int log2K = -1;
            if ((K & (K - 1)) == 0) {
                log2K = 0;
                while ((1ull << log2K) < K) log2K++;
            }
            const dim3 blk(32, 8), grd((cpr + 31) / 32, L / 8);
#define CHUNK(KIND) ising_chunk_kernel<KIND><<<grd, blk, 0, st>>>(g, d_spins, L, ft, (uint32_t)K, log2K, colour)
            RNGB200_DISPATCH_KIND(g.kind, CHUNK)
#undef CHUNK
            count_launch();
            return cudaGetLastError();
        }
    }
    const uint64_t grid = (g.S + 255) / 256;
    if (grid > 0x7fffffffull) return cudaErrorInvalidConfiguration;
#define GENERIC(KIND) \
    ising_half_sweep_generic_kernel<KIND><<<(unsigned)grid, 256, 0, st>>>(g, d_spins, L, tab, K, colour)
    if (g.kind == RNG_LFIB521) GENERIC(RNG_LFIB521);
    else if (g.kind == RNG_LFIB1279) GENERIC(RNG_LFIB1279);
    else {
        RNGB200_DISPATCH_KIND(g.kind, GENERIC)
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
