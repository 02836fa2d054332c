// fill.cu -- fill mode: advance every stream by n draws and write them stream-major to HBM
// (SURVEY.md 8(a) rows a2-a5, a7).  out[s*n + j] = draw j of stream s.
//
// Two kernel families:
//  * philox_fill_kernel: Philox is stateless, so ANY thread can compute any
//    (stream, 4-word block).  Consecutive threads take consecutive blocks of a row and each
//    stores its whole block with one 128-bit store: coalesced by construction.
//  * rowtile_fill_kernel: generators with per-thread state (LCG64, XORWOW, xs1024) produce
//    a row per thread.  A warp stages a [32 rows][KT draws] tile in shared memory (128-bit
//    conflict-free stores), then writes every row segment with full-line 128-bit stores.
#include "internal.h"
#include "streams.cuh"

namespace rngb200 {

__device__ __forceinline__ uint32_t out_word(uint32_t u, bool f32)
{
    return f32 ? __float_as_uint(u32_to_f32(u)) : u;
}

// ------------------------------------------------------------------------------------
// Philox direct fill.  Row s of this call covers draws [d0, d0+n) of stream s, i.e. the
// 4-word blocks b0 = d0/4 .. b1 = (d0+n-1)/4.  A tile is 256*U consecutive blocks of one
// row; tiles are handed to CTAs grid-stride.  ALIGNED (d0 % 4 == 0 and n % 4 == 0): every
// block is written whole with a 128-bit store; otherwise word by word with bounds checks.
// ------------------------------------------------------------------------------------
template <bool F32, bool ALIGNED, int U>
__global__ void __launch_bounds__(256) philox_fill_kernel(uint32_t *__restrict__ out, uint64_t S, uint64_t first,
                                                         uint64_t seed, uint64_t d0, uint64_t n,
                                                         uint64_t blocks_per_row, uint32_t tiles_per_row,
                                                         uint64_t n_tiles)
{
    const uint64_t b0 = d0 >> 2;
    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        const uint64_t s = t / tiles_per_row;        // uniform per CTA
        const uint32_t c = (uint32_t)(t % tiles_per_row);
        const uint64_t key = (first + s) ^ seed;     // R-C2: key = stream id ^ seed
        const uint32_t k0 = (uint32_t)key, k1 = (uint32_t)(key >> 32);
        uint32_t *row = out + s * n;
#pragma unroll
        for (int u = 0; u < U; u++) {
            const uint64_t rb = (uint64_t)c * (256 * U) + u * 256 + threadIdx.x; // block within the row
            if (rb >= blocks_per_row) continue;
            const uint64_t b = b0 + rb; // counter = index of the 4-word block
            uint4 r = philox4x32<10>((uint32_t)b, (uint32_t)(b >> 32), 0u, 0u, k0, k1);
            r.x = out_word(r.x, F32);
            r.y = out_word(r.y, F32);
            r.z = out_word(r.z, F32);
            r.w = out_word(r.w, F32);
            if (ALIGNED) {
                __stcs(reinterpret_cast<uint4 *>(row + 4 * rb), r); // streaming 128-bit store
            } else {
                const int64_t j = (int64_t)(4 * b) - (int64_t)d0; // position of word 0 in the row
                if (j >= 0 && (uint64_t)j < n) row[j] = r.x;
                if (j + 1 >= 0 && (uint64_t)(j + 1) < n) row[j + 1] = r.y;
                if (j + 2 >= 0 && (uint64_t)(j + 2) < n) row[j + 2] = r.z;
                if (j + 3 >= 0 && (uint64_t)(j + 3) < n) row[j + 3] = r.w;
            }
        }
    }
}

// ------------------------------------------------------------------------------------
// Row-tile fill for stateful generators: thread s owns stream s and its output row.
// ------------------------------------------------------------------------------------
constexpr int KT = 32;            // draws per row per tile (one 128-byte line)
constexpr int KT_STRIDE = KT + 4; // padded row stride in words: 16-byte aligned rows and
                                  // conflict-free 128-bit accesses (8 lanes x 4 banks)
constexpr int FILL_WARPS = 8;

template <int KIND, bool F32>
__global__ void __launch_bounds__(FILL_WARPS * 32) rowtile_fill_kernel(Gen g, uint32_t *__restrict__ out, uint64_t n)
{
    __shared__ __align__(16) uint32_t tiles[FILL_WARPS][32 * KT_STRIDE];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *tile = tiles[warp];
    const uint64_t s0 = ((uint64_t)blockIdx.x * FILL_WARPS + warp) * 32ull; // first row of this warp
    if (s0 >= g.S) return;
    const uint64_t s = s0 + lane;
    const bool live = s < g.S;
    const uint32_t rows = (uint32_t)((g.S - s0 < 32ull) ? (g.S - s0) : 32ull);
    const bool vec_ok = (n & 3ull) == 0ull; // every row start is then 16-byte aligned

    Stream<KIND> gen;
    if (live) gen.load(g, s);

    for (uint64_t j0 = 0; j0 < n; j0 += KT) {
        const uint32_t kk = (uint32_t)((n - j0 < (uint64_t)KT) ? (n - j0) : (uint64_t)KT);
        // ---- generate: lane writes kk draws into its own tile row ----
        // (xs1024 is cooperative: S % 32 == 0, so `live` is warp-uniform for it)
        if (live) {
            uint32_t *my = tile + lane * KT_STRIDE;
            if (kk == KT) {
#pragma unroll
                for (int q = 0; q < KT / 4; q++) {
                    uint4 v;
                    v.x = out_word(gen.next(), F32);
                    v.y = out_word(gen.next(), F32);
                    v.z = out_word(gen.next(), F32);
                    v.w = out_word(gen.next(), F32);
                    *reinterpret_cast<uint4 *>(my + 4 * q) = v;
                }
            } else {
                for (uint32_t q = 0; q < kk; q++) my[q] = out_word(gen.next(), F32);
            }
        }
        __syncwarp();
        // ---- write out: row segments of kk words, stream-major ----
        if (kk == KT && vec_ok) {
#pragma unroll
            for (int it = 0; it < KT / 4; it++) {
                const int v = it * 32 + lane;
                const int r = v / (KT / 4), c4 = v % (KT / 4);
                if ((uint32_t)r < rows) {
                    const uint4 val = *reinterpret_cast<const uint4 *>(tile + r * KT_STRIDE + 4 * c4);
                    __stcs(reinterpret_cast<uint4 *>(out + (s0 + r) * n + j0 + 4 * c4), val);
                }
            }
        } else {
            for (uint32_t r = 0; r < rows; r++)
                for (uint32_t c = lane; c < kk; c += 32) out[(s0 + r) * n + j0 + c] = tile[r * KT_STRIDE + c];
        }
        __syncwarp();
    }
    if (live) gen.store(g, s);
}

template <int KIND>
static cudaError_t launch_rowtile(const Gen &g, void *d_out, uint64_t n, bool f32, cudaStream_t st)
{
    const uint64_t warps = (g.S + 31) / 32;
    const uint64_t grid = (warps + FILL_WARPS - 1) / FILL_WARPS;
    if (grid > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    if (f32)
        rowtile_fill_kernel<KIND, true><<<(unsigned)grid, FILL_WARPS * 32, 0, st>>>(g, (uint32_t *)d_out, n);
    else
        rowtile_fill_kernel<KIND, false><<<(unsigned)grid, FILL_WARPS * 32, 0, st>>>(g, (uint32_t *)d_out, n);
    count_launch();
    return cudaGetLastError();
}

static int g_sm_count = 0;
static int sm_count()
{
    if (!g_sm_count) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&g_sm_count, cudaDevAttrMultiProcessorCount, dev);
        if (g_sm_count <= 0) g_sm_count = 148;
    }
    return g_sm_count;
}

static cudaError_t launch_philox_fill(const Gen &g, void *d_out, uint64_t n, bool f32, cudaStream_t st)
{
    constexpr int U = 4;
    const uint64_t d0 = g.draws_done;
    const uint64_t blocks_per_row = ((d0 + n - 1) >> 2) - (d0 >> 2) + 1;
    const uint64_t tpr = (blocks_per_row + 256 * U - 1) / (256 * U);
    if (tpr > 0xffffffffull) return cudaErrorInvalidConfiguration;
    const uint64_t n_tiles = g.S * tpr;
    const bool aligned = ((d0 | n) & 3ull) == 0ull;
    // persistent-style grid: a multiple of the SM count, 8 resident CTAs of 256 threads per SM
    uint64_t grid = (uint64_t)sm_count() * 8ull;
    if (grid > n_tiles) grid = n_tiles;
    uint32_t *o = (uint32_t *)d_out;
#define PHILOX_LAUNCH(F, A) \
    philox_fill_kernel<F, A, U><<<(unsigned)grid, 256, 0, st>>>(o, g.S, g.first, g.seed, d0, n, blocks_per_row, \
                                                              (uint32_t)tpr, n_tiles)
    if (f32) {
        if (aligned) PHILOX_LAUNCH(true, true);
        else PHILOX_LAUNCH(true, false);
    } else {
        if (aligned) PHILOX_LAUNCH(false, true);
        else PHILOX_LAUNCH(false, false);
    }
#undef PHILOX_LAUNCH
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_fill(const rng_handle &h, void *d_out, uint64_t n, bool f32, cudaStream_t st)
{
    const Gen &g = h.g;
    switch (g.kind) {
    case RNG_LCG64: return launch_rowtile<RNG_LCG64>(g, d_out, n, f32, st);
    case RNG_LCG64_LEAPFROG: return launch_rowtile<RNG_LCG64_LEAPFROG>(g, d_out, n, f32, st);
    case RNG_XORWOW: return launch_rowtile<RNG_XORWOW>(g, d_out, n, f32, st);
    case RNG_XS1024W: return launch_rowtile<RNG_XS1024W>(g, d_out, n, f32, st);
    case RNG_PHILOX4X32_10: return launch_philox_fill(g, d_out, n, f32, st);
    default: return cudaErrorInvalidValue;
    }
}

} // namespace rngb200
