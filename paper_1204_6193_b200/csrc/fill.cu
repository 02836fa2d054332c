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

// ------------------------------------------------------------------------------------
// Philox direct fill.  Row s of this call covers draws [d0, d0+n) of stream s, i.e. the
// 4-word blocks b0 = d0/4 .. b1 = (d0+n-1)/4.  A tile is 256*U consecutive blocks of one
// row; tiles are handed to CTAs grid-stride.  ALIGNED (d0 % 4 == 0 and n % 4 == 0): every
// block is written whole with a 128-bit store; otherwise word by word with bounds checks.
// ------------------------------------------------------------------------------------
template <bool F32, bool ALIGNED, int U, int R>
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
            uint4 r = philox4x32<R>((uint32_t)b, (uint32_t)(b >> 32), 0u, 0u, k0, k1);
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
// Philox warp-tile fill (the aligned fast path: d0 % 4 == 0 and n % 4 == 0).
// A tile is 32*U*T consecutive 4-word blocks of ONE row and belongs to one warp; it is
// processed as T groups of 32*U blocks, lane l computing blocks l, l+32, ... of the group so
// that every store instruction of the warp writes 512 contiguous bytes.
//  * The row (hence the key) is fixed per tile and the warp index comes from a broadcast
//    shuffle, which makes it provably warp-uniform: the ten round keys k + r*(W0,W1) are
//    computed once per tile in UNIFORM registers and cost no per-thread registers or
//    per-block instructions.  What is left per round and block is Philox's own arithmetic
//    (PAPER.md:290-294): 2 IMAD.WIDE + 2 LOP3 (three-input xor with a uniform operand).
//  * The counter is (lo32(b), hi32(b), 0, 0) (R-C2), so the first round's second S-box
//    multiplies zero and folds away at compile time.
//  * U independent blocks per lane are interleaved (the full-tile path has no per-block
//    predicate, so ptxas keeps them interleaved) and hide the IMAD -> LOP3 -> IMAD chain.
//  * Persistent grid: warps stride over tiles; (row, tile-in-row) advance incrementally
//    (one 64-bit division per warp).  Tried in round 2 and rejected: handing out chunks of tiles through an
//    atomic ticket counter, which lifts the store-bound xs1024 fill (fill_xs1024.cu).  Here it measured
//    651 us (static) against 673 us (tickets of 16 tiles) and 708 us (8 tiles) per 4 GiB: this kernel is bound by
//    its IMAD.WIDE arithmetic, not by an uneven share of the write bandwidth, and same-address atomics cost
//    about 3 ns each.
// ------------------------------------------------------------------------------------
// the four words of a block as they are stored: the draws, or the bits of their float images (form CVT of the
// fixed map, generators.cuh)
template <bool F32, int CVT>
__device__ __forceinline__ uint4 philox_out(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3)
{
    if (!F32) return make_uint4(c0, c1, c2, c3);
    return make_uint4(__float_as_uint(u32_to_f32_form<CVT>(c0)), __float_as_uint(u32_to_f32_form<CVT>(c1)),
                      __float_as_uint(u32_to_f32_form<CVT>(c2)), __float_as_uint(u32_to_f32_form<CVT>(c3)));
}

// U independent 4-word blocks per lane (blocks rb0, rb0+32, ...), ten rounds interleaved,
// one 128-bit streaming store each.  CHECK = bounds-check each block (ragged last tile).
template <bool F32, int U, bool CHECK, int R, int CVT>
__device__ __forceinline__ void philox_group(uint32_t *__restrict__ row, uint64_t b0, uint32_t rb0,
                                             uint32_t blocks_per_row, const uint32_t (&rk0)[R],
                                             const uint32_t (&rk1)[R])
{
    uint32_t c0[U], c1[U], c2[U], c3[U];
#pragma unroll
    for (int u = 0; u < U; u++) {
        const uint64_t b = b0 + rb0 + 32u * u; // counter = index of the 4-word block (R-C2)
        c0[u] = (uint32_t)b;
        c1[u] = (uint32_t)(b >> 32);
        c2[u] = 0u;
        c3[u] = 0u;
    }
#pragma unroll
    for (int r = 0; r < R; r++) {
#pragma unroll
        for (int u = 0; u < U; u++) {
            const uint64_t p0 = (uint64_t)kPhM0 * c0[u];
            const uint64_t p1 = (uint64_t)kPhM1 * c2[u];
            const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1[u] ^ rk0[r];
            const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3[u] ^ rk1[r];
            c1[u] = (uint32_t)p1;
            c3[u] = (uint32_t)p0;
            c0[u] = n0;
            c2[u] = n2;
        }
    }
    uint4 *dst = reinterpret_cast<uint4 *>(row) + rb0; // one address per lane; the U stores use immediate offsets
#pragma unroll
    for (int u = 0; u < U; u++) {
        if (!CHECK || rb0 + 32u * u < blocks_per_row) {
            __stcs(dst + 32 * u, philox_out<F32, CVT>(c0[u], c1[u], c2[u], c3[u])); // streaming 128-bit store
        }
    }
}

// Full tile whose blocks all share the high counter word (every tile except one per 2^32
// blocks of a row): the structure of the counter (lo32(b), hi32(b), 0, 0) (R-C2) removes two
// of the 2R multiplies of each block.
//  * round 1: the second S-box multiplies zero; the first one, M0 * lo32(b), is linear in b:
//    the lane's blocks are b, b+32, ..., so p0(b + 32u) = p0(b) + u * (32 M0) as 64-bit
//    integers (lo32 does not wrap inside the tile): one IMAD.WIDE per lane and group, then
//    64-bit additions on the otherwise half-idle alu pipe.
//  * round 2: its first S-box input is hi32(b) ^ k0 (round 1 left c0 = hi(M1*0) ^ c1 ^ k0),
//    the same for every block of the tile: one product per lane and group (`q`).
// Rounds 3..R are the generic round.  Same bits as philox4x32<R> (tests compare both paths
// with the oracle, also across a 2^32-block boundary).
template <bool F32, int U, int R, int CVT>
__device__ __forceinline__ void philox_group_fast(uint32_t *__restrict__ row, uint32_t blo, uint32_t bhi, uint32_t rb0,
                                                  const uint32_t (&rk0)[R], const uint32_t (&rk1)[R])
{
    static_assert(R >= 3, "needs three rounds");
    uint32_t c0[U], c1[U], c2[U], c3[U];
    const uint64_t p00 = (uint64_t)kPhM0 * blo;                       // round 1, block u = 0
    const uint64_t q = (uint64_t)kPhM0 * (bhi ^ rk0[0]);              // round 2, first S-box: tile-uniform input
    // q and the round keys are warp-uniform: fold them into ONE uniform operand per xor here, because a LOP3
    // takes a single uniform-register source and ptxas otherwise copies the second one into a vector register
    // for every block (12 IMAD.U32 per group of 8 blocks in round 1's build)
    uint32_t hq1 = (uint32_t)(q >> 32) ^ rk1[1];                      // round 2: c2 = hi(q) ^ a3 ^ k1'
    uint32_t lq2 = (uint32_t)q ^ rk1[2];                              // round 3: c2 = hi(p0) ^ c3 ^ k1'', c3 = lo(q)
    hq1 = __shfl_sync(0xffffffffu, hq1, 0);                           // (a shuffle is opaque to the xor re-association
    lq2 = __shfl_sync(0xffffffffu, lq2, 0);                           //  of nvvm and ptxas, which would unfold them)
    constexpr uint64_t STEP = 32ull * kPhM0;
#pragma unroll
    for (int u = 0; u < U; u++) {
        const uint64_t p0 = p00 + (uint64_t)u * STEP;                 // = M0 * (blo + 32u)
        // after round 1: (c0,c1,c2,c3) = (bhi ^ k0, 0, hi(p0) ^ k1, lo(p0))
        const uint32_t a2 = (uint32_t)(p0 >> 32) ^ rk1[0];
        const uint32_t a3 = (uint32_t)p0;
        // round 2
        const uint64_t p1 = (uint64_t)kPhM1 * a2;
        const uint32_t b0 = (uint32_t)(p1 >> 32) ^ rk0[1];            // ^ c1 (= 0)
        const uint32_t b2 = hq1 ^ a3;
        // round 3 (c3 = lo(q) is uniform and already folded into lq2)
        const uint64_t r0 = (uint64_t)kPhM0 * b0;
        const uint64_t r1 = (uint64_t)kPhM1 * b2;
        c0[u] = (uint32_t)(r1 >> 32) ^ (uint32_t)p1 ^ rk0[2];
        c2[u] = (uint32_t)(r0 >> 32) ^ lq2;
        c1[u] = (uint32_t)r1;
        c3[u] = (uint32_t)r0;
    }
#pragma unroll
    for (int r = 3; r < R; r++) {
#pragma unroll
        for (int u = 0; u < U; u++) {
            const uint64_t p0 = (uint64_t)kPhM0 * c0[u];
            const uint64_t p1 = (uint64_t)kPhM1 * c2[u];
            const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1[u] ^ rk0[r];
            const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3[u] ^ rk1[r];
            c1[u] = (uint32_t)p1;
            c3[u] = (uint32_t)p0;
            c0[u] = n0;
            c2[u] = n2;
        }
    }
    uint4 *dst = reinterpret_cast<uint4 *>(row) + rb0;
#pragma unroll
    for (int u = 0; u < U; u++) {
        __stcs(dst + 32 * u, philox_out<F32, CVT>(c0[u], c1[u], c2[u], c3[u]));
    }
}

// ALLFAST (host-checked: every tile is full and no tile of the call crosses a 2^32-block boundary): the per-tile
// bookkeeping shrinks to the key schedule and the row pointer.
template <bool F32, int U, int T, int R, bool ALLFAST, int CVT>
__global__ void __launch_bounds__(256) philox_fill_warp_kernel(uint32_t *__restrict__ out, uint64_t first, uint64_t seed,
                                                              uint64_t b0, uint64_t n, uint32_t blocks_per_row,
                                                              uint32_t tiles_per_row, uint64_t n_tiles)
{
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t warp_in_cta = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0); // warp-uniform by construction
    const uint64_t n_warps = (uint64_t)gridDim.x * (blockDim.x >> 5);
    uint64_t t = (uint64_t)blockIdx.x * (blockDim.x >> 5) + warp_in_cta;
    if (t >= n_tiles) return;
    uint64_t s = t / tiles_per_row;                    // row of this warp's first tile
    uint32_t c = (uint32_t)(t - s * tiles_per_row);    // tile within the row
    const uint64_t ds = n_warps / tiles_per_row;       // per-iteration advance of (s, c)
    const uint32_t dc = (uint32_t)(n_warps - ds * tiles_per_row);
    for (; t < n_tiles; t += n_warps) {
        const uint64_t key = (first + s) ^ seed; // R-C2: key = stream id ^ seed
        uint32_t rk0[R], rk1[R];
#pragma unroll
        for (int r = 0; r < R; r++) {
            rk0[r] = (uint32_t)key + (uint32_t)r * kPhW0;
            rk1[r] = (uint32_t)(key >> 32) + (uint32_t)r * kPhW1;
        }
        uint32_t *row = out + s * n;
        if (ALLFAST) {
#pragma unroll 1
            for (int g = 0; g < T; g++) {
                const uint32_t rb0 = (c * T + g) * (32u * U) + lane;
                philox_group_fast<F32, U, R, CVT>(row, (uint32_t)b0 + rb0, (uint32_t)(b0 >> 32), rb0, rk0, rk1);
            }
            s += ds;
            c += dc;
            if (c >= tiles_per_row) {
                c -= tiles_per_row;
                s++;
            }
            continue;
        }
        const bool tile_full = (uint64_t)(c + 1u) * (T * 32u * U) <= (uint64_t)blocks_per_row; // warp-uniform
        // first and last block index of the tile (warp-uniform); equal high words <=> lo32 does not wrap
        const uint64_t bt0 = b0 + (uint64_t)c * (T * 32u * U), bt1 = bt0 + (T * 32u * U - 1u);
        if (tile_full && (uint32_t)(bt0 >> 32) == (uint32_t)(bt1 >> 32)) {
#pragma unroll 1
            for (int g = 0; g < T; g++) {
                const uint32_t rb0 = (c * T + g) * (32u * U) + lane;
                philox_group_fast<F32, U, R, CVT>(row, (uint32_t)b0 + rb0, (uint32_t)(bt0 >> 32), rb0, rk0, rk1);
            }
        } else if (tile_full) {
#pragma unroll 1
            for (int g = 0; g < T; g++)
                philox_group<F32, U, false, R, CVT>(row, b0, (c * T + g) * (32u * U) + lane, blocks_per_row, rk0, rk1);
        } else {
#pragma unroll 1
            for (int g = 0; g < T; g++)
                philox_group<F32, U, true, R, CVT>(row, b0, (c * T + g) * (32u * U) + lane, blocks_per_row, rk0, rk1);
        }
        s += ds;
        c += dc;
        if (c >= tiles_per_row) {
            c -= tiles_per_row;
            s++;
        }
    }
}

// ------------------------------------------------------------------------------------
// Row-tile fill for stateful generators: thread s owns stream s and its output row.
// ------------------------------------------------------------------------------------
// A warp stages a [32 rows][KT draws] tile; KT = 64 makes every row segment 256 contiguous
// bytes, which on B200 lifts the ceiling of this write pattern from 5.6 to 6.6 TB/s for
// 4 KiB rows (microbenchmark of the bare pattern), KT = 32 halves the shared memory.
constexpr int FILL_WARPS = 4;

template <int KIND, bool F32, int KT>
__global__ void __launch_bounds__(FILL_WARPS * 32) rowtile_fill_kernel(Gen g, uint32_t *__restrict__ out, uint64_t n)
{
    constexpr int KT_STRIDE = KT + 4; // padded row stride in words: 16-byte aligned rows and
                                      // conflict-free 128-bit accesses (8 lanes x 4 banks)
    constexpr int CPR = KT / 4;       // 16-byte chunks per row segment
    constexpr int RPI = 32 / CPR;     // rows per warp store instruction
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
            const uint32_t c4 = (uint32_t)lane % CPR, r0 = (uint32_t)lane / CPR;
            uint32_t *gp = out + (s0 + r0) * n + j0 + 4u * c4;
            const uint32_t *tp = tile + r0 * KT_STRIDE + 4u * c4;
            const uint64_t gstep = (uint64_t)RPI * n;
            if (rows == 32u) {
#pragma unroll
                for (int h = 0; h < 32 / RPI; h += 8) { // eight loads in flight, then eight stores
                    uint4 v[8];
#pragma unroll
                    for (int i = 0; i < 8; i++) v[i] = *reinterpret_cast<const uint4 *>(tp + (h + i) * RPI * KT_STRIDE);
#pragma unroll
                    for (int i = 0; i < 8; i++) __stcs(reinterpret_cast<uint4 *>(gp + (uint64_t)(h + i) * gstep), v[i]);
                }
            } else {
                for (uint32_t r = r0; r < rows; r += RPI)
                    __stcs(reinterpret_cast<uint4 *>(out + (s0 + r) * n + j0 + 4u * c4),
                           *reinterpret_cast<const uint4 *>(tile + r * KT_STRIDE + 4u * c4));
            }
        } else {
            for (uint32_t r = 0; r < rows; r++)
                for (uint32_t c = lane; c < kk; c += 32) out[(s0 + r) * n + j0 + c] = tile[r * KT_STRIDE + c];
        }
        __syncwarp();
    }
    if (live) gen.store(g, s);
}

// ------------------------------------------------------------------------------------
// LCG64 with FEW streams (BASELINE config 1: 1024 streams x 4096 draws): one thread per
// stream would leave the chip empty and serialise 4096 dependent multiplies per thread.
// The paper's skip-ahead (eq.(2)) is applied INSIDE each stream instead:
// one CTA per stream, lane t starts at x_{4t} = step^(4t)(x_0) (table mult4, built by the
// seeding kernel), writes draws 4t..4t+3 with one 128-bit store and leaps by
// step^1024 = pow2[10] to its next chunk.  Same bits as the sequential walk, coalesced for
// free (a warp instruction stores 512 contiguous bytes).  Thread 0 writes the stream's final
// state x_n = step^n(x_0), composed from the pow2 table over the bits of n.
// ------------------------------------------------------------------------------------
template <bool F32>
__global__ void __launch_bounds__(256) lcg_intra_fill_kernel(Gen g, uint32_t *__restrict__ out, uint64_t n)
{
    pdl_entry(); // back-to-back calls on one handle: the state comes from the previous launch (internal.h)
    const uint64_t s = blockIdx.x;
    const uint32_t t = threadIdx.x;
    const LcgTable *__restrict__ tab = g.lcg;
    uint64_t *xs = (uint64_t *)g.state;
    const uint64_t x0 = xs[s];
    const Affine step = tab->pow2[0], leap = tab->pow2[10];
    uint64_t x = affine_apply(tab->mult4[t], x0); // x_{4t}
    // The stream's final state x_n = step^n(x_0) depends on x_0 only: the last warp computes and stores it
    // NOW (after every lane has read x_0), so that its dependent table loads overlap the other warps' stores
    // instead of trailing the CTA.
    __syncthreads();
    if (t == 255u) {
        uint64_t y = x0;
        for (int m = 0; m < 64 && (n >> m) != 0ull; m++)
            if ((n >> m) & 1ull) y = affine_apply(tab->pow2[m], y);
        xs[s] = y;
    }
    uint32_t *row = out + s * n;
    const bool vec_ok = (n & 3ull) == 0ull;
    for (uint64_t j = 4ull * t; j < n; j += 1024ull) {
        uint64_t y = x;
        uint4 v;
        v.x = out_word((uint32_t)(y >> 32), F32); // 32 most significant bits
        y = affine_apply(step, y);
        v.y = out_word((uint32_t)(y >> 32), F32);
        y = affine_apply(step, y);
        v.z = out_word((uint32_t)(y >> 32), F32);
        y = affine_apply(step, y);
        v.w = out_word((uint32_t)(y >> 32), F32);
        if (vec_ok) {
            __stcs(reinterpret_cast<uint4 *>(row + j), v);
        } else {
            row[j] = v.x;
            if (j + 1 < n) row[j + 1] = v.y;
            if (j + 2 < n) row[j + 2] = v.z;
            if (j + 3 < n) row[j + 3] = v.w;
        }
        x = affine_apply(leap, x);
    }
}

static cudaError_t launch_lcg_intra(const Gen &g, void *d_out, uint64_t n, bool f32, cudaStream_t st)
{
    if (g.S > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    // small grids (this path is chosen for few streams) are launch-bound: programmatic dependent launch
    PdlLaunch pl(dim3((unsigned)g.S), dim3(256), 0, st, g.S * 256ull <= kPdlMaxThreads);
    uint32_t *o = (uint32_t *)d_out;
    const cudaError_t e = f32 ? cudaLaunchKernelEx(&pl.cfg, lcg_intra_fill_kernel<true>, g, o, n)
                              : cudaLaunchKernelEx(&pl.cfg, lcg_intra_fill_kernel<false>, g, o, n);
    count_launch();
    return e != cudaSuccess ? e : cudaGetLastError();
}

static int sm_count()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) cudaGetLastError();
    return sm_count(dev);
}

template <int KIND>
static cudaError_t launch_rowtile(const Gen &g, void *d_out, uint64_t n, bool f32, int variant, cudaStream_t st)
{
    const uint64_t warps = (g.S + 31) / 32;
    const uint64_t grid = (warps + FILL_WARPS - 1) / FILL_WARPS;
    if (grid > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    uint32_t *o = (uint32_t *)d_out;
    // variant "store": 0 = automatic (64-draw tiles for rows of at least 64 draws), 1 = 32-draw tiles, 2 = 64-draw tiles
    const bool wide = variant == 2 || (variant == 0 && n >= 64);
#define ROWTILE(KT)                                                                                   \
    do {                                                                                              \
        if (f32) rowtile_fill_kernel<KIND, true, KT><<<(unsigned)grid, FILL_WARPS * 32, 0, st>>>(g, o, n); \
        else rowtile_fill_kernel<KIND, false, KT><<<(unsigned)grid, FILL_WARPS * 32, 0, st>>>(g, o, n);    \
    } while (0)
    if (wide) ROWTILE(64);
    else ROWTILE(32);
#undef ROWTILE
    count_launch();
    return cudaGetLastError();
}

template <bool F32, int U, int T, int R, int CVT = 0>
static cudaError_t launch_philox_warp(const Gen &g, uint32_t *o, uint64_t n, uint64_t blocks_per_row, cudaStream_t st,
                                      bool one_shot = false)
{
    const uint64_t tpr = (blocks_per_row + 32 * U * T - 1) / (32 * U * T);
    const uint64_t n_tiles = g.S * tpr;
    // persistent grid: a multiple of the SM count; 8 warps per CTA, CTAs resident per SM by registers
    static int per_sm = 0; // a property of the kernel on sm_100a; the same on every device this library targets
    if (!per_sm) {
        int b = 0;
        cudaError_t e =
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, philox_fill_warp_kernel<F32, U, T, R, false, CVT>, 256, 0);
        if (e != cudaSuccess) return e;
        per_sm = b > 0 ? b : 1;
    }
    uint64_t grid = (uint64_t)sm_count() * per_sm;
    const uint64_t need = (n_tiles + 7) / 8;
    if (grid > need || (one_shot && need <= 0x7fffffffull)) grid = need; // one_shot: one tile per warp, CTAs handed out by the hardware
    const uint64_t b0 = g.draws_done >> 2;
    // every tile full, and the call's blocks share the high counter word: the lean per-tile path
    const bool allfast = blocks_per_row % (32 * U * T) == 0 && (b0 >> 32) == ((b0 + blocks_per_row - 1) >> 32);
    if (allfast)
        philox_fill_warp_kernel<F32, U, T, R, true, CVT><<<(unsigned)grid, 256, 0, st>>>(o, g.first, g.seed, b0, n,
                                                                              (uint32_t)blocks_per_row, (uint32_t)tpr, n_tiles);
    else
        philox_fill_warp_kernel<F32, U, T, R, false, CVT><<<(unsigned)grid, 256, 0, st>>>(o, g.first, g.seed, b0, n,
                                                                               (uint32_t)blocks_per_row, (uint32_t)tpr, n_tiles);
    count_launch();
    return cudaGetLastError();
}

template <int R>
static cudaError_t launch_philox_fill(const Gen &g, void *d_out, uint64_t n, bool f32, int variant, int cvt,
                                      cudaStream_t st)
{
    const uint64_t d0 = g.draws_done;
    const uint64_t blocks_per_row = ((d0 + n - 1) >> 2) - (d0 >> 2) + 1;
    const bool aligned = ((d0 | n) & 3ull) == 0ull;
    uint32_t *o = (uint32_t *)d_out;
    if (aligned && blocks_per_row <= 0x7fffffffull) {
#define PW(U, T) (f32 ? launch_philox_warp<true, U, T, R>(g, o, n, blocks_per_row, st) \
                      : launch_philox_warp<false, U, T, R>(g, o, n, blocks_per_row, st))
        if (f32 && variant == 0 && cvt >= 1 && cvt <= 3) { // variant "cvt": the float map in another exact form
            switch (cvt) {
            case 1: return launch_philox_warp<true, 8, 1, R, 1>(g, o, n, blocks_per_row, st);
            case 2: return launch_philox_warp<true, 8, 1, R, 2>(g, o, n, blocks_per_row, st);
            default: return launch_philox_warp<true, 8, 1, R, 3>(g, o, n, blocks_per_row, st);
            }
        }
        // Grid: Philox4x32-10 is paced by its IMAD.WIDE arithmetic, every SM finishes its share at the same time and
        // the persistent grid wins (624 us against 700 us per 4 GiB with one CTA per 8 tiles); the 7-round variant
        // is store-bound, where a static split waits for the SMs that get the smaller share of the write bandwidth
        // (DESIGN.md 6.4): one short-lived CTA per 8 tiles, handed out by the hardware, 690 -> 568 us = 7.56 TB/s.
        // variant "store": 3 = one-shot CTAs, 4 = persistent grid, whatever R.
        const bool one_shot = variant == 3 || (variant != 4 && R < 10);
        switch (variant) { // identical bits; (U, T) = blocks interleaved per lane, groups per tile
        case 1: return PW(4, 2);
        case 2: return PW(2, 4);
        default: return f32 ? launch_philox_warp<true, 8, 1, R>(g, o, n, blocks_per_row, st, one_shot)
                            : launch_philox_warp<false, 8, 1, R>(g, o, n, blocks_per_row, st, one_shot);
        }
#undef PW
    }
    // general path: any draw offset / any n, word-by-word stores with bounds checks
    constexpr int U = 4;
    const uint64_t tpr = (blocks_per_row + 256 * U - 1) / (256 * U);
    if (tpr > 0xffffffffull) return cudaErrorInvalidConfiguration;
    const uint64_t n_tiles = g.S * tpr;
    uint64_t grid = (uint64_t)sm_count() * 8ull;
    if (grid > n_tiles) grid = n_tiles;
    if (f32)
        philox_fill_kernel<true, false, U, R><<<(unsigned)grid, 256, 0, st>>>(o, g.S, g.first, g.seed, d0, n, blocks_per_row,
                                                                          (uint32_t)tpr, n_tiles);
    else
        philox_fill_kernel<false, false, U, R><<<(unsigned)grid, 256, 0, st>>>(o, g.S, g.first, g.seed, d0, n, blocks_per_row,
                                                                           (uint32_t)tpr, n_tiles);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_fill(const rng_handle &h, void *d_out, uint64_t n, bool f32, cudaStream_t st)
{
    const Gen &g = h.g;
    if (g.kind == RNG_LCG64 || g.kind == RNG_LCG64_LEAPFROG) {
        // variant "lcg": 0 = automatic, 1 = one thread per stream (row tiles), 2 = one CTA per stream
        const bool few = g.S < 65536ull && n >= 512ull;
        if (h.var_lcg == 2 || (h.var_lcg == 0 && few)) return launch_lcg_intra(g, d_out, n, f32, st);
    }
    switch (g.kind) {
    case RNG_LCG64: return launch_rowtile<RNG_LCG64>(g, d_out, n, f32, h.var_store, st);
    case RNG_LCG64_LEAPFROG: return launch_rowtile<RNG_LCG64_LEAPFROG>(g, d_out, n, f32, h.var_store, st);
    case RNG_XORWOW: return launch_rowtile<RNG_XORWOW>(g, d_out, n, f32, h.var_store, st);
    case RNG_XS1024W:
        if (h.var_xs1024 == 64) return launch_rowtile<RNG_XS1024W>(g, d_out, n, f32, h.var_store, st);
        return launch_xs1024_fill(h, d_out, n, f32, st);
    case RNG_PHILOX4X32_10: return launch_philox_fill<10>(g, d_out, n, f32, h.var_store, h.var_cvt, st);
    case RNG_PHILOX4X32_7: return launch_philox_fill<7>(g, d_out, n, f32, h.var_store, h.var_cvt, st);
    case RNG_LCG32: return launch_rowtile<RNG_LCG32>(g, d_out, n, f32, h.var_store, st);
    case RNG_LCG64_BOTH: return launch_rowtile<RNG_LCG64_BOTH>(g, d_out, n, f32, h.var_store, st);
    case RNG_LCG32_LEAPFROG: return launch_rowtile<RNG_LCG32_LEAPFROG>(g, d_out, n, f32, h.var_store, st);
    case RNG_MWC: return launch_rowtile<RNG_MWC>(g, d_out, n, f32, h.var_store, st);
    case RNG_MWC_MULTI: return launch_rowtile<RNG_MWC_MULTI>(g, d_out, n, f32, h.var_store, st);
    case RNG_LFIB521:
    case RNG_LFIB1279: return launch_lfib_fill(g, d_out, n, f32, h.var_store, st);
    default: return cudaErrorInvalidValue;
    }
}

} // namespace rngb200
