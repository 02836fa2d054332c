// fill_xs1024.cu -- fill and in-register draw kernels of the paper's XORShift1024/Weyl
// generator for an instance spread
// over P = 32/K lanes (xs1024.cuh).  Results are identical for every K; K is a measurement
// knob (rng_set_variant("xs1024", K)), the default is chosen per mode from B200 measurements
// (DESIGN.md section 6).
//
// Streams 32g..32g+31 are the words of instance g (R-D4), so lane l of a warp that hosts K
// instances owns the K consecutive rows K*l .. K*l+K-1 of the warp's 32K rows: state loads
// and stores are one contiguous K-word access per lane.
//
// Fill mode writes stream-major rows, so a row only becomes a full 128-byte line after 32
// updates of its instance.  The warp therefore stages a [32K rows][32 draws] tile in shared
// memory and writes whole lines (a B200 microbenchmark of the alternative -- each thread
// storing 32-byte row pieces directly -- reaches only 1.4 TB/s: partially written lines get
// evicted from L2).  See xs1024_fill_kernel for the tile layout and the TMA bulk-store write-out.
#include <cstring>

#include <cuda.h>

#include "internal.h"
#include "xs1024.cuh"

namespace rngb200 {

// ---- TMA tensor store of a staged tile (shared -> global) ----
__device__ __forceinline__ void tma_store_3d(const CUtensorMap *tm, const uint32_t *ssrc, int c0, int c1, int c2)
{
    const uint32_t saddr = (uint32_t)__cvta_generic_to_shared(ssrc);
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(tm), "r"(saddr),
                 "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void fence_generic_to_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read_all() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }

// Tile layout (per warp, 1 KiB aligned): row r = K*lane + j of the warp's 32K rows sits in
// slot j*32 + lane; a slot is 128 dense bytes = the row's 32 draws; its eight 16-byte chunks
// are XOR-swizzled with slot & 7 = lane & 7.  The generating 128-bit stores of a quarter-warp
// then hit eight different bank groups, the write-out loads (eight lanes -> the eight chunks
// of one row) are conflict-free, and the layout is exactly TMA's SWIZZLE_128B box of a
// rank-3 tensor map over the output with dimensions (draw, row / K, row % K).
// TMA: lane 0 hands the whole tile to the TMA unit with ONE cp.async.bulk.tensor (shared ->
// global; columns past n and rows past S are clipped by the unit, so ragged tiles need no
// special case) and the warp goes on generating; it waits for the copy to have READ the tile
// only just before overwriting it.  No LDS/STG write-out at all.
// !TMA (and rows that are not 16-byte aligned, n % 4 != 0): LDS.128 + streaming STG.128.
template <int K, bool F32, int WARPS, bool TMA>
__global__ void __launch_bounds__(WARPS * 32)
    xs1024_fill_kernel(Gen g, uint32_t *__restrict__ out, uint64_t n, const __grid_constant__ CUtensorMap tmap)
{
    extern __shared__ __align__(1024) uint32_t xs_tiles[];
    constexpr int P = 32 / K;
    constexpr int ROWS = 32 * K;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *tile = xs_tiles + warp * (ROWS * 32);
    const uint64_t wg = (uint64_t)blockIdx.x * WARPS + warp;
    const uint64_t s0 = wg * (uint64_t)ROWS; // first row of this warp
    if (s0 >= g.S) return;                   // warp-uniform
    const int p = (P == 1) ? 0 : (lane & (P - 1));
    const uint64_t my0 = s0 + (uint64_t)K * lane; // S % 32 == 0 and K | 32: my K rows are all live or all dead
    const bool live = my0 < g.S;
    const uint32_t rows = (uint32_t)((g.S - s0 < (uint64_t)ROWS) ? (g.S - s0) : (uint64_t)ROWS);
    const bool vec_ok = (n & 3ull) == 0ull;
    uint32_t *state = (uint32_t *)g.state;

    uint32_t w[K];
#pragma unroll
    for (int j = 0; j < K; j++) w[j] = 0u;
    if (live) load_words<K>(state + my0, w);
    XsMasks<K> m;
    m.init(p);
    uint32_t nupd = (uint32_t)g.draws_done; // the Weyl term only needs the update count mod 2^32
    const uint32_t swz = (uint32_t)lane & 7u;
    uint32_t *myrows = tile + lane * 32; // + j * 32 * 32
    bool pending = false;               // a tensor store may still be reading the tile

    for (uint64_t j0 = 0; j0 < n; j0 += 32) {
        const uint32_t kk = (uint32_t)((n - j0 < 32ull) ? (n - j0) : 32ull);
        // ---- generate kk updates; lane writes draws of its K rows, four at a time ----
        uint32_t c = 0;
        for (; 4u * c + 4u <= kk; c++) {
            uint32_t o[K][4];
#pragma unroll
            for (int u = 0; u < 4; u++) {
                xs1024_update_k<K>(w, m);
                nupd++;
                const uint32_t wt = xs1024_weyl_term(nupd);
#pragma unroll
                for (int j = 0; j < K; j++) o[j][u] = out_word(wt + w[j], F32);
            }
            if (TMA && pending) { // warp-uniform
                if (lane == 0) bulk_wait_read_all();
                __syncwarp();
                pending = false;
            }
            const uint32_t phys = (c ^ swz) * 4u;
#pragma unroll
            for (int j = 0; j < K; j++)
                *reinterpret_cast<uint4 *>(myrows + j * 1024 + phys) = make_uint4(o[j][0], o[j][1], o[j][2], o[j][3]);
        }
        if (4u * c < kk) { // ragged tail of the call
            if (TMA && pending) {
                if (lane == 0) bulk_wait_read_all();
                __syncwarp();
                pending = false;
            }
            for (uint32_t u = 4u * c; u < kk; u++) {
                xs1024_update_k<K>(w, m);
                nupd++;
                const uint32_t wt = xs1024_weyl_term(nupd);
#pragma unroll
                for (int j = 0; j < K; j++) myrows[j * 1024 + ((u >> 2) ^ swz) * 4u + (u & 3u)] = out_word(wt + w[j], F32);
            }
        }
        if (TMA && vec_ok) {
            // ---- one tensor store for the whole tile: box (32 draws, 32 lanes, K words) ----
            fence_generic_to_async(); // my generic-proxy writes -> visible to the async proxy
            __syncwarp();
            if (lane == 0) {
                tma_store_3d(&tmap, tile, (int)j0, (int)(wg * 32ull), 0);
                bulk_commit();
            }
            pending = true;
            continue;
        }
        __syncwarp();
        // ---- write out: every warp instruction stores four complete 128-byte lines ----
        if (kk == 32u && vec_ok) {
            // lane -> chunk (lane & 7) of rows (lane >> 3), +4, +8, ...
            const uint32_t ch = (uint32_t)lane & 7u, r0 = (uint32_t)lane >> 3;
            uint32_t *gp = out + (s0 + r0) * n + j0 + 4u * ch;
            const uint64_t gstep = 4ull * n;
            if (rows == (uint32_t)ROWS) {
#pragma unroll 8
                for (int it = 0; it < 8 * K; it++) {
                    const uint32_t r = 4u * (uint32_t)it + r0;
                    const uint32_t slot = (r % K) * 32u + r / K;
                    const uint4 v = *reinterpret_cast<const uint4 *>(tile + slot * 32u + ((ch ^ (slot & 7u)) * 4u));
                    __stcs(reinterpret_cast<uint4 *>(gp), v);
                    gp += gstep;
                }
            } else {
                for (uint32_t r = r0; r < rows; r += 4u, gp += gstep) {
                    const uint32_t slot = (r % K) * 32u + r / K;
                    const uint4 v = *reinterpret_cast<const uint4 *>(tile + slot * 32u + ((ch ^ (slot & 7u)) * 4u));
                    __stcs(reinterpret_cast<uint4 *>(gp), v);
                }
            }
        } else {
            for (uint32_t r = 0; r < rows; r++) {
                const uint32_t slot = (r % K) * 32u + r / K;
                for (uint32_t q = lane; q < kk; q += 32)
                    out[(s0 + r) * n + j0 + q] = tile[slot * 32u + (((q >> 2) ^ (slot & 7u)) * 4u) + (q & 3u)];
            }
        }
        __syncwarp();
    }
    if (live) store_words<K>(state + my0, w);
    if (TMA && pending && lane == 0) bulk_wait_read_all(); // the tile must outlive the copy that reads it
}

// ---- the fill kernel of the TMA path: persistent warps that draw their work from a ticket counter ----
// One CTA per SM for the whole call; a warp processes items (an item = the K instances = 32K rows that one warp
// hosts) until the tickets run out.  What this buys over one short-lived CTA per item (xs1024_fill_kernel<.., TMA =
// true>, kept for comparison as variant "xsfill" 1):
//   * the next item's state (K words per lane) is loaded while the current item is generated, so no warp sits on a
//     global-load latency while holding 16 KiB of shared memory;
//   * with NT = 2 tiles per warp the TMA unit reads tile A while the warp generates into tile B
//     (cp.async.bulk.wait_group.read NT-1 before a tile is reused);
//   * there is no CTA tail waiting for its last copy per item, only one per call.
// With n = 64 per call (C4: 64 calls of 64 draws, the 4 GiB buffer holds no more) an item is just two tiles, so
// these per-item costs were a large share of a warp's life.
// Work distribution is DYNAMIC (atomic ticket per item, fetched one item ahead so that its latency and the state
// load hide behind the generation): at the HBM limit the SMs of a B200 do not all get the same share of the write
// bandwidth, and a static "item += number of warps" split waits for the slowest SM -- the bare store pattern of
// this kernel runs at 5.9 TB/s with the static split and at 7.0-7.3 TB/s with tickets, which is what a grid of
// one-shot CTAs gets from the hardware's own CTA scheduler (B200 microbenchmark).
// Tickets: *ticket is zero between launches.  Tickets 0 .. n_items-1 are the items; every warp takes exactly one
// ticket beyond that range before it leaves, so the launch hands out n_items + (number of warps) tickets in all, and
// the warp that draws the very last one knows that no other atomic on the counter is still to come: it puts the
// counter back to zero.  A launch therefore depends on nothing the host remembers about earlier launches (a launch
// that never runs, or a captured launch replayed any number of times, leaves the counter as it found it).
template <int K, bool F32, int WARPS, int NT>
__global__ void __launch_bounds__(WARPS * 32, 1)
    xs1024_fill_persistent_kernel(Gen g, uint64_t n, const __grid_constant__ CUtensorMap tmap,
                                  unsigned long long *__restrict__ ticket)
{
    extern __shared__ uint32_t xs_tiles_raw[];
    constexpr int P = 32 / K;
    constexpr int ROWS = 32 * K;
    constexpr uint32_t TILE_WORDS = ROWS * 32;
    // SWIZZLE_128B wants the box 1 KiB aligned in shared memory (an offset into the array, so that the pointer
    // keeps its address space and the tile stores stay STS)
    const uint32_t pad = (1024u - ((uint32_t)__cvta_generic_to_shared(xs_tiles_raw) & 1023u)) & 1023u;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *tiles = xs_tiles_raw + (pad >> 2) + (uint32_t)warp * (NT * TILE_WORDS);
    const uint64_t n_items = (g.S + ROWS - 1) / ROWS;
    const int p = (P == 1) ? 0 : (lane & (P - 1));
    uint32_t *state = (uint32_t *)g.state;
    XsMasks<K> m;
    m.init(p);
    const uint32_t swz = (uint32_t)lane & 7u;
    const uint32_t nupd0 = (uint32_t)g.draws_done;
    uint32_t tcount = 0; // tiles handed to the TMA unit so far (all by lane 0 of this warp)

    // One ticket per item: handing out chunks of 2..16 consecutive items per ticket measured 4-15 % SLOWER (the
    // items being written at any moment then spread over a proportionally wider address window).
    auto take = [&]() -> uint64_t { // warp-uniform next item
        unsigned long long v = 0ull;
        if (lane == 0) {
            v = atomicAdd(ticket, 1ull);
            if (v == n_items + (uint64_t)gridDim.x * WARPS - 1ull) atomicExch(ticket, 0ull); // the last ticket of the launch
        }
        return __shfl_sync(0xffffffffu, v, 0);
    };
    uint32_t w[K], wn[K];
    uint64_t item = take();
    if (item >= n_items) return;
    {
        const uint64_t my0 = item * ROWS + (uint64_t)K * lane;
#pragma unroll
        for (int j = 0; j < K; j++) wn[j] = 0u;
        if (my0 < g.S) load_words<K>(state + my0, wn);
    }
    while (item < n_items) {
        const uint64_t my0 = item * ROWS + (uint64_t)K * lane;
        const bool live = my0 < g.S;
#pragma unroll
        for (int j = 0; j < K; j++) w[j] = wn[j];
        const uint64_t next = take();
        { // prefetch the next item's state
            const uint64_t nx = next * ROWS + (uint64_t)K * lane;
#pragma unroll
            for (int j = 0; j < K; j++) wn[j] = 0u;
            if (next < n_items && nx < g.S) load_words<K>(state + nx, wn);
        }
        uint32_t nupd = nupd0;
        for (uint64_t j0 = 0; j0 < n; j0 += 32) {
            const uint32_t kk = (uint32_t)((n - j0 < 32ull) ? (n - j0) : 32ull); // a multiple of 4 (n % 4 == 0)
            uint32_t *tile = tiles + (NT == 1 ? 0u : (tcount % NT) * TILE_WORDS);
            uint32_t *myrows = tile + lane * 32;
            for (uint32_t c = 0; 4u * c < kk; c++) {
                uint32_t o[K][4];
#pragma unroll
                for (int u = 0; u < 4; u++) {
                    xs1024_update_k<K>(w, m);
                    nupd++;
                    const uint32_t wt = xs1024_weyl_term(nupd);
#pragma unroll
                    for (int j = 0; j < K; j++) o[j][u] = out_word(wt + w[j], F32);
                }
                if (c == 0 && tcount >= NT) { // the copy that last read this tile must be done reading it
                    if (lane == 0) asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(NT - 1) : "memory");
                    __syncwarp();
                }
                const uint32_t phys = (c ^ swz) * 4u;
#pragma unroll
                for (int j = 0; j < K; j++)
                    *reinterpret_cast<uint4 *>(myrows + j * 1024 + phys) = make_uint4(o[j][0], o[j][1], o[j][2], o[j][3]);
            }
            fence_generic_to_async(); // my generic-proxy writes -> visible to the async proxy
            __syncwarp();
            if (lane == 0) {
                tma_store_3d(&tmap, tile, (int)j0, (int)(item * 32ull), 0);
                bulk_commit();
            }
            tcount++;
        }
        if (live) store_words<K>(state + my0, w);
        item = next;
    }
    if (lane == 0) bulk_wait_read_all(); // the tiles must outlive the copies that read them
}

// In-register draw mode (row a6): {xor, sum} of n draws per stream.  The Weyl term is the
// same for every word, so its sum is accumulated once per update and added at the end.
template <int K, int THREADS>
__global__ void __launch_bounds__(THREADS) xs1024_draw_kernel(Gen g, uint32_t *__restrict__ out, uint64_t n)
{
    constexpr int P = 32 / K;
    constexpr int ROWS = 32 * K;
    const int lane = threadIdx.x & 31;
    const uint64_t wg = ((uint64_t)blockIdx.x * THREADS + threadIdx.x) >> 5;
    const uint64_t s0 = wg * (uint64_t)ROWS;
    if (s0 >= g.S) return; // warp-uniform
    const int p = (P == 1) ? 0 : (lane & (P - 1));
    const uint64_t my0 = s0 + (uint64_t)K * lane;
    const bool live = my0 < g.S;
    uint32_t *state = (uint32_t *)g.state;
    uint32_t w[K], x[K], sm[K];
#pragma unroll
    for (int j = 0; j < K; j++) w[j] = 0u, x[j] = 0u, sm[j] = 0u;
    if (live) load_words<K>(state + my0, w);
    XsMasks<K> m;
    m.init(p);
    uint32_t nupd = (uint32_t)g.draws_done, wsum = 0u;
#pragma unroll 1
    for (uint64_t i = 0; i < n; i++) {
        xs1024_update_k<K>(w, m);
        nupd++;
        const uint32_t wt = xs1024_weyl_term(nupd);
        wsum += wt;
#pragma unroll
        for (int j = 0; j < K; j++) {
            x[j] ^= wt + w[j];
            sm[j] += w[j];
        }
    }
    if (live) {
        store_words<K>(state + my0, w);
        uint32_t o[2 * K];
#pragma unroll
        for (int j = 0; j < K; j++) o[2 * j] = x[j], o[2 * j + 1] = sm[j] + wsum;
        store_words<2 * K>(out + 2ull * my0, o);
    }
}

// The A/B partner of xs1024_draw_kernel<1, ..>: the same one-word-per-thread layout with the exchange through
// shared memory, i.e. the paper's Listing 1 as it has to be written since Volta -- its padded
// per-warp array (zeros on both sides stand for the words shifted in from outside the state),
// with __syncwarp() wherever the listing relies on implicit warp synchrony and `volatile` (footnote 3,
// PAPER.md:189, expects shuffles to replace it).  Variant "xs1024" = 33, draw mode only; same bits as every other
// layout.  Measured against the shuffle form in DESIGN.md section 8.
template <int THREADS>
__global__ void __launch_bounds__(THREADS) xs1024_draw_smem_kernel(Gen g, uint32_t *__restrict__ out, uint64_t n)
{
    constexpr int PAD = 11, ROW = PAD + 32 + PAD;
    __shared__ uint32_t rows[THREADS / 32][ROW];
    const int lane = threadIdx.x & 31;
    const uint64_t wg = ((uint64_t)blockIdx.x * THREADS + threadIdx.x) >> 5;
    const uint64_t s0 = wg * 32ull;
    if (s0 >= g.S) return; // warp-uniform (S is a multiple of 32)
    uint32_t *r = rows[threadIdx.x >> 5] + PAD; // r[-11 .. -1] and r[32 .. 42] stay zero
    if (lane < PAD) r[-1 - lane] = 0u, r[32 + lane] = 0u;
    uint32_t *state = (uint32_t *)g.state;
    uint32_t v = state[s0 + lane], x = 0u, sum = 0u, wsum = 0u;
    r[lane] = v;
    __syncwarp();
    uint32_t nupd = (uint32_t)g.draws_done;
#pragma unroll 1
    for (uint64_t i = 0; i < n; i++) {
        uint32_t a = r[lane + 10], b = r[lane + 11]; // A: X ^= X << 329
        __syncwarp();
        v ^= (a << 9) | (b >> 23);
        r[lane] = v;
        __syncwarp();
        a = r[lane - 10], b = r[lane - 11];          // B: X ^= X >> 347
        __syncwarp();
        v ^= (a >> 27) | (b << 5);
        r[lane] = v;
        __syncwarp();
        a = r[lane + 10], b = r[lane + 11];          // C: X ^= X << 344
        __syncwarp();
        v ^= (a << 24) | (b >> 8);
        r[lane] = v;
        __syncwarp();
        nupd++;
        const uint32_t wt = xs1024_weyl_term(nupd);
        wsum += wt;
        x ^= wt + v;
        sum += v;
    }
    state[s0 + lane] = v;
    reinterpret_cast<uint2 *>(out)[s0 + lane] = make_uint2(x, sum + wsum);
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        else
            cudaGetLastError();
    }
    return fn;
}

// rank-3 view of the stream-major output out[row*n + draw], row = K*l + j:
// dimensions (draw: n, l: S/K, j: K), box (32, 32, K), SWIZZLE_128B
static bool make_out_tensor_map(CUtensorMap *tm, uint32_t *out, uint64_t S, uint64_t n, int K)
{
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc || (n & 3ull) || n > 0xffffffffull || ((uintptr_t)out & 15u)) return false;
    const cuuint64_t dims[3] = {n, S / (uint64_t)K, (cuuint64_t)K};
    const cuuint64_t strides[2] = {(cuuint64_t)K * n * 4ull, n * 4ull};
    if (strides[0] >= (1ull << 40)) return false;
    const cuuint32_t box[3] = {32u, 32u, (cuuint32_t)K};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT32, 3, out, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) ==
           CUDA_SUCCESS;
}

template <int K, int WARPS, bool TMA>
static cudaError_t launch_xs_fill(const Gen &g, uint32_t *o, uint64_t n, bool f32, const CUtensorMap &tm, cudaStream_t st)
{
    constexpr size_t smem = (size_t)WARPS * 32 * K * 32 * 4;
    const uint64_t inst = g.S / 32, warps = (inst + K - 1) / K, grid = (warps + WARPS - 1) / WARPS;
    if (grid > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    if (smem > 48 * 1024) { // per device and cheap: set on every launch rather than behind a per-process flag
        const cudaError_t e = f32 ? cudaFuncSetAttribute(xs1024_fill_kernel<K, true, WARPS, TMA>,
                                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
                                  : cudaFuncSetAttribute(xs1024_fill_kernel<K, false, WARPS, TMA>,
                                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    if (f32) xs1024_fill_kernel<K, true, WARPS, TMA><<<(unsigned)grid, WARPS * 32, smem, st>>>(g, o, n, tm);
    else xs1024_fill_kernel<K, false, WARPS, TMA><<<(unsigned)grid, WARPS * 32, smem, st>>>(g, o, n, tm);
    count_launch();
    return cudaGetLastError();
}

template <int K, int WARPS, int NT>
static cudaError_t launch_xs_fill_persistent(const rng_handle &h, uint64_t n, bool f32, const CUtensorMap &tm, int sms,
                                             cudaStream_t st)
{
    const Gen &g = h.g;
    constexpr size_t smem = (size_t)WARPS * NT * 32 * K * 32 * 4 + 1024; // + alignment slack
    static_assert(smem <= 227 * 1024, "tiles exceed the shared memory of a CTA");
    const uint64_t items = (g.S + 32 * K - 1) / (32 * K);
    uint64_t grid = (items + WARPS - 1) / WARPS;
    if (grid > (uint64_t)sms) grid = (uint64_t)sms;
    auto kf = xs1024_fill_persistent_kernel<K, true, WARPS, NT>;
    auto ku = xs1024_fill_persistent_kernel<K, false, WARPS, NT>;
    // unconditional (cheap; a per-process flag would be wrong with more than one device)
    cudaError_t e = cudaFuncSetAttribute(f32 ? kf : ku, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    unsigned long long *tk = (unsigned long long *)h.ticket;
    if (f32) kf<<<(unsigned)grid, WARPS * 32, smem, st>>>(g, n, tm, tk);
    else ku<<<(unsigned)grid, WARPS * 32, smem, st>>>(g, n, tm, tk);
    count_launch();
    return cudaGetLastError();
}

// variant "xs1024" = K (0: default); variant "store": 0 = default, 1 = LDS/STG write-out, 2 = TMA tensor store;
// variant "xsfill" (TMA path only): 0 = by row length (below), 1 = one short-lived warp per item (round 1's
// kernel), 2 = persistent warps with one tile each, 3 = persistent warps with two ping-pong tiles each.
// Default by row length n, from 4 GiB fills on a B200 (K = 4; TB/s for variants 1 / 2 / 3):
//   n = 64: 5.70 / 6.16 / 4.00    n = 128: 5.52 / 6.02 / 3.99    n = 256: 5.04 / 4.85 / 4.29
//   n = 1024: 4.70 / 4.28 / 4.64  n = 4096: 3.47 / 3.36 / 4.83
// (short rows: the tiles of a warp complete whole rows at once and more warps matter; long rows: the next 128
// bytes of a row should follow quickly, which the second tile does)
cudaError_t launch_xs1024_fill(const rng_handle &h, void *d_out, uint64_t n, bool f32, cudaStream_t st)
{
    uint32_t *o = (uint32_t *)d_out;
    const int K = (h.var_xs1024 == 1 || h.var_xs1024 == 2 || h.var_xs1024 == 8 || h.var_xs1024 == 16) ? h.var_xs1024 : 4;
    alignas(64) CUtensorMap tm;
    memset(&tm, 0, sizeof tm);
    const bool tma = h.var_store != 1 && make_out_tensor_map(&tm, o, h.g.S, n, K);
    const int mode = h.var_xsfill >= 1 && h.var_xsfill <= 3 ? h.var_xsfill : n <= 128 ? 2 : n < 2048 ? 1 : 3;
    if (tma && mode != 1) {
        const int sms = sm_count(h.device);
        const bool pp = mode == 3;
        // warps per CTA = what 224 KiB of tiles allow
        switch (K) {
        case 1: return pp ? launch_xs_fill_persistent<1, 28, 2>(h, n, f32, tm, sms, st)
                          : launch_xs_fill_persistent<1, 32, 1>(h, n, f32, tm, sms, st);
        case 2: return pp ? launch_xs_fill_persistent<2, 14, 2>(h, n, f32, tm, sms, st)
                          : launch_xs_fill_persistent<2, 28, 1>(h, n, f32, tm, sms, st);
        case 8: return pp ? launch_xs_fill_persistent<8, 3, 2>(h, n, f32, tm, sms, st)
                          : launch_xs_fill_persistent<8, 7, 1>(h, n, f32, tm, sms, st);
        case 16: return launch_xs_fill_persistent<16, 3, 1>(h, n, f32, tm, sms, st);
        default: return pp ? launch_xs_fill_persistent<4, 7, 2>(h, n, f32, tm, sms, st)
                           : launch_xs_fill_persistent<4, 14, 1>(h, n, f32, tm, sms, st);
        }
    }
#define XSF(KK, WARPS) \
    (tma ? launch_xs_fill<KK, WARPS, true>(h.g, o, n, f32, tm, st) : launch_xs_fill<KK, WARPS, false>(h.g, o, n, f32, tm, st))
    switch (K) {
    case 1: return XSF(1, 8);
    case 2: return XSF(2, 4);
    case 8: return XSF(8, 2);
    case 16: return XSF(16, 1);
    default: return XSF(4, 2);
    }
#undef XSF
}

template <int K, int THREADS>
static cudaError_t launch_xs_draw(const Gen &g, uint32_t *o, uint64_t n, cudaStream_t st)
{
    const uint64_t inst = g.S / 32, warps = (inst + K - 1) / K, wpc = THREADS / 32, grid = (warps + wpc - 1) / wpc;
    if (grid > 0x7fffffffull) return cudaErrorInvalidConfiguration;
    xs1024_draw_kernel<K, THREADS><<<(unsigned)grid, THREADS, 0, st>>>(g, o, n);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_xs1024_draw(const rng_handle &h, uint32_t *d_out, uint64_t n, cudaStream_t st)
{
    // the API asks for 8-byte alignment only; K >= 2 stores 16-byte vectors
    if (((uintptr_t)d_out & 15u) != 0u) return launch_xs_draw<1, 256>(h.g, d_out, n, st);
    switch (h.var_xs1024) {
    case 33: { // K = 1 with the paper's shared-memory exchange (measurement partner of case 1)
        const uint64_t grid = (h.g.S / 32 + 7) / 8;
        if (grid > 0x7fffffffull) return cudaErrorInvalidConfiguration;
        xs1024_draw_smem_kernel<256><<<(unsigned)grid, 256, 0, st>>>(h.g, d_out, n);
        count_launch();
        return cudaGetLastError();
    }
    case 1: return launch_xs_draw<1, 256>(h.g, d_out, n, st);
    case 2: return launch_xs_draw<2, 256>(h.g, d_out, n, st);
    case 4: return launch_xs_draw<4, 256>(h.g, d_out, n, st);
    case 8: return launch_xs_draw<8, 128>(h.g, d_out, n, st);
    case 16: return launch_xs_draw<16, 128>(h.g, d_out, n, st);
    case 0:
    case 32:
    default: return launch_xs_draw<32, 128>(h.g, d_out, n, st);
    }
}

} // namespace rngb200
