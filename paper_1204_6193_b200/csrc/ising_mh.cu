// ising_mh.cu -- the paper's own consumer kernel: double-checkerboard Metropolis with multi-hit
// updates (PAPER.md:56 "a double checkerboard decomposition", :58 "updating the spins of a tile
// once (k = 1) ... two random numbers are produced per state load and save operation ... multi-hit
// updates (k = 100), 200 random numbers are produced per access to global memory"; the kernel is
// described in Refs.[13,25], the order used here is reading R-E9 of DESIGN.md).
//
//   The lattice is cut into T x T tiles; tile (tx, ty) has coarse colour (tx+ty)&1.  A sweep is
//   coarse colour 0, then 1; one launch per coarse colour, one CTA of T*T/2 threads per tile of that
//   colour.  The CTA loads its tile and the one-site halo around it into shared memory (the halo
//   belongs to resting tiles of the other coarse colour), every thread loads ITS generator state
//   once, and the tile receives k hits: a hit = all sites of fine colour 0, barrier, all sites of
//   fine colour 1, barrier.  Thread t owns the horizontal domino (2 xh, 2 xh + 1) of row y_l,
//   t = y_l T/2 + xh, i.e. one site of each fine colour, and keeps both spins in registers; the
//   three foreign neighbours of a site come from shared memory.  Stream s = p T*T/2 + t for tile
//   number p = ty (L/T/2) + txh of either coarse colour (S = L*L/4 streams, one per thread, as in the
//   paper: 1024^2 sites <-> 262144 threads); a stream spends its draws in the order
//   (coarse colour, hit, fine colour).  2k draws per state load: the paper's k = 1 and k = 100
//   columns of Table 1 are this kernel with k_hits = 1 and 100.
// Acceptance as everywhere: flip iff (r >> 8) < T[(h+4)/2]  (exactly (float)(r>>8) 2^-24 < P).
// Product code (sm_100a); shares nothing with oracle/.
#include <atomic>

#include "internal.h"
#include "streams.cuh"

namespace rngb200 {

// A CTA hosts blockDim.x / (T*T/2) tiles, each in its own slab of shared memory (one tile per CTA in the plain case).
// WARP_TILE: tile = 8, a tile is exactly one warp (32 dominoes) and the two barriers of a hit are __syncwarp()
// instead of __syncthreads().  The lagged Fibonacci kinds share their ring among the 256 threads of a CTA
// (lfib.cuh), so their CTA hosts 256 / (T*T/2) tiles (T = 16: two, T = 8: eight) and keeps the block barriers:
// stream s = p T*T/2 + t is then blockIdx.x*256 + threadIdx.x, the instance <-> CTA map that generator needs.
template <int KIND, bool WARP_TILE>
__global__ void ising_multihit_kernel(Gen g, int8_t *__restrict__ sp, uint32_t L, IsingTable tab, uint32_t T,
                                      uint32_t k_hits, uint32_t C, uint32_t n_tiles)
{
    extern __shared__ __align__(16) int8_t mh_smem[]; // 16 words of thresholds, then the tile slab(s)
    // thresholds indexed by h + 4 (h = spin * neighbour sum, even): word address = 4 h + const, one IMAD
    uint32_t *thr = reinterpret_cast<uint32_t *>(mh_smem);
    for (uint32_t i = threadIdx.x; i < 5u; i += blockDim.x) thr[2u * i] = tab.T[i]; // a 2 x 2 tile has 2 threads
    // Programmatic dependent launch: this grid may have been scheduled while the previous half-sweep was still
    // draining; everything above is independent of it, everything below (spins, generator state) is not.
    // Let the next launch be scheduled right away: it waits at the same point for THIS grid to complete.
    pdl_entry();
    const uint32_t RS = T + 8u, half = T >> 1;
    // (T+2) rows of RS bytes; interior row y_l at row y_l+1, columns 4 .. 4+T-1, halo columns 3 and 4+T
    const uint32_t tile_threads = half * T;
    const uint32_t sub = WARP_TILE ? (threadIdx.x >> 5) : threadIdx.x / tile_threads; // tile of this CTA
    int8_t *tile = mh_smem + 64 + sub * (((T + 2u) * RS + 15u) & ~15u);
    const uint32_t t = threadIdx.x - sub * tile_threads;
    const uint32_t nth = (L / T) >> 1;
    const uint32_t p = blockIdx.x * (blockDim.x / tile_threads) + sub;
    const bool tile_live = p < n_tiles; // warp-uniform; dead warps still take part in the CTA barrier below
    if (WARP_TILE && !tile_live) {
        __syncthreads();
        return;
    }
    const uint32_t ty = p / nth, txh = p - ty * nth;
    const uint32_t tx = 2u * txh + ((ty + C) & 1u);
    const uint32_t x0 = tx * T, y0 = ty * T; // tile origin (both even: local parity = global parity)
    const uint32_t yl = t / half, xh = t - yl * half;

    // ---- load: own domino (also kept in registers), then the halo by the first T threads ----
    int8_t *grow = sp + (uint64_t)(y0 + yl) * L + x0 + 2u * xh;
    const uint16_t dom = *reinterpret_cast<const uint16_t *>(grow);
    int8_t *mine = tile + (yl + 1u) * RS + 4u + 2u * xh;
    *reinterpret_cast<uint16_t *>(mine) = dom;
    if (t < T) {
        const uint32_t yu = y0 ? y0 - 1u : L - 1u, yd = (y0 + T == L) ? 0u : y0 + T;
        const uint32_t xl = x0 ? x0 - 1u : L - 1u, xr = (x0 + T == L) ? 0u : x0 + T;
        tile[0u * RS + 4u + t] = sp[(uint64_t)yu * L + x0 + t];
        tile[(T + 1u) * RS + 4u + t] = sp[(uint64_t)yd * L + x0 + t];
        tile[(t + 1u) * RS + 3u] = sp[(uint64_t)(y0 + t) * L + xl];
        tile[(t + 1u) * RS + 4u + T] = sp[(uint64_t)(y0 + t) * L + xr];
    }
    const uint64_t s = (uint64_t)p * tile_threads + t;
    Stream<KIND> gen;
    gen.load(g, s);
    __syncthreads(); // thresholds and tile(s) are in place
    auto hit_barrier = [&]() {
        if constexpr (WARP_TILE) __syncwarp();
        else __syncthreads();
    };

    // fine colour c site of the domino: x_l = 2 xh + ((y_l + c) & 1)
    const uint32_t par = yl & 1u;       // colour-0 site is byte `par` of the domino, colour-1 site byte 1-par
    int sa = (int)(int8_t)(par ? (dom >> 8) : (dom & 0xff));  // colour 0
    int sb = (int)(int8_t)(par ? (dom & 0xff) : (dom >> 8));  // colour 1
    const char *thr4 = reinterpret_cast<const char *>(thr) + 16; // + 4 h
    int8_t *pa = mine + par, *pb = mine + (1u - par);
    // foreign horizontal neighbour: the site beyond the domino on the side away from the partner
    const int da = par ? 1 : -1; // colour-0 site at byte par: partner on the other side
    for (uint32_t hit = 0; hit < k_hits; hit++) {
        {
            const int nn = sb + (int)pa[da] + (int)pa[-(int)RS] + (int)pa[RS];
            const uint32_t th = *reinterpret_cast<const uint32_t *>(thr4 + 4 * sa * nn);
            const uint32_t r = gen.next();
            if ((r >> 8) < th) {
                sa = -sa;
                *pa = (int8_t)sa;
            }
        }
        hit_barrier();
        {
            const int nn = sa + (int)pb[-da] + (int)pb[-(int)RS] + (int)pb[RS];
            const uint32_t th = *reinterpret_cast<const uint32_t *>(thr4 + 4 * sb * nn);
            const uint32_t r = gen.next();
            if ((r >> 8) < th) {
                sb = -sb;
                *pb = (int8_t)sb;
            }
        }
        hit_barrier();
    }
    gen.store(g, s);
    const uint32_t lo = (uint32_t)(uint8_t)(par ? sb : sa), hi = (uint32_t)(uint8_t)(par ? sa : sb);
    *reinterpret_cast<uint16_t *>(grow) = (uint16_t)(lo | (hi << 8));
}

// ---- the whole call in ONE launch: persistent tiles, generator state in registers, halos through inboxes ----------
// PAPER.md:58 defines the k = 1 column of Table 1 by what a tile visit costs besides its 2k draws: one generator
// state load and store, and (on any GPU) one kernel launch per coarse colour.  At 1024^2 a half-sweep is 0.3 us of
// arithmetic under a 4.6 us launch.  Here every tile of BOTH coarse colours stays in the shared memory of one CTA for
// all n_sweeps, every stream's state stays in the registers of its thread (a thread serves up to ROUNDS streams), and
// the only thing that crosses CTAs is the one-site halo: after its k hits a tile writes each of its four border lines
// as ONE 64-bit word {stage number : 20, T spin bits : up to 44} into the inbox of the neighbouring tile (four words
// = one 32-byte sector per tile), and a tile's next visit waits until the four words of its inbox carry the previous
// stage's number.  A single aligned 64-bit store carries data and flag together, so no fence, atomic or grid-wide
// barrier is needed.  Stage e = 2 sweep + colour + 1 needs the posts of stage e - 1; a poster cannot run ahead, because
// its own next visit needs this tile's post of stage e.  All CTAs must be co-resident (cooperative launch, one CTA
// per SM).  Measured on a B200: the CTA runs its tiles in lockstep (block barriers around the
// exchange) and ONE warp per CTA polls all inboxes with 16-byte loads -- letting every tile poll and proceed on its
// own (named barriers) was twice as slow, and __nanosleep in the poll loop sleeps for microseconds.
// Same trajectory as one launch per coarse colour (tests compare both with the oracle).
constexpr uint32_t kMhEpochBits = 20u; // stages per call < 2^20; T <= 44 spin bits below them

__device__ __forceinline__ void mh_post(unsigned long long *slot, unsigned long long v)
{
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(slot), "l"(v) : "memory");
}
__device__ __forceinline__ void mh_peek2(const unsigned long long *p, unsigned long long &a, unsigned long long &b)
{
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}

template <int KIND, int ROUNDS>
__global__ void __launch_bounds__(1024, 1)
    ising_multihit_coop_kernel(Gen g, int8_t *__restrict__ sp, uint32_t L, IsingTable tab, uint32_t T, uint32_t k_hits,
                               uint32_t n_sweeps, uint32_t n_pairs, unsigned long long *__restrict__ inbox)
{
    // 16 words of thresholds, the polled inbox words [round][slot][4], then the slabs [round][slot][colour]
    extern __shared__ __align__(16) int8_t mh_smem[];
    uint32_t *thr = reinterpret_cast<uint32_t *>(mh_smem);
    if (threadIdx.x < 5u) thr[2u * threadIdx.x] = tab.T[threadIdx.x];
    const uint32_t RS = T + 8u, half = T >> 1, tile_threads = half * T, ntx = L / T, nth = ntx >> 1;
    const uint32_t slots = blockDim.x / tile_threads, slot = threadIdx.x / tile_threads;
    const uint32_t t = threadIdx.x - slot * tile_threads;
    const uint32_t slab_bytes = ((T + 2u) * RS + 15u) & ~15u;
    unsigned long long *staged = reinterpret_cast<unsigned long long *>(mh_smem + 64);
    int8_t *slabs = mh_smem + 64 + ROUNDS * slots * 32u;
    const uint32_t yl = t / half, xh = t - yl * half, par = yl & 1u;
    const int da = par ? 1 : -1;
    const char *thr4 = reinterpret_cast<const char *>(thr) + 16;
    auto tile_barrier = [&]() {
        if (tile_threads == 32u) __syncwarp();
        else asm volatile("bar.sync %0, %1;" ::"r"(slot + 1u), "r"(tile_threads) : "memory");
    };

    Stream<KIND> gen[ROUNDS];
    uint32_t pair[ROUNDS], ty_[ROUNDS], txh_[ROUNDS];
    // ---- load every tile of this CTA (both colours) with its initial halo; load the generator states ----
#pragma unroll
    for (int r = 0; r < ROUNDS; r++) {
        pair[r] = ((uint32_t)r * gridDim.x + blockIdx.x) * slots + slot; // rounds interleave the CTAs: even load
        ty_[r] = pair[r] / nth;
        txh_[r] = pair[r] - ty_[r] * nth;
        if (pair[r] >= n_pairs) continue; // uniform per tile
        for (uint32_t C = 0; C < 2u; C++) {
            int8_t *tile = slabs + ((r * slots + slot) * 2u + C) * slab_bytes;
            const uint32_t tx = 2u * txh_[r] + ((ty_[r] + C) & 1u), x0 = tx * T, y0 = ty_[r] * T;
            const int8_t *grow = sp + (uint64_t)(y0 + yl) * L + x0 + 2u * xh;
            *reinterpret_cast<uint16_t *>(tile + (yl + 1u) * RS + 4u + 2u * xh) = *reinterpret_cast<const uint16_t *>(grow);
            if (t < T) {
                const uint32_t yu = y0 ? y0 - 1u : L - 1u, yd = (y0 + T == L) ? 0u : y0 + T;
                const uint32_t xl = x0 ? x0 - 1u : L - 1u, xr = (x0 + T == L) ? 0u : x0 + T;
                tile[0u * RS + 4u + t] = sp[(uint64_t)yu * L + x0 + t];
                tile[(T + 1u) * RS + 4u + t] = sp[(uint64_t)yd * L + x0 + t];
                tile[(t + 1u) * RS + 3u] = sp[(uint64_t)(y0 + t) * L + xl];
                tile[(t + 1u) * RS + 4u + T] = sp[(uint64_t)(y0 + t) * L + xr];
            }
        }
        gen[r].load(g, (uint64_t)pair[r] * tile_threads + t);
    }
    __syncthreads();

    const uint32_t round_stride = slots * 2u * slab_bytes; // bytes between the slabs of round r and r + 1
    const uint32_t mine_off = (yl + 1u) * RS + 4u + 2u * xh;
    for (uint32_t sweep = 0; sweep < n_sweeps; sweep++) {
        for (uint32_t C = 0; C < 2u; C++) {
            const unsigned long long stage = 2ull * sweep + C + 1ull;
            int8_t *tile0 = slabs + (slot * 2u + C) * slab_bytes; // round r: + r * round_stride
            if (stage > 1ull) {
                // ---- the first warp of the CTA waits for the inboxes of all its tiles of this colour ----
                if (threadIdx.x < 32u) {
                    for (uint32_t tt = threadIdx.x; tt < (uint32_t)ROUNDS * slots; tt += 32u) {
                        const uint32_t r = tt / slots, sl = tt - r * slots;
                        const uint32_t pr = (r * gridDim.x + blockIdx.x) * slots + sl;
                        if (pr >= n_pairs) continue;
                        const uint32_t tyq = pr / nth, tx = 2u * (pr - tyq * nth) + ((tyq + C) & 1u);
                        const unsigned long long *box = inbox + (uint64_t)(tyq * ntx + tx) * 4u;
                        unsigned long long w0, w1, w2, w3;
                        const unsigned long long want = stage - 1ull;
                        do {
                            mh_peek2(box, w0, w1);
                            mh_peek2(box + 2, w2, w3);
                        } while ((w0 >> (64u - kMhEpochBits)) != want || (w1 >> (64u - kMhEpochBits)) != want ||
                                 (w2 >> (64u - kMhEpochBits)) != want || (w3 >> (64u - kMhEpochBits)) != want);
                        staged[tt * 4u + 0u] = w0, staged[tt * 4u + 1u] = w1, staged[tt * 4u + 2u] = w2, staged[tt * 4u + 3u] = w3;
                    }
                }
                __syncthreads();
                // ---- unpack: halo above (0), below (1), left (2), right (3) of every round's tile ----
                if (t < 32u) {
#pragma unroll
                    for (int q = 0; q < 4 * ROUNDS; q++) {
                        if (pair[q >> 2] >= n_pairs) continue;
                        const unsigned long long vq = staged[((q >> 2) * slots + slot) * 4u + (q & 3)];
                        int8_t *tile = tile0 + (q >> 2) * round_stride;
                        int8_t *hp = (q & 3) == 0 ? tile + 4u : (q & 3) == 1 ? tile + (T + 1u) * RS + 4u : (q & 3) == 2 ? tile + RS + 3u : tile + RS + 4u + T;
                        const uint32_t step = (q & 3) < 2 ? 1u : RS;
                        for (uint32_t i = t; i < T; i += 32u) hp[i * step] = ((vq >> i) & 1ull) ? (int8_t)-1 : (int8_t)1;
                    }
                }
            }
            __syncthreads();
            int sa[ROUNDS], sb[ROUNDS];
#pragma unroll
            for (int r = 0; r < ROUNDS; r++) {
                const int8_t *mine = tile0 + r * round_stride + mine_off;
                sa[r] = (int)mine[par];
                sb[r] = (int)mine[1u - par];
            }
            for (uint32_t hit = 0; hit < k_hits; hit++) { // the rounds interleaved: one barrier serves both tiles
#pragma unroll
                for (int r = 0; r < ROUNDS; r++) {
                    if (pair[r] >= n_pairs) continue;
                    int8_t *pa = tile0 + r * round_stride + mine_off + par;
                    const int nn = sb[r] + (int)pa[da] + (int)pa[-(int)RS] + (int)pa[RS];
                    const uint32_t th = *reinterpret_cast<const uint32_t *>(thr4 + 4 * sa[r] * nn);
                    const uint32_t rnd = gen[r].next();
                    if ((rnd >> 8) < th) {
                        sa[r] = -sa[r];
                        *pa = (int8_t)sa[r];
                    }
                }
                tile_barrier();
#pragma unroll
                for (int r = 0; r < ROUNDS; r++) {
                    if (pair[r] >= n_pairs) continue;
                    int8_t *pb = tile0 + r * round_stride + mine_off + (1u - par);
                    const int nn = sa[r] + (int)pb[-da] + (int)pb[-(int)RS] + (int)pb[RS];
                    const uint32_t th = *reinterpret_cast<const uint32_t *>(thr4 + 4 * sb[r] * nn);
                    const uint32_t rnd = gen[r].next();
                    if ((rnd >> 8) < th) {
                        sb[r] = -sb[r];
                        *pb = (int8_t)sb[r];
                    }
                }
                tile_barrier();
            }
            if (t < 32u) { // pack my border lines (0 top row, 1 bottom row, 2 left column, 3 right column) with warp
                           // votes; lane q writes line q & 3 of round q >> 2 into the facing neighbour's inbox
                unsigned long long mine_word = 0ull;
#pragma unroll
                for (int q = 0; q < 4 * ROUNDS; q++) {
                    const int8_t *tile = tile0 + (q >> 2) * round_stride;
                    const int8_t *bp = (q & 3) == 0 ? tile + RS + 4u : (q & 3) == 1 ? tile + T * RS + 4u : (q & 3) == 2 ? tile + RS + 4u : tile + RS + 3u + T;
                    const uint32_t step = (q & 3) < 2 ? 1u : RS;
                    unsigned long long w = (unsigned long long)__ballot_sync(0xffffffffu, t < T && bp[t * step] < 0);
                    if (T > 32u) w |= (unsigned long long)__ballot_sync(0xffffffffu, t + 32u < T && bp[(t + 32u < T ? t + 32u : 0u) * step] < 0) << 32;
                    if (t == (uint32_t)q) mine_word = w;
                }
                const uint32_t qr = t >> 2, side = t & 3u;
                if (qr < (uint32_t)ROUNDS) {
                    uint32_t pr = pair[0], tyq = ty_[0], txq = txh_[0];
#pragma unroll
                    for (int r = 1; r < ROUNDS; r++)
                        if (qr == (uint32_t)r) pr = pair[r], tyq = ty_[r], txq = txh_[r];
                    if (pr < n_pairs) {
                        const uint32_t tx = 2u * txq + ((tyq + C) & 1u);
                        const uint32_t nx = side == 2u ? (tx ? tx - 1u : ntx - 1u) : side == 3u ? (tx + 1u == ntx ? 0u : tx + 1u) : tx;
                        const uint32_t ny = side == 0u ? (tyq ? tyq - 1u : ntx - 1u) : side == 1u ? (tyq + 1u == ntx ? 0u : tyq + 1u) : tyq;
                        // my top row is the upper neighbour's halo below (1), my left column the left neighbour's halo to the right (3)
                        mh_post(inbox + ((uint64_t)(ny * ntx + nx) * 4u + (side ^ 1u)), (stage << (64u - kMhEpochBits)) | mine_word);
                    }
                }
            }
        }
    }
    __syncthreads();
    // ---- write the tiles back, store the generator states ----
#pragma unroll
    for (int r = 0; r < ROUNDS; r++) {
        if (pair[r] >= n_pairs) continue;
        for (uint32_t C = 0; C < 2u; C++) {
            const int8_t *tile = slabs + ((r * slots + slot) * 2u + C) * slab_bytes;
            const uint32_t tx = 2u * txh_[r] + ((ty_[r] + C) & 1u), x0 = tx * T, y0 = ty_[r] * T;
            *reinterpret_cast<uint16_t *>(sp + (uint64_t)(y0 + yl) * L + x0 + 2u * xh) =
                *reinterpret_cast<const uint16_t *>(tile + (yl + 1u) * RS + 4u + 2u * xh);
        }
        gen[r].store(g, (uint64_t)pair[r] * tile_threads + t);
    }
}

// geometry of the one-launch path, or slots = 0 when the call does not qualify
struct MhCoop {
    uint32_t slots, rounds, grid, threads;
    size_t smem;
};
// does `device` accept cooperative launches at all (cached per device; false when the query fails)
static bool coop_launch_supported(int device)
{
    static std::atomic<int> cache[64]; // 0 = not asked, 1 = no, 2 = yes
    if (device < 0 || device >= 64) return false;
    int v = cache[device].load(std::memory_order_relaxed);
    if (v == 0) {
        int ok = 0;
        if (cudaDeviceGetAttribute(&ok, cudaDevAttrCooperativeLaunch, device) != cudaSuccess) {
            cudaGetLastError();
            ok = 0;
        }
        v = ok ? 2 : 1;
        cache[device].store(v, std::memory_order_relaxed);
    }
    return v == 2;
}

static MhCoop mh_coop_plan(const rng_handle &h, uint32_t L, uint32_t T, uint32_t n_sweeps)
{
    MhCoop c{0u, 0u, 0u, 0u, 0};
    const uint32_t tile_threads = T * T / 2u;
    if (!coop_launch_supported(h.device)) return c;       // e.g. some MPS / partitioned set-ups: per-colour launches
    if (kind_is_lfib(h.g.kind)) return c;                 // ring shared by a 256-thread CTA: its own CTA shape
    if (tile_threads % 32u || tile_threads > 1024u || T > 44u) return c; // named barriers count whole warps
    if (2ull * n_sweeps >= (1ull << kMhEpochBits)) return c;
    uint32_t slots = 1024u / tile_threads;
    if (tile_threads > 32u && slots > 15u) slots = 15u;   // named barriers 1..15
    const uint32_t pairs = (L / T) * (L / T) / 2u;
    const uint32_t sms = (uint32_t)sm_count(h.device);
    const uint32_t rounds = (pairs + sms * slots - 1u) / (sms * slots);
    if (rounds > 2u) return c;                            // a thread keeps at most two streams in registers
    const size_t slab = ((size_t)(T + 2u) * (T + 8u) + 15u) & ~(size_t)15u;
    c.slots = slots, c.rounds = rounds;
    c.grid = (pairs + slots * rounds - 1u) / (slots * rounds);
    if (c.grid > sms) c.grid = sms;
    c.threads = slots * tile_threads;
    c.smem = 64 + (size_t)rounds * slots * 32u + (size_t)rounds * slots * 2u * slab;
    return c;
}

// force = take the one-launch path whenever the call qualifies; otherwise only where it measured faster than one
// launch per coarse colour on a B200 (us per sweep, XORWOW, tile 16; one launch / per-colour launches):
//   L = 256: k = 1 5.07 / 4.91, k = 4 7.20 / 5.86      L = 512: k = 1 5.18 / 6.97, k = 4 7.33 / 9.13
//   L = 1024 (two streams per thread): k = 1 8.82 / 9.24, k = 4 12.81 / 11.82
// i.e. a stage costs about 2.5 us (post -> L2 -> poll round trip plus three block barriers) against 2.5-4.6 us for a
// launch with programmatic dependent launch: worth it for a single round of at least 512 tile pairs and few hits.
bool ising_multihit_coop_eligible(const rng_handle &h, uint32_t L, uint32_t T, uint32_t k_hits, uint32_t n_sweeps, bool force)
{
    const MhCoop c = mh_coop_plan(h, L, T, n_sweeps);
    if (!c.slots) return false;
    if (force) return true;
    return c.rounds == 1u && k_hits <= 4u && (L / T) * (L / T) / 2u >= 512u;
}

// the whole call (n_sweeps sweeps of both coarse colours) in one cooperative launch; `mailbox` = the tiles' inboxes,
// (L/T)^2 * 4 words of device memory, zeroed by this function on the stream before the launch (stage numbers restart at 1 every call)
cudaError_t launch_ising_multihit_coop(const rng_handle &h, int8_t *d_spins, uint32_t L, const IsingTable &tab, uint32_t T,
                                       uint32_t k_hits, uint32_t n_sweeps, uint64_t draws_done, unsigned long long *mailbox,
                                       cudaStream_t st)
{
    const MhCoop c = mh_coop_plan(h, L, T, n_sweeps);
    if (!c.slots) return cudaErrorInvalidConfiguration;
    Gen g = h.g;
    g.draws_done = draws_done;
    uint32_t pairs = (L / T) * (L / T) / 2u;
    cudaError_t e = cudaMemsetAsync(mailbox, 0, (size_t)(L / T) * (L / T) * 4u * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    IsingTable tabv = tab;
    uint32_t Lv = L, Tv = T, kv = k_hits, nv = n_sweeps;
    void *args[] = {&g, &d_spins, &Lv, &tabv, &Tv, &kv, &nv, &pairs, &mailbox};
    const void *fn = nullptr;
#define MHC(KIND) fn = c.rounds == 1u ? (const void *)ising_multihit_coop_kernel<KIND, 1> : (const void *)ising_multihit_coop_kernel<KIND, 2>
    switch (g.kind) {
    case RNG_LCG64: MHC(RNG_LCG64); break;
    case RNG_LCG64_LEAPFROG: MHC(RNG_LCG64_LEAPFROG); break;
    case RNG_XORWOW: MHC(RNG_XORWOW); break;
    case RNG_PHILOX4X32_10: MHC(RNG_PHILOX4X32_10); break;
    case RNG_XS1024W: MHC(RNG_XS1024W); break;
    case RNG_PHILOX4X32_7: MHC(RNG_PHILOX4X32_7); break;
    case RNG_LCG32: MHC(RNG_LCG32); break;
    case RNG_LCG64_BOTH: MHC(RNG_LCG64_BOTH); break;
    case RNG_LCG32_LEAPFROG: MHC(RNG_LCG32_LEAPFROG); break;
    case RNG_MWC: MHC(RNG_MWC); break;
    case RNG_MWC_MULTI: MHC(RNG_MWC_MULTI); break;
    default: return cudaErrorInvalidValue;
    }
#undef MHC
    if (c.smem > 48u * 1024u) {
        e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);
        if (e != cudaSuccess) return e;
    }
    // every CTA must be resident at once (the tiles wait for their neighbours' halos): ask the occupancy
    // calculator, not the SM count alone -- fewer SMs (MPS, partitions) or spills would make the launch too large
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, (int)c.threads, c.smem);
    if (e != cudaSuccess) return e;
    if ((uint64_t)per_sm * (uint64_t)sm_count(h.device) < c.grid) return cudaErrorCooperativeLaunchTooLarge;
    e = cudaLaunchCooperativeKernel(fn, dim3(c.grid), dim3(c.threads), args, c.smem, st);
    if (e != cudaSuccess) return e; // refused: nothing ran (the caller may fall back to per-colour launches)
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_ising_multihit(const rng_handle &h, int8_t *d_spins, uint32_t L, const IsingTable &tab, uint32_t T,
                                  uint32_t k_hits, uint64_t draws_done, int coarse, cudaStream_t st)
{
    Gen g = h.g;
    g.draws_done = draws_done;
    const uint32_t tiles = (L / T) * (L / T) / 2u;
    const size_t slab = ((size_t)(T + 2u) * (T + 8u) + 15u) & ~(size_t)15u;
    // programmatic dependent launch (internal.h) when the grid is at most about one wave
    const bool pdl = (uint64_t)L * L / 4ull <= kPdlMaxThreads; // one thread per stream of the active colour
    const uint32_t C = (uint32_t)coarse;
    cudaError_t e = cudaSuccess;
    if (kind_is_lfib(g.kind)) { // CTA = one 256-stream instance = 256 / (T*T/2) tiles (api.cu admits T = 8, 16 only)
        const uint32_t tpc = 256u / (T * T / 2u); // tiles % tpc == 0 because L % 32 == 0
        PdlLaunch pl(dim3(tiles / tpc), dim3(256), 64 + tpc * slab, st, pdl);
        if (g.kind == RNG_LFIB1279)
            e = cudaLaunchKernelEx(&pl.cfg, ising_multihit_kernel<RNG_LFIB1279, false>, g, d_spins, L, tab, T, k_hits, C, tiles);
        else
            e = cudaLaunchKernelEx(&pl.cfg, ising_multihit_kernel<RNG_LFIB521, false>, g, d_spins, L, tab, T, k_hits, C, tiles);
    } else if (T == 8u) { // one warp per tile, four tiles per CTA
        const uint32_t wpc = 4u;
        PdlLaunch pl(dim3((tiles + wpc - 1u) / wpc), dim3(wpc * 32u), 64 + wpc * slab, st, pdl);
#define MH(KIND) e = cudaLaunchKernelEx(&pl.cfg, ising_multihit_kernel<KIND, true>, g, d_spins, L, tab, T, k_hits, C, tiles)
        RNGB200_DISPATCH_KIND(g.kind, MH)
#undef MH
    } else {
        PdlLaunch pl(dim3(tiles), dim3(T * T / 2u), 64 + slab, st, pdl);
#define MH(KIND) e = cudaLaunchKernelEx(&pl.cfg, ising_multihit_kernel<KIND, false>, g, d_spins, L, tab, T, k_hits, C, tiles)
        RNGB200_DISPATCH_KIND(g.kind, MH)
#undef MH
    }
    count_launch();
    return e != cudaSuccess ? e : cudaGetLastError();
}

} // namespace rngb200
