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
