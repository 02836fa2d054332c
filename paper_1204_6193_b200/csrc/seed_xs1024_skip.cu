// seed_xs1024_skip.cu -- a1 for RNG_XS1024W_SKIP: the paper's own seeding of its generator
// (PAPER.md:228).  All instances start from ONE state and instance g skips g * 2^137 updates,
// "by multiplying the state with the precomputed 2^137-th power of the recursion matrix M".
// The paper copies that matrix from a header and multiplies once per instance, one after the
// other ("very long kernel running times"), and suggests "including higher powers of the block
// skip matrix to reduce the number of multiplications needed".  Here everything is computed on
// the device at rng_create time, and the higher powers are used as a doubling tree:
//   1. M as a bit matrix: row r = one cooperative update (generators.cuh) of the unit vector r;
//   2. J_0 = M^(2^137) by 137 squarings, J_k = J_{k-1}^2 = M^(2^(137+k));
//   3. X(G0) = X_0 J^G0 for the shard's first instance G0, over the set bits of G0;
//   4. level k: X(G0 + i + 2^k) = X(G0 + i) J_k for all i < 2^k at once.
// Every instance costs ONE vector-matrix product however many instances there are.  Steps 1 and 2 do not depend on
// the seed: their result is kept per device for the life of the process (xs_skip_matrices).
// A matrix is uint32 [1024][32]: row r = image of the unit vector "word r/32, bit r%32"
// (word 0 most significant, R-D1); a product X A is the XOR of the rows of A at the set bits of
// X, with lane l of a warp holding word l of X and of the result.  128 KiB per matrix: L1/L2.
// Product code (sm_100a); shares nothing with oracle/.
#include <mutex>

#include "internal.h"

namespace rngb200 {

constexpr int XS_MAT_WORDS = 1024 * 32;

// lane's word of X A; xw = lane's word of X.  All 32 lanes must call.
__device__ __forceinline__ uint32_t xs_vecmat(uint32_t xw, const uint32_t *__restrict__ A, int lane)
{
    uint32_t acc0 = 0u, acc1 = 0u, acc2 = 0u, acc3 = 0u;
#pragma unroll 1
    for (int w = 0; w < 32; w++) {
        const uint32_t xv = __shfl_sync(0xffffffffu, xw, w); // warp-uniform
        if (xv == 0u) continue;
        const uint32_t *rows = A + (w * 32) * 32 + lane;
#pragma unroll
        for (int b = 0; b < 32; b += 4) { // predicated, independent loads: many in flight
            const uint32_t r0 = (xv >> b) & 1u ? rows[(b + 0) * 32] : 0u;
            const uint32_t r1 = (xv >> (b + 1)) & 1u ? rows[(b + 1) * 32] : 0u;
            const uint32_t r2 = (xv >> (b + 2)) & 1u ? rows[(b + 2) * 32] : 0u;
            const uint32_t r3 = (xv >> (b + 3)) & 1u ? rows[(b + 3) * 32] : 0u;
            acc0 ^= r0, acc1 ^= r1, acc2 ^= r2, acc3 ^= r3;
        }
    }
    return (acc0 ^ acc1) ^ (acc2 ^ acc3);
}

// step 1: one warp per row
__global__ void __launch_bounds__(256) xs_unit_matrix_kernel(uint32_t *__restrict__ M)
{
    const int r = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (r >= 1024) return;
    uint32_t s = (lane == (r >> 5)) ? (1u << (r & 31)) : 0u;
    s = xs1024_update_coop(s, lane);
    M[r * 32 + lane] = s;
}

// step 2: dst = src^2, (A A)[r] = A[r] A; one warp per row
__global__ void __launch_bounds__(256) xs_matrix_square_kernel(uint32_t *__restrict__ dst, const uint32_t *__restrict__ src)
{
    const int r = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (r >= 1024) return;
    dst[r * 32 + lane] = xs_vecmat(src[r * 32 + lane], src, lane);
}

// step 3: one warp.  X_0 = the randomly seeded state of instance 0 (R-D7b: words 2k, 2k+1 =
// lo32, hi32 of SM_seed[k], all-zero guard as in seed_xs1024_kernel); then X_0 J^G0.
struct XsSkipPtrs {
    const uint32_t *J[64];
};
__global__ void __launch_bounds__(32) xs_skip_start_kernel(uint32_t *__restrict__ state, const XsSkipPtrs ptrs, uint64_t G0,
                                                           uint64_t seed)
{
    const int lane = threadIdx.x;
    const uint64_t z = splitmix64_at(seed, (uint64_t)(lane >> 1));
    uint32_t x = (lane & 1) ? (uint32_t)(z >> 32) : (uint32_t)z;
    if (!__any_sync(0xffffffffu, x != 0u) && lane == 31) x = 1u;
    for (int k = 0; k < 64 && (G0 >> k) != 0ull; k++)
        if ((G0 >> k) & 1ull) x = xs_vecmat(x, ptrs.J[k], lane);
    state[lane] = x;
}

// step 4: instances [0, have) are done; warp i computes instance have + i = instance i times Jk
__global__ void __launch_bounds__(256) xs_skip_level_kernel(uint32_t *__restrict__ state, const uint32_t *__restrict__ Jk,
                                                            uint64_t have, uint64_t n_inst)
{
    const uint64_t i = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (i >= have || have + i >= n_inst) return; // warp-uniform
    state[(have + i) * 32 + lane] = xs_vecmat(state[i * 32 + lane], Jk, lane);
}

// ---- large levels: the product through byte tables ("four Russians") ----
// For a level with many instances the rows of J_k are first combined into a table T[c][v] = XOR of the rows
// 8c + b over the set bits b of the byte value v (c = 0..127, v = 0..255; 4 MiB, L2-resident): a product is then 128
// table rows instead of one predicated row load for each of the 1024 bits -- a sixth of the instructions.
// Byte c of X = byte c % 4 of word c / 4; bit b of that byte is bit 8 (c % 4) + b of the word, i.e. row
// 32 (c / 4) + 8 (c % 4) + b = 8c + b of the matrix.
constexpr int XS_TAB_WORDS = 128 * 256 * 32;

// one CTA per table position c: generation j doubles the table, entry v in [2^j, 2^(j+1)) = entry v - 2^j ^ row 8c + j
__global__ void __launch_bounds__(256) xs_byte_table_kernel(uint32_t *__restrict__ T, const uint32_t *__restrict__ J)
{
    __shared__ uint32_t tab[256 * 32];
    const int c = (int)blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (warp == 0) tab[lane] = 0u;
    __syncthreads();
    for (int j = 0; j < 8; j++) {
        const uint32_t row = J[(8 * c + j) * 32 + lane];
        for (int v = (1 << j) + warp; v < (2 << j); v += 8) tab[v * 32 + lane] = tab[(v - (1 << j)) * 32 + lane] ^ row;
        __syncthreads();
    }
    uint32_t *t = T + (size_t)c * 256 * 32;
    for (int i = threadIdx.x; i < 256 * 32; i += 256) t[i] = tab[i];
}

__global__ void __launch_bounds__(256) xs_skip_level_table_kernel(uint32_t *__restrict__ state, const uint32_t *__restrict__ T,
                                                                  uint64_t have, uint64_t n_inst)
{
    const uint64_t i = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (i >= have || have + i >= n_inst) return; // warp-uniform
    const uint32_t xw = state[i * 32 + lane];
    uint32_t acc0 = 0u, acc1 = 0u, acc2 = 0u, acc3 = 0u;
#pragma unroll 4
    for (int w = 0; w < 32; w++) {
        const uint32_t xv = __shfl_sync(0xffffffffu, xw, w); // warp-uniform word w of X
        const uint32_t *t = T + (size_t)(4 * w) * 256 * 32 + lane;
        acc0 ^= t[(size_t)(xv & 255u) * 32];
        acc1 ^= t[(size_t)(256 + ((xv >> 8) & 255u)) * 32];
        acc2 ^= t[(size_t)(512 + ((xv >> 16) & 255u)) * 32];
        acc3 ^= t[(size_t)(768 + (xv >> 24)) * 32];
    }
    state[(have + i) * 32 + lane] = (acc0 ^ acc1) ^ (acc2 ^ acc3);
}

// The skip matrices J_k = M^(2^(137+k)) depend on the generator only, not on the seed or the handle: they are
// computed once per device and process (the paper ships its matrix in a header; 128 KiB per level here, 2.5 MiB for
// 2^19 instances) and extended when a later handle needs more levels.  Complete levels are immutable, and the stream
// that computed them was synchronised before `levels` was raised, so any later stream may read them.
struct XsSkipCache {
    uint32_t *J[64] = {};
    int levels = 0;
};
static std::mutex g_xs_skip_mutex;
static XsSkipCache g_xs_skip_cache[64]; // by device ordinal

// makes J_0 .. J_{levels-1} of `device` available; *launched = kernels launched for it
static cudaError_t xs_skip_matrices(int device, int levels, cudaStream_t st, uint32_t *const **J, uint64_t *launched)
{
    *launched = 0;
    if (device < 0 || device >= 64 || levels > 64) return cudaErrorInvalidValue;
    std::lock_guard<std::mutex> lock(g_xs_skip_mutex);
    XsSkipCache &c = g_xs_skip_cache[device];
    *J = c.J;
    if (c.levels >= levels) return cudaSuccess;
    cudaError_t e = cudaSuccess;
    for (int k = c.levels; k < levels && e == cudaSuccess; k++)
        if (!c.J[k]) e = cudaMalloc((void **)&c.J[k], (size_t)XS_MAT_WORDS * 4);
    if (e != cudaSuccess) return e;
    if (c.levels == 0) {
        uint32_t *tmp = nullptr;
        e = cudaMalloc((void **)&tmp, (size_t)2 * XS_MAT_WORDS * 4);
        if (e != cudaSuccess) return e;
        uint32_t *a = tmp, *b = tmp + XS_MAT_WORDS;
        xs_unit_matrix_kernel<<<128, 256, 0, st>>>(a);
        for (int i = 0; i < 137; i++) { // M^(2^137): the sub-stream length of PAPER.md:228
            xs_matrix_square_kernel<<<128, 256, 0, st>>>(i == 136 ? c.J[0] : b, a);
            uint32_t *t = a;
            a = b;
            b = t;
        }
        *launched += 138;
        // a launch that was refused is reported by cudaGetLastError, not by the synchronise: J[0] counts as
        // valid (for every later handle of the process) only when both are clean
        e = cudaGetLastError();
        const cudaError_t es = cudaStreamSynchronize(st);
        cudaFree(tmp);
        if (e == cudaSuccess) e = es;
        if (e != cudaSuccess) return e; // levels stays 0: the next handle computes J[0] again
        c.levels = 1;
    }
    for (int k = c.levels; k < levels; k++) {
        xs_matrix_square_kernel<<<128, 256, 0, st>>>(c.J[k], c.J[k - 1]);
        (*launched)++;
    }
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) c.levels = levels;
    return e;
}

cudaError_t launch_seed_xs1024_skip(const Gen &g, int device, cudaStream_t st)
{
    const uint64_t n_inst = g.S / 32, G0 = g.first / 32;
    int levels = 0; // matrices J_0 .. J_{levels-1}
    while (levels < 64 && (((G0 >> levels) != 0ull) || ((1ull << levels) < n_inst))) levels++;
    if (levels < 1) levels = 1;
    uint32_t *const *J = nullptr;
    uint64_t launches = 0;
    cudaError_t e = xs_skip_matrices(device, levels, st, &J, &launches);
    if (e != cudaSuccess) return e;
    // the start kernel walks the set bits of G0 through a table of the levels' pointers
    XsSkipPtrs ptrs;
    for (int k = 0; k < 64; k++) ptrs.J[k] = k < levels ? J[k] : nullptr;
    xs_skip_start_kernel<<<1, 32, 0, st>>>((uint32_t *)g.state, ptrs, G0, g.seed);
    launches++;
    int k = 0;
    uint32_t *table = nullptr; // byte table of the current level (levels of at least kTableFrom instances)
    constexpr uint64_t kTableFrom = 4096;
    for (uint64_t have = 1; have < n_inst; have <<= 1, k++) {
        const uint64_t warps = (n_inst - have < have) ? (n_inst - have) : have;
        const uint64_t grid = (warps * 32 + 255) / 256;
        if (grid > 0x7fffffffull) {
            e = cudaErrorInvalidConfiguration;
            break;
        }
        if (warps >= kTableFrom) {
            if (!table) e = cudaMalloc((void **)&table, (size_t)XS_TAB_WORDS * 4);
            if (e != cudaSuccess) break;
            xs_byte_table_kernel<<<128, 256, 0, st>>>(table, J[k]); // stream order: after the previous level's reads
            xs_skip_level_table_kernel<<<(unsigned)grid, 256, 0, st>>>((uint32_t *)g.state, table, have, n_inst);
            launches += 2;
        } else {
            xs_skip_level_kernel<<<(unsigned)grid, 256, 0, st>>>((uint32_t *)g.state, J[k], have, n_inst);
            launches++;
        }
    }
    count_launch(launches);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (table) { // the table must outlive the kernels that read it
        const cudaError_t es = cudaStreamSynchronize(st);
        cudaFree(table);
        if (e == cudaSuccess) e = es;
    }
    return e;
}

} // namespace rngb200
