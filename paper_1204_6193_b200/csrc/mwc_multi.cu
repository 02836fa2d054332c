// mwc_multi.cu -- a1 for RNG_MWC_MULTI: one multiply-with-carry multiplier per stream (the
// paper's Table 1 row "MWC, different a").  "It is possible to systematically generate multipliers by finding
// the largest safe prime am-1 with a less than 2^32 (which is just the a = 4294967118 above) and then
// systematically working one's way down ... To check for primality one uses ... Rabin-Miller."  The paper
// generates them on the host with an arbitrary-precision library and ships them to the GPU; here the search
// runs on the device at rng_create time: candidates a = 2^32-1, 2^32-2, ... are tested in parallel (trial
// division, then Miller-Rabin with the twelve bases 2..37, a proof below 3.3e24), survivors are numbered by
// a block-wise prefix sum, and multiplier number (first + s) goes to local stream s.  About one candidate in
// 600 qualifies.  The host only loops over chunks of candidates until enough have been found.
// State layout (SoA, coalesced): u32 x[S], c[S], a[S].   Product code (sm_100a); shares nothing with oracle/.
#include "internal.h"

namespace rngb200 {

__device__ __forceinline__ uint64_t mulmod64(uint64_t a, uint64_t b, uint64_t n)
{
    return (uint64_t)((unsigned __int128)a * b % n);
}
__device__ uint64_t powmod64(uint64_t a, uint64_t e, uint64_t n)
{
    uint64_t r = 1ull;
    a %= n;
    while (e) {
        if (e & 1ull) r = mulmod64(r, a, n);
        a = mulmod64(a, a, n);
        e >>= 1;
    }
    return r;
}
// Miller-Rabin for one base; n odd > 2, n - 1 = d 2^r
__device__ bool mr_round(uint64_t n, uint64_t d, int r, uint64_t base)
{
    uint64_t x = powmod64(base, d, n);
    if (x == 1ull || x == n - 1ull) return true;
    for (int k = 1; k < r; k++) {
        x = mulmod64(x, x, n);
        if (x == n - 1ull) return true;
    }
    return false;
}
__device__ bool is_prime64(uint64_t n)
{
    const uint32_t small[17] = {2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37, 41, 43, 47, 53, 59};
    if (n < 2ull) return false;
#pragma unroll 1
    for (int i = 0; i < 17; i++)
        if (n % small[i] == 0ull) return n == small[i];
    uint64_t d = n - 1ull;
    int r = 0;
    while ((d & 1ull) == 0ull) {
        d >>= 1;
        r++;
    }
#pragma unroll 1
    for (int i = 0; i < 12; i++) // bases 2..37: deterministic for n < 3.3e24
        if (!mr_round(n, d, r, small[i])) return false;
    return true;
}
// a qualifies iff p = a 2^32 - 1 and (p - 1)/2 are both prime (a m - 1 is a safe prime)
__device__ bool mwc_is_multiplier(uint32_t a)
{
    const uint64_t p = ((uint64_t)a << 32) - 1ull;
    return a > 0u && is_prime64((p - 1ull) >> 1) && is_prime64(p);
}

constexpr int MWC_BLOCK = 256;

// pass 1: candidate i of the chunk is a = top - i; flag it and count per block
__global__ void __launch_bounds__(MWC_BLOCK) mwc_flag_kernel(uint32_t top, uint32_t n_cand, uint8_t *__restrict__ flags,
                                                            uint32_t *__restrict__ block_count)
{
    const uint32_t i = blockIdx.x * MWC_BLOCK + threadIdx.x;
    const bool ok = i < n_cand && i <= top - 1u && mwc_is_multiplier(top - i);
    if (i < n_cand) flags[i] = ok ? 1u : 0u;
    const int cnt = __syncthreads_count(ok);
    if (threadIdx.x == 0) block_count[blockIdx.x] = (uint32_t)cnt;
}
// pass 2 (one CTA): exclusive prefix sum of the block counts, offset by the running total *found
__global__ void __launch_bounds__(1024) mwc_scan_kernel(uint32_t *__restrict__ block_count, uint32_t n_blocks,
                                                        unsigned long long *__restrict__ found)
{
    __shared__ uint32_t part[1024];
    const uint32_t per = (n_blocks + 1023u) / 1024u, lo = threadIdx.x * per;
    uint32_t sum = 0;
    for (uint32_t k = lo; k < lo + per && k < n_blocks; k++) sum += block_count[k];
    part[threadIdx.x] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t run = 0;
        for (int t = 0; t < 1024; t++) {
            const uint32_t v = part[t];
            part[t] = run;
            run += v;
        }
        part[0] = 0; // (already)
        block_count[n_blocks] = run; // total of this chunk
    }
    __syncthreads();
    uint32_t run = part[threadIdx.x];
    for (uint32_t k = lo; k < lo + per && k < n_blocks; k++) {
        const uint32_t v = block_count[k];
        block_count[k] = run;
        run += v;
    }
    (void)found;
}
// pass 3: the flagged candidate with running number idx (counted from the top, over all chunks so far) is
// multiplier number idx; local stream idx - first receives it
__global__ void __launch_bounds__(MWC_BLOCK) mwc_assign_kernel(uint32_t top, uint32_t n_cand, const uint8_t *__restrict__ flags,
                                                              const uint32_t *__restrict__ block_excl, uint64_t base,
                                                              uint64_t first, uint64_t S, uint32_t *__restrict__ a_out)
{
    __shared__ uint32_t warp_sum[MWC_BLOCK / 32];
    const uint32_t i = blockIdx.x * MWC_BLOCK + threadIdx.x;
    const bool ok = i < n_cand && flags[i];
    const unsigned bal = __ballot_sync(0xffffffffu, ok);
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    if (lane == 0) warp_sum[warp] = (uint32_t)__popc(bal);
    __syncthreads();
    uint32_t before = (uint32_t)__popc(bal & ((1u << lane) - 1u));
    for (uint32_t w = 0; w < warp; w++) before += warp_sum[w];
    if (ok) {
        const uint64_t idx = base + block_excl[blockIdx.x] + before;
        if (idx >= first && idx < first + S) a_out[idx - first] = top - i;
    }
}

// (x_0, c_0) = (lo32, hi32 mod a_s) of SM_seed[s], fixed points moved (R-M1 with the stream's own multiplier)
__global__ void seed_mwc_multi_kernel(uint32_t *__restrict__ w, uint64_t S, uint64_t first, uint64_t seed)
{
    const uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= S) return;
    const uint64_t z = splitmix64_at(seed, first + s);
    const uint32_t a = w[2 * S + s];
    uint32_t x = (uint32_t)z, c = (uint32_t)(z >> 32) % a;
    if (x == 0u && c == 0u) x = 1u;
    if (x == 0xffffffffu && c == a - 1u) c = a - 2u;
    w[s] = x;
    w[S + s] = c;
}

cudaError_t launch_seed_mwc_multi(const Gen &g, cudaStream_t st)
{
    constexpr uint32_t CHUNK = 1u << 22; // candidates per pass
    constexpr uint32_t NBLK = CHUNK / MWC_BLOCK;
    uint8_t *flags = nullptr;
    uint32_t *blk = nullptr;
    cudaError_t e = cudaMalloc((void **)&flags, CHUNK);
    if (e == cudaSuccess) e = cudaMalloc((void **)&blk, (NBLK + 1) * sizeof(uint32_t));
    if (e != cudaSuccess) {
        cudaFree(flags);
        return e;
    }
    uint32_t *w = (uint32_t *)g.state;
    const uint64_t need = g.first + g.S;
    uint64_t found = 0, top = 0xffffffffull, launches = 0;
    while (found < need && top >= 1ull && e == cudaSuccess) {
        const uint32_t n_cand = (uint32_t)(top < CHUNK ? top : CHUNK);
        const uint32_t nb = (n_cand + MWC_BLOCK - 1) / MWC_BLOCK;
        mwc_flag_kernel<<<nb, MWC_BLOCK, 0, st>>>((uint32_t)top, n_cand, flags, blk);
        mwc_scan_kernel<<<1, 1024, 0, st>>>(blk, nb, nullptr);
        mwc_assign_kernel<<<nb, MWC_BLOCK, 0, st>>>((uint32_t)top, n_cand, flags, blk, found, g.first, g.S, w + 2 * g.S);
        launches += 3;
        uint32_t got = 0;
        e = cudaMemcpyAsync(&got, blk + nb, sizeof got, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st); // control flow only: how many were found so far
        found += got;
        top -= n_cand;
    }
    if (e == cudaSuccess && found < need) e = cudaErrorInvalidValue; // more streams than multipliers below 2^32
    if (e == cudaSuccess) {
        const unsigned B = 256, grid = (unsigned)((g.S + B - 1) / B);
        seed_mwc_multi_kernel<<<grid, B, 0, st>>>(w, g.S, g.first, g.seed);
        launches++;
        e = cudaGetLastError();
    }
    count_launch(launches);
    const cudaError_t es = cudaStreamSynchronize(st);
    cudaFree(flags);
    cudaFree(blk);
    return e != cudaSuccess ? e : es;
}

} // namespace rngb200
