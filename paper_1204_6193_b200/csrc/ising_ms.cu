// ising_ms.cu -- a8, multi-spin-coded form of the checkerboard Metropolis half-sweep
// (BASELINE.json config 5; readings R-E1..E7).  Same trajectory, bit for
// bit, as the byte kernels in ising.cu: only the in-flight representation differs.
//
// Representation (device scratch owned by the handle, alive for one ising_sweep call):
// one bit plane per colour, plane_c[q >> 5] bit (q & 31) = 1 iff the spin of the colour-c
// site q is -1, with q = y*(L/2) + xh the site number of R-E6 (x = 2*xh + ((y+c)&1)).
// A 32-bit word is 32 consecutive sites of one row (needs L % 64 == 0).  The int8 lattice
// is packed once at the start of ising_sweep and unpacked once at the end.
//
// Neighbours of the 32 sites of word (y, j) of colour c, all in the OTHER plane N:
//   up    N[(y-1) W + j]      down  N[(y+1) W + j]      same index  N[y W + j]
//   and the same row shifted by one site: towards xh-1 if p = (y+c)&1 is 0, towards xh+1
//   if p is 1 (one funnel shift with the adjacent word, periodic).
// nbar = number of neighbours anti-aligned with the site = bit-sliced sum of the four
// words (N_k xor C); aligned neighbours (h+4)/2 = 4 - nbar.  For beta >= 0 the Metropolis
// table has T[i] = 2^24 (always flip) for h <= 0, so
//   flip = (nbar >= 2) | (r <= thr0) | ((nbar & 1) & (r <= thr1)),
//   thr0 = 256 T[4] - 1 (nbar = 0), thr1 = 256 T[3] - 1 (nbar = 1), thr0 <= thr1,
// where (r >> 8) < T  <=>  r <= 256 T - 1 for 1 <= T <= 2^24.  The host takes the byte
// kernels when the table does not have this shape.
//
// The two compares of a draw are two carry chains: sub.cc thr - r leaves the carry flag set
// iff there is no borrow (r <= thr: the hardware subtracts as thr + ~r + 1), and
// addc acc,acc,acc shifts that flag into an accumulator; after 32 draws the bit-reversed
// accumulator is the word of accept bits.  4 integer adds per site, no
// per-site table lookup, select or byte extraction; the random numbers stay in registers.
//
// Thread <-> stream mapping (R-E6: stream s owns sites [sK, (s+1)K) and spends one draw
// per site in increasing q):
//   STREAM mode (K % 32 == 0): one thread per stream, its K/32 words in order, generator
//     state in registers for all K draws (the paper's "many numbers per state load"
//     regime).
//   WORD mode (K in {4, 8, 16}): one thread per word = 32/K consecutive streams.
#include "internal.h"
#include "streams.cuh"

namespace rngb200 {

struct MsThr {
    uint32_t thr0, thr1;
};

// acc <- 2 acc + (r <= thr), for both thresholds
__device__ __forceinline__ void ms_cmp_insert(uint32_t r, const MsThr &t, uint32_t &n0, uint32_t &n1)
{
    asm("{\n\t"
        ".reg .u32 t;\n\t"
        "sub.cc.u32 t, %2, %4;\n\t"
        "addc.u32 %0, %0, %0;\n\t"
        "sub.cc.u32 t, %3, %4;\n\t"
        "addc.u32 %1, %1, %1;\n\t"
        "}"
        : "+r"(n0), "+r"(n1)
        : "r"(t.thr0), "r"(t.thr1), "r"(r));
}

// the four neighbour words of word (y, j) and the word itself
struct MsWord {
    uint32_t *cptr;
    uint32_t C, U, D, H0, H1;
    __device__ __forceinline__ void load(uint32_t *__restrict__ Cp, const uint32_t *__restrict__ Np, uint32_t L,
                                         uint32_t wpr, uint32_t y, uint32_t j, uint32_t colour)
    {
        const uint32_t yu = y ? y - 1u : L - 1u, yd = (y + 1u == L) ? 0u : y + 1u;
        const uint32_t base = y * wpr;
        cptr = Cp + base + j;
        C = *cptr;
        U = Np[yu * wpr + j];
        D = Np[yd * wpr + j];
        H0 = Np[base + j];
        if (((y + colour) & 1u) == 0u) { // active sites at even x: other horizontal neighbour is xh-1
            const uint32_t Hn = Np[base + (j ? j - 1u : wpr - 1u)];
            H1 = __funnelshift_l(Hn, H0, 1); // (H0 << 1) | (Hn >> 31)
        } else {
            const uint32_t Hn = Np[base + (j + 1u == wpr ? 0u : j + 1u)];
            H1 = __funnelshift_r(H0, Hn, 1); // (H0 >> 1) | (Hn << 31)
        }
    }
    // n0, n1: bit (31-k) = (r_k <= thr0 / thr1), k = site within the word
    __device__ __forceinline__ void update_store(uint32_t n0, uint32_t n1)
    {
        const uint32_t A0 = __brev(n0), A1 = __brev(n1);
        const uint32_t x0 = U ^ C, x1 = D ^ C, x2 = H0 ^ C, x3 = H1 ^ C;
        const uint32_t s = x0 ^ x1 ^ x2, cy = (x0 & x1) | (x0 & x2) | (x1 & x2);
        const uint32_t b0 = s ^ x3, cy2 = s & x3;
        const uint32_t flip = (cy | cy2) | A0 | (b0 & A1);
        *cptr = C ^ flip;
    }
};

// ---- STREAM mode -------------------------------------------------------------------
template <int KIND>
__global__ void __launch_bounds__(64) ising_ms_stream_kernel(Gen g, uint32_t *__restrict__ Cp,
                                                             const uint32_t *__restrict__ Np, uint32_t L, MsThr thr,
                                                             uint32_t W, uint32_t colour)
{
    const uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.S) return; // xs1024: S % 32 == 0 and blockDim % 32 == 0, whole warps leave together
    const uint32_t wpr = L >> 6;
    uint32_t widx = (uint32_t)s * W;
    uint32_t y = widx / wpr, j = widx - y * wpr;
    if (kind_is_philox(KIND)) {
        const uint64_t key = (g.first + s) ^ g.seed;
        const uint32_t k0 = (uint32_t)key, k1 = (uint32_t)(key >> 32);
        uint64_t b = g.draws_done >> 2; // draws_done % 4 == 0 (host-checked): whole blocks
        for (uint32_t i = 0; i < W; i++) {
            MsWord mw;
            mw.load(Cp, Np, L, wpr, y, j, colour);
            uint32_t n0 = 0u, n1 = 0u;
#pragma unroll
            for (int gi = 0; gi < 8; gi++, b++) {
                const uint4 o = philox4x32<philox_rounds(KIND)>((uint32_t)b, (uint32_t)(b >> 32), 0u, 0u, k0, k1);
                ms_cmp_insert(o.x, thr, n0, n1);
                ms_cmp_insert(o.y, thr, n0, n1);
                ms_cmp_insert(o.z, thr, n0, n1);
                ms_cmp_insert(o.w, thr, n0, n1);
            }
            mw.update_store(n0, n1);
            if (++j == wpr) {
                j = 0;
                y++;
            }
        }
    } else {
        Stream<KIND> gen;
        gen.load(g, s);
        const uint32_t one = g.k_one; // the compares fill the alu pipe: XORWOW's additions go to the fma pipe
        for (uint32_t i = 0; i < W; i++) {
            MsWord mw;
            mw.load(Cp, Np, L, wpr, y, j, colour);
            uint32_t n0 = 0u, n1 = 0u;
#pragma unroll
            for (int k = 0; k < 32; k++) {
                uint32_t r;
                if constexpr (KIND == RNG_XORWOW) r = gen.st.next_fma_adds(one);
                else r = gen.next();
                ms_cmp_insert(r, thr, n0, n1);
            }
            mw.update_store(n0, n1);
            if (++j == wpr) {
                j = 0;
                y++;
            }
        }
        gen.store(g, s);
    }
}

// N consecutive 32-bit words, 4N-byte aligned (N = 2, 4, 8)
template <int N>
__device__ __forceinline__ void load_vec(const uint32_t *__restrict__ p, uint32_t (&v)[N])
{
    if constexpr (N == 2) {
        const uint2 t = *reinterpret_cast<const uint2 *>(p);
        v[0] = t.x, v[1] = t.y;
    } else {
#pragma unroll
        for (int q = 0; q < N / 4; q++) {
            const uint4 t = reinterpret_cast<const uint4 *>(p)[q];
            v[4 * q] = t.x, v[4 * q + 1] = t.y, v[4 * q + 2] = t.z, v[4 * q + 3] = t.w;
        }
    }
}
template <int N>
__device__ __forceinline__ void store_vec(uint32_t *__restrict__ p, const uint32_t (&v)[N])
{
    if constexpr (N == 2) {
        *reinterpret_cast<uint2 *>(p) = make_uint2(v[0], v[1]);
    } else {
#pragma unroll
        for (int q = 0; q < N / 4; q++)
            reinterpret_cast<uint4 *>(p)[q] = make_uint4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
    }
}

// ---- WORD mode: K in {4, 8, 16}, 32/K streams per word -------------------------------
template <int KIND, int K>
__global__ void __launch_bounds__(128) ising_ms_word_kernel(Gen g, uint32_t *__restrict__ Cp,
                                                            const uint32_t *__restrict__ Np, uint32_t L, MsThr thr,
                                                            uint32_t n_words, uint32_t colour)
{
    const uint32_t widx = blockIdx.x * blockDim.x + threadIdx.x;
    if (widx >= n_words) return;
    const uint32_t wpr = L >> 6;
    const uint32_t y = widx / wpr, j = widx - y * wpr;
    MsWord mw;
    mw.load(Cp, Np, L, wpr, y, j, colour);
    uint32_t n0 = 0u, n1 = 0u;
    const uint64_t s0 = (uint64_t)widx * (32 / K);
    if (kind_is_philox(KIND) && (uint32_t)(g.first + s0) <= 0xffffffffu - 32u / K) {
        // The 32/K streams of this word are consecutive ids sharing the high key word, and every
        // stream is at the same counter (all streams advance in lockstep), so with the counter
        // (lo32(b), hi32(b), 0, 0) of R-C2:
        //  * round 1: M0 * lo32(b) is the same for every thread (uniform datapath) and M1 * 0 = 0;
        //  * round 2: its second S-box input, hi(M0 lo32(b)) ^ k1, is shared by all streams of the word,
        //    its first one, hi32(b) ^ k0, by all blocks of a stream;
        //  * key schedule: k1 + r W1 once per word; k0 + r W0 once per stream, pinned to the alu pipe (the
        //    multiplies fill the fma pipe: measured 1087 flips/ns with these adds on the fma pipe).
        // Same bits as philox4x32<R> (the `else` branch and the byte kernels; tests compare all of them).
        constexpr int R = philox_rounds(KIND);
        constexpr int NS = 32 / K, NBS = K / 4;
        const uint64_t b0 = g.draws_done >> 2; // draws_done % 4 == 0
        const uint64_t id0 = (g.first + s0) ^ g.seed;
        const uint32_t lo_id = (uint32_t)(g.first + s0), lo_seed = (uint32_t)g.seed;
        const uint32_t zero = g.k_zero;
        uint32_t rk1[R];
#pragma unroll
        for (int r = 0; r < R; r++) rk1[r] = (uint32_t)(id0 >> 32) + (uint32_t)r * kPhW1;
#pragma unroll
        for (int a = 0; a < NS; a++) {
            const uint32_t k0 = (lo_id + (uint32_t)a) ^ lo_seed;
            uint32_t rk0[R];
            rk0[0] = k0;
#pragma unroll
            for (int r = 1; r < R; r++) rk0[r] = add_on_alu_pipe(k0, (uint32_t)r * kPhW0, zero);
#pragma unroll
            for (int j = 0; j < NBS; j++) {
                const uint64_t ctr = b0 + (uint64_t)j;           // uniform
                const uint64_t pu = (uint64_t)kPhM0 * (uint32_t)ctr; // uniform: round 1, first S-box
                uint32_t c0 = (uint32_t)(ctr >> 32) ^ rk0[0];    // round 1 output: hi(M1*0) ^ c1 ^ k0
                uint32_t c1 = 0u;
                uint32_t c2 = (uint32_t)(pu >> 32) ^ rk1[0];
                uint32_t c3 = (uint32_t)pu;
#pragma unroll
                for (int r = 1; r < R; r++) {
                    const uint64_t p0 = (uint64_t)kPhM0 * c0;
                    const uint64_t p1 = (uint64_t)kPhM1 * c2;
                    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk0[r];
                    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk1[r];
                    c1 = (uint32_t)p1;
                    c3 = (uint32_t)p0;
                    c0 = n0;
                    c2 = n2;
                }
                ms_cmp_insert(c0, thr, n0, n1);
                ms_cmp_insert(c1, thr, n0, n1);
                ms_cmp_insert(c2, thr, n0, n1);
                ms_cmp_insert(c3, thr, n0, n1);
            }
        }
    } else if (kind_is_philox(KIND)) {
        const uint64_t b0 = g.draws_done >> 2; // draws_done % 4 == 0
#pragma unroll
        for (int gi = 0; gi < 8; gi++) {
            const uint64_t s = s0 + (4 * gi) / K;
            const uint64_t b = b0 + ((4 * gi) % K) / 4;
            const uint64_t key = (g.first + s) ^ g.seed;
            const uint4 o = philox4x32<philox_rounds(KIND)>((uint32_t)b, (uint32_t)(b >> 32), 0u, 0u, (uint32_t)key, (uint32_t)(key >> 32));
            ms_cmp_insert(o.x, thr, n0, n1);
            ms_cmp_insert(o.y, thr, n0, n1);
            ms_cmp_insert(o.z, thr, n0, n1);
            ms_cmp_insert(o.w, thr, n0, n1);
        }
    } else if constexpr (KIND == RNG_XORWOW) {
        // the 32/K streams of this word are consecutive in the interleaved state w[k*S + s]:
        // one vector load / store per state word instead of one access per stream and word
        constexpr int NS = 32 / K;
        const uint32_t one = g.k_one;
        uint32_t *w = (uint32_t *)g.state;
        uint32_t st[6][NS];
#pragma unroll
        for (int k = 0; k < 6; k++) load_vec<NS>(w + (uint64_t)k * g.S + s0, st[k]);
#pragma unroll
        for (int a = 0; a < NS; a++) {
            Xorwow x{st[0][a], st[1][a], st[2][a], st[3][a], st[4][a], st[5][a]};
#pragma unroll
            for (int k = 0; k < K; k++) ms_cmp_insert(x.next_fma_adds(one), thr, n0, n1);
            st[0][a] = x.x, st[1][a] = x.y, st[2][a] = x.z, st[3][a] = x.w, st[4][a] = x.v, st[5][a] = x.d;
        }
#pragma unroll
        for (int k = 0; k < 6; k++) store_vec<NS>(w + (uint64_t)k * g.S + s0, st[k]);
    } else {
#pragma unroll
        for (int a = 0; a < 32 / K; a++) {
            Stream<KIND> gen;
            gen.load(g, s0 + a);
#pragma unroll
            for (int k = 0; k < K; k++) ms_cmp_insert(gen.next(), thr, n0, n1);
            gen.store(g, s0 + a);
        }
    }
    mw.update_store(n0, n1);
}

// ---- pack / unpack / energy ----------------------------------------------------------
// thread per 64 bytes of a row: even-x bytes are colour (y&1), odd-x bytes the other one
__global__ void __launch_bounds__(256) ising_ms_pack_kernel(const int8_t *__restrict__ sp, uint32_t *__restrict__ plane0,
                                                            uint32_t *__restrict__ plane1, uint32_t L, uint32_t n_words)
{
    const uint32_t widx = blockIdx.x * blockDim.x + threadIdx.x;
    if (widx >= n_words) return;
    const uint32_t wpr = L >> 6, y = widx / wpr, j = widx - y * wpr;
    const uint4 *src = reinterpret_cast<const uint4 *>(sp + (uint64_t)y * L + 64u * j);
    uint32_t e = 0u, o = 0u;
#pragma unroll
    for (int v = 0; v < 4; v++) {
        const uint4 q = src[v];
        const uint32_t w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
        for (int k = 0; k < 4; k++) {
            const int kk = 4 * v + k; // word of the 64-byte run: bytes 4kk .. 4kk+3 = sites 2kk, 2kk+1 of each colour
            e |= ((w[k] >> 1) & 1u) << (2 * kk) | ((w[k] >> 17) & 1u) << (2 * kk + 1); // -1 = 0xff has bit 1 set
            o |= ((w[k] >> 9) & 1u) << (2 * kk) | ((w[k] >> 25) & 1u) << (2 * kk + 1);
        }
    }
    if (y & 1u) {
        plane1[widx] = e;
        plane0[widx] = o;
    } else {
        plane0[widx] = e;
        plane1[widx] = o;
    }
}

__global__ void __launch_bounds__(256) ising_ms_unpack_kernel(int8_t *__restrict__ sp, const uint32_t *__restrict__ plane0,
                                                              const uint32_t *__restrict__ plane1, uint32_t L,
                                                              uint32_t n_words)
{
    const uint32_t widx = blockIdx.x * blockDim.x + threadIdx.x;
    if (widx >= n_words) return;
    const uint32_t wpr = L >> 6, y = widx / wpr, j = widx - y * wpr;
    const uint32_t e = (y & 1u) ? plane1[widx] : plane0[widx];
    const uint32_t o = (y & 1u) ? plane0[widx] : plane1[widx];
    uint4 *dst = reinterpret_cast<uint4 *>(sp + (uint64_t)y * L + 64u * j);
#pragma unroll
    for (int v = 0; v < 4; v++) {
        uint32_t w[4];
#pragma unroll
        for (int k = 0; k < 4; k++) {
            const int kk = 4 * v + k;
            const uint32_t f = ((e >> (2 * kk)) & 1u) | ((o >> (2 * kk)) & 1u) << 8 | ((e >> (2 * kk + 1)) & 1u) << 16 |
                               ((o >> (2 * kk + 1)) & 1u) << 24;
            w[k] = 0x01010101u + f * 0xfeu; // +1 = 0x01, -1 = 0xff
        }
        dst[v] = make_uint4(w[0], w[1], w[2], w[3]);
    }
}

// E = -sum_<ij> s_i s_j.  Every bond joins the two colours, so summing nbar over the sites
// of colour 0 counts each anti-aligned bond once:  E = 2 * anti - 2 * L^2.
__global__ void __launch_bounds__(256) ising_ms_energy_kernel(const uint32_t *__restrict__ plane0,
                                                              const uint32_t *__restrict__ plane1, uint32_t L,
                                                              uint32_t n_words, unsigned long long *__restrict__ out)
{
    const uint32_t wpr = L >> 6;
    long long acc = 0;
    for (uint32_t widx = blockIdx.x * blockDim.x + threadIdx.x; widx < n_words; widx += gridDim.x * blockDim.x) {
        const uint32_t y = widx / wpr, j = widx - y * wpr;
        MsWord mw;
        mw.load(const_cast<uint32_t *>(plane0), plane1, L, wpr, y, j, 0u);
        const uint32_t x0 = mw.U ^ mw.C, x1 = mw.D ^ mw.C, x2 = mw.H0 ^ mw.C, x3 = mw.H1 ^ mw.C;
        acc += __popc(x0) + __popc(x1) + __popc(x2) + __popc(x3);
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    __shared__ long long part[8];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        long long t = 0;
        for (int w = 0; w < 8; w++) t += part[w];
        t *= 2;
        if (blockIdx.x == 0) t -= 2ll * (long long)L * (long long)L;
        atomicAdd(out, (unsigned long long)t);
    }
}

// ---- host side -----------------------------------------------------------------------
bool ising_ms_eligible(const rng_handle &h, uint32_t L, const IsingTable &tab, uint64_t K, uint64_t draws_done)
{
    if (L % 64u || L > 65536u) return false;
    if (h.g.kind == RNG_LFIB521 || h.g.kind == RNG_LFIB1279) return false; // CTA-shared state: byte kernel only
    const uint32_t one = 1u << 24;
    if (tab.T[0] != one || tab.T[1] != one || tab.T[2] != one) return false;
    if (tab.T[4] < 1u || tab.T[4] > tab.T[3] || tab.T[3] > one) return false;
    const int kind = h.g.kind;
    if (kind_is_philox(kind) && (draws_done & 3ull)) return false;
    if (K % 32ull == 0ull) return K / 32ull <= 0xffffffffull && h.g.S <= 0x7fffffffull;
    if (K == 4 || K == 8 || K == 16) return kind != RNG_XS1024W;
    return false;
}

cudaError_t launch_ising_ms_pack(const int8_t *d_spins, uint32_t *planes, uint32_t L, cudaStream_t st)
{
    const uint32_t n_words = (uint32_t)((uint64_t)L * L / 64);
    ising_ms_pack_kernel<<<(n_words + 255) / 256, 256, 0, st>>>(d_spins, planes, planes + n_words, L, n_words);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_ising_ms_unpack(int8_t *d_spins, const uint32_t *planes, uint32_t L, cudaStream_t st)
{
    const uint32_t n_words = (uint32_t)((uint64_t)L * L / 64);
    ising_ms_unpack_kernel<<<(n_words + 255) / 256, 256, 0, st>>>(d_spins, planes, planes + n_words, L, n_words);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_ising_ms_energy(const uint32_t *planes, uint32_t L, int64_t *d_out, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(d_out, 0, sizeof(int64_t), st);
    if (e != cudaSuccess) return e;
    const uint32_t n_words = (uint32_t)((uint64_t)L * L / 64);
    uint32_t grid = (n_words + 255) / 256;
    if (grid > 148u * 8u) grid = 148u * 8u;
    ising_ms_energy_kernel<<<grid, 256, 0, st>>>(planes, planes + n_words, L, n_words, (unsigned long long *)d_out);
    count_launch();
    return cudaGetLastError();
}

template <int KIND>
static void launch_ms_word(const Gen &g, uint32_t *Cp, const uint32_t *Np, uint32_t L, MsThr thr, uint32_t n_words,
                           uint64_t K, uint32_t colour, cudaStream_t st)
{
    const uint32_t grid = (n_words + 127) / 128;
    switch (K) {
    case 4: ising_ms_word_kernel<KIND, 4><<<grid, 128, 0, st>>>(g, Cp, Np, L, thr, n_words, colour); break;
    case 8: ising_ms_word_kernel<KIND, 8><<<grid, 128, 0, st>>>(g, Cp, Np, L, thr, n_words, colour); break;
    default: ising_ms_word_kernel<KIND, 16><<<grid, 128, 0, st>>>(g, Cp, Np, L, thr, n_words, colour); break;
    }
}

cudaError_t launch_ising_ms_half_sweep(const rng_handle &h, uint32_t *planes, uint32_t L, const IsingTable &tab, uint64_t K,
                                       uint64_t draws_done, int colour, cudaStream_t st)
{
    Gen g = h.g;
    g.draws_done = draws_done;
    const uint32_t n_words = (uint32_t)((uint64_t)L * L / 64);
    uint32_t *Cp = planes + (colour ? n_words : 0u);
    const uint32_t *Np = planes + (colour ? 0u : n_words);
    MsThr thr;
    thr.thr0 = (uint32_t)(((uint64_t)tab.T[4] << 8) - 1ull);
    thr.thr1 = (uint32_t)(((uint64_t)tab.T[3] << 8) - 1ull);
    if (K % 32ull == 0ull) {
        const uint32_t W = (uint32_t)(K / 32ull);
        const uint32_t grid = (uint32_t)((g.S + 63) / 64);
#define MS_STREAM(KIND) ising_ms_stream_kernel<KIND><<<grid, 64, 0, st>>>(g, Cp, Np, L, thr, W, (uint32_t)colour)
        RNGB200_DISPATCH_KIND(g.kind, MS_STREAM)
#undef MS_STREAM
    } else {
        switch (g.kind) {
        case RNG_LCG64: launch_ms_word<RNG_LCG64>(g, Cp, Np, L, thr, n_words, K, colour, st); break;
        case RNG_LCG64_LEAPFROG: launch_ms_word<RNG_LCG64_LEAPFROG>(g, Cp, Np, L, thr, n_words, K, colour, st); break;
        case RNG_XORWOW: launch_ms_word<RNG_XORWOW>(g, Cp, Np, L, thr, n_words, K, colour, st); break;
        case RNG_PHILOX4X32_10: launch_ms_word<RNG_PHILOX4X32_10>(g, Cp, Np, L, thr, n_words, K, colour, st); break;
        case RNG_PHILOX4X32_7: launch_ms_word<RNG_PHILOX4X32_7>(g, Cp, Np, L, thr, n_words, K, colour, st); break;
        case RNG_LCG32: launch_ms_word<RNG_LCG32>(g, Cp, Np, L, thr, n_words, K, colour, st); break;
        case RNG_LCG64_BOTH: launch_ms_word<RNG_LCG64_BOTH>(g, Cp, Np, L, thr, n_words, K, colour, st); break;
        case RNG_MWC: launch_ms_word<RNG_MWC>(g, Cp, Np, L, thr, n_words, K, colour, st); break;
        case RNG_MWC_MULTI: launch_ms_word<RNG_MWC_MULTI>(g, Cp, Np, L, thr, n_words, K, colour, st); break;
        case RNG_LCG32_LEAPFROG: launch_ms_word<RNG_LCG32_LEAPFROG>(g, Cp, Np, L, thr, n_words, K, colour, st); break;
        default: return cudaErrorInvalidValue;
        }
    }
    count_launch();
    return cudaGetLastError();
}

} // namespace rngb200
