// internal.h -- handle layout and the launch functions the C-ABI (api.cu) calls.
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/rng_b200.h"
#include "generators.cuh"

namespace rngb200 {

// Device-side LCG table built by the seeding kernel (eq.(2)):
//   pow2[m]  = step^(2^m),  m = 0..63     (pow2[0] is the per-draw step map itself)
//   mult4[t] = step^(4 t),  t = 0..255    (lane offsets of the intra-stream leapfrog)
// where step = (a, c) for RNG_LCG64 and (a, c)^n_total for RNG_LCG64_LEAPFROG.
struct LcgTable {
    Affine pow2[64];
    Affine mult4[256];
};

// Device state layout (all coalesced for "thread s handles stream s"):
//   LCG64 / LEAPFROG : u64 x[S]
//   XORWOW           : u32 w[6][S]   (word k of stream s at w[k*S + s]; k = x,y,z,w,v,d)
//   PHILOX           : none
//   XS1024W          : u32 w[S]      (word `lane` of instance g at w[32 g + lane])
//   MWC              : u64 (c << 32 | x)[S]
//   MWC_MULTI        : u32 w[3][S]   (x, c and the stream's multiplier a)
//   LCG32 / LEAPFROG : u32 x[S]   (leapfrog: the step map (a,c)^n_total mod 2^32 sits in LcgTable::pow2[0])
//   LFIB521 / 1279   : float u[S/256][r]  (an instance's last r numbers, oldest first)
struct Gen {
    int kind;
    uint64_t S;          // local streams
    uint64_t first;      // global id of local stream 0
    uint64_t n_total;    // global number of streams
    uint64_t seed;
    uint64_t draws_done; // per stream, all streams in lockstep
    void *state;         // device
    const LcgTable *lcg; // device (LCG kinds only)
    // the constants 1 and 0 as kernel parameters: values ptxas cannot fold, used to pin an
    // addition to the fma pipe (a*one + b) or the alu pipe (a + b + zero); see generators.cuh
    uint32_t k_one, k_zero;
};

} // namespace rngb200

struct rng_handle {
    rngb200::Gen g;
    int device;
    uint64_t state_bytes;
    void *staging;          // device staging for the *_host entry points
    uint64_t staging_bytes;
    int64_t *energy_scratch; // device, 1 x int64
    // work tickets of the persistent fill kernels: a device counter that is zero between launches (the warp
    // that draws a launch's last ticket resets it, fill_xs1024.cu)
    uint64_t *ticket;            // device, 1 x uint64 (zero at rng_create)
    uint32_t *ms_planes;     // device scratch of the multi-spin Ising path: two bit planes of L*L/64 words
    uint64_t ms_planes_bytes;
    unsigned long long *mh_mailbox; // device scratch of the one-launch multi-hit path: (L/T)^2 * 4 halo words
    uint64_t mh_mailbox_bytes;
    int var_xs1024, var_ising, var_store, var_lcg, var_xsfill, var_cvt;
    int api_kind; // the kind rng_create was called with (g.kind is RNG_XS1024W for RNG_XS1024W_SKIP)
};

// run MACRO(KIND) for the runtime kind (every kind that has a Stream<KIND>)
#define RNGB200_DISPATCH_KIND(kind, MACRO)                          \
    switch (kind) {                                                 \
    case RNG_LCG64: MACRO(RNG_LCG64); break;                        \
    case RNG_LCG64_LEAPFROG: MACRO(RNG_LCG64_LEAPFROG); break;      \
    case RNG_XORWOW: MACRO(RNG_XORWOW); break;                      \
    case RNG_PHILOX4X32_10: MACRO(RNG_PHILOX4X32_10); break;        \
    case RNG_XS1024W: MACRO(RNG_XS1024W); break;                    \
    case RNG_PHILOX4X32_7: MACRO(RNG_PHILOX4X32_7); break;          \
    case RNG_LCG32: MACRO(RNG_LCG32); break;                        \
    case RNG_LCG64_BOTH: MACRO(RNG_LCG64_BOTH); break;              \
    case RNG_LCG32_LEAPFROG: MACRO(RNG_LCG32_LEAPFROG); break;      \
    case RNG_MWC: MACRO(RNG_MWC); break;                            \
    case RNG_MWC_MULTI: MACRO(RNG_MWC_MULTI); break;                \
    default: return cudaErrorInvalidValue;                          \
    }

namespace rngb200 {

// Programmatic dependent launch for chains of short, dependent launches (the half-sweeps of a call): with this
// attribute the next grid is scheduled while the current one drains; the kernels order themselves with
// pdl_entry() (griddepcontrol.launch_dependents + griddepcontrol.wait, no-ops without the attribute), which must
// come before their first access to anything the previous launch wrote.  Only worth it when the grid is small:
// waiting CTAs of a big dependent grid take resources from the grid they wait for (measured: 85 -> 113 flips/ns for
// the 1024^2 multi-hit k = 1 half-sweeps), so `enable` is false above about one wave of threads.  It is NOT used for
// the multi-spin half-sweeps of ising_ms.cu: their grids are compute-bound and far from launch-bound, and the
// waiting CTAs of the next grid cost them 22 % (1796 -> 1404 flips/ns measured).
struct PdlLaunch {
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[1];
    PdlLaunch(dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool enable)
    {
        cfg = cudaLaunchConfig_t{};
        cfg.gridDim = grid;
        cfg.blockDim = block;
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = enable ? 1u : 0u;
    }
};
constexpr uint64_t kPdlMaxThreads = 148ull * 2048ull; // one wave of resident threads on a B200
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_entry()
{
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}
#endif

void count_launch(uint64_t n = 1);
// sets the calling thread's rng_last_error() message and returns `code` (for entry points outside api.cu)
int report_error(int code, const char *fmt, ...);
// number of SMs of `device` (cached per device; 148 on a B200)
int sm_count(int device);

// seed.cu
cudaError_t launch_seed(const Gen &g, LcgTable *tab, cudaStream_t st);
// mwc_multi.cu (RNG_MWC_MULTI: multiplier search + seeding; synchronises the stream, frees its scratch)
cudaError_t launch_seed_mwc_multi(const Gen &g, cudaStream_t st);
// lfib.cu (RNG_LFIB521 / RNG_LFIB1279: seeding and fill; draws and Ising go through Stream<KIND>)
cudaError_t launch_seed_lfib(const Gen &g, cudaStream_t st);
cudaError_t launch_lfib_fill(const Gen &g, void *d_out, uint64_t n, bool f32, int variant, cudaStream_t st);
cudaError_t launch_lfib_draw(const Gen &g, uint32_t *d_out, uint64_t n, cudaStream_t st);
// seed_xs1024_skip.cu (RNG_XS1024W_SKIP; synchronises the stream, frees its scratch)
cudaError_t launch_seed_xs1024_skip(const Gen &g, int device, cudaStream_t st);
// fill.cu  (f32 = apply the (u>>8)*2^-24 map; out is uint32_t* or float*)
cudaError_t launch_fill(const rng_handle &h, void *d_out, uint64_t n, bool f32, cudaStream_t st);
// fill_xs1024.cu (XORShift1024/Weyl, K words per lane; variant "xs1024" = K, 64 = the generic kernels)
cudaError_t launch_xs1024_fill(const rng_handle &h, void *d_out, uint64_t n, bool f32, cudaStream_t st);
cudaError_t launch_xs1024_draw(const rng_handle &h, uint32_t *d_out, uint64_t n, cudaStream_t st);
// draw.cu
cudaError_t launch_draw_reduce(const rng_handle &h, uint32_t *d_out, uint64_t n, cudaStream_t st);
// ising.cu
struct IsingTable {
    uint32_t T[5]; // integer thresholds: (r>>8) < T[i]  <=>  u < P[i]
};
cudaError_t launch_ising_half_sweep(const rng_handle &h, int8_t *d_spins, uint32_t L, const IsingTable &tab,
                                    uint64_t K, uint64_t draws_done, int colour, cudaStream_t st);
// ising_ms.cu (multi-spin-coded half-sweeps on bit planes; same trajectory as ising.cu)
bool ising_ms_eligible(const rng_handle &h, uint32_t L, const IsingTable &tab, uint64_t K, uint64_t draws_done);
cudaError_t launch_ising_ms_pack(const int8_t *d_spins, uint32_t *planes, uint32_t L, cudaStream_t st);
cudaError_t launch_ising_ms_unpack(int8_t *d_spins, const uint32_t *planes, uint32_t L, cudaStream_t st);
cudaError_t launch_ising_ms_energy(const uint32_t *planes, uint32_t L, int64_t *d_out, cudaStream_t st);
cudaError_t launch_ising_ms_half_sweep(const rng_handle &h, uint32_t *planes, uint32_t L, const IsingTable &tab, uint64_t K,
                                       uint64_t draws_done, int colour, cudaStream_t st);
// ising_mh.cu (the paper's double-checkerboard multi-hit kernel; one launch per coarse colour)
cudaError_t launch_ising_multihit(const rng_handle &h, int8_t *d_spins, uint32_t L, const IsingTable &tab, uint32_t T,
                                  uint32_t k_hits, uint64_t draws_done, int coarse, cudaStream_t st);
// the whole ising_sweep_multihit call in one cooperative launch (tiles resident in shared memory, mailbox halos)
bool ising_multihit_coop_eligible(const rng_handle &h, uint32_t L, uint32_t T, uint32_t k_hits, uint32_t n_sweeps, bool force);
cudaError_t launch_ising_multihit_coop(const rng_handle &h, int8_t *d_spins, uint32_t L, const IsingTable &tab, uint32_t T,
                                       uint32_t k_hits, uint32_t n_sweeps, uint64_t draws_done, unsigned long long *mailbox,
                                       cudaStream_t st);
cudaError_t launch_ising_init_random(int8_t *d_spins, uint32_t L, uint64_t seed, cudaStream_t st);
cudaError_t launch_ising_energy(const int8_t *d_spins, uint32_t L, int64_t *d_out, cudaStream_t st);

} // namespace rngb200
