// ising_static.cu -- ising_sweep_philox_static: the multi-spin Ising sweep for callers that must not allocate.
//
// Who this is for.  Some programs that want to run a sweep are not in a position to ask CUDA for memory at
// that moment: a simulation that shares the GPU with a framework whose caching allocator already holds all of
// HBM (cudaMalloc would fail, or evict the framework's cache); a time-critical loop with other streams in flight
// (cudaMalloc and cudaFree synchronise the whole device); a process held to a fixed memory budget that was
// accounted for when the library was loaded.  ising_sweep() is no use to them twice over: the handle it needs
// comes from rng_create (cudaMalloc), and its multi-spin path allocates the two bit planes it works on.
//
// What it does instead.  The generator is Philox4x32-10, which has no stored state (key = stream id ^ seed,
// counter = draw index: PAPER.md:284-296), so no handle exists; the caller carries `draws_done` itself.  The bit
// planes -- the one piece of scratch the kernels of ising_ms.cu need beyond the caller's lattice -- live in the
// file-scope device array below, which is part of the library image: every GPU on which the library's module is
// loaded holds these 2 MiB from then until the process exits, whether or not this entry point is ever called.
// That fixes the largest lattice at L = 4096 (L*L/8 bytes of planes); anything larger is refused, never grown.
//
// The kernels are exactly those ising_sweep() launches (pack, half-sweeps, energy, unpack); only the origin of the
// planes pointer differs, so the trajectory is bit-identical to ising_sweep() on an RNG_PHILOX4X32_10 handle with
// the same n_streams, seed and draws_done.
#include <mutex>

#include "internal.h"

using namespace rngb200;

namespace {

constexpr uint32_t kStaticMaxL = RNG_ISING_STATIC_MAX_L;
constexpr uint64_t kStaticPlaneWords = (uint64_t)kStaticMaxL * kStaticMaxL / 32; // two planes of L*L/64 words each

// The scratch.  In HOST code this name is only a stand-in the runtime uses to find the symbol -- it is not a
// device address and must never be handed to a kernel.  The address each device gives the array is asked for
// once per device by static_planes() below.
static __device__ __align__(256) uint32_t g_static_planes[kStaticPlaneWords];

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
uint32_t *g_planes_on_device[kMaxDevices]; // device address of g_static_planes on device i, or NULL = not asked yet

// Device address of the scratch array on `device`, which must be the current device.  The first call per device
// asks the runtime (cudaGetSymbolAddress: this may load the library's module on that device, which is why the
// first call should not come inside a stream capture); later calls read the cached pointer.
int static_planes(int device, uint32_t **out)
{
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_planes_on_device[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_planes);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return report_error(RNG_E_CUDA, "ising_sweep_philox_static: cudaGetSymbolAddress on device %d: %s", device,
                                cudaGetErrorString(e));
        }
        g_planes_on_device[device] = (uint32_t *)p;
    }
    *out = g_planes_on_device[device];
    return RNG_OK;
}

#define CU_STATIC(call)                                                                                              \
    do {                                                                                                             \
        const cudaError_t e__ = (call);                                                                              \
        if (e__ != cudaSuccess)                                                                                      \
            return report_error(RNG_E_CUDA, "ising_sweep_philox_static: %s: %s", #call, cudaGetErrorString(e__));    \
    } while (0)

} // namespace

extern "C" int ising_sweep_philox_static(uint64_t n_streams, uint64_t seed, uint64_t draws_done, int8_t *d_spins, uint32_t L,
                                         double beta, uint32_t n_sweeps, int64_t *d_energy_trace, void *cuda_stream)
{
    const char *me = "ising_sweep_philox_static";
    if (!d_spins) return report_error(RNG_E_INVAL, "%s: d_spins is NULL", me);
    if (((uintptr_t)d_spins & 15u) != 0) return report_error(RNG_E_INVAL, "%s: d_spins must be 16-byte aligned", me);
    if (d_energy_trace && ((uintptr_t)d_energy_trace & 7u) != 0)
        return report_error(RNG_E_INVAL, "%s: d_energy_trace must be 8-byte aligned", me);
    if (L > kStaticMaxL)
        return report_error(RNG_E_INVAL, "%s: L = %u is beyond the built-in scratch (L <= %u: %llu bytes of bit planes)", me, L,
                            kStaticMaxL, (unsigned long long)(kStaticPlaneWords * 4));
    if (L < 64 || L % 64u) return report_error(RNG_E_INVAL, "%s: L must be a multiple of 64 (32 sites of one colour per word)", me);
    if (!(beta >= 0.0)) return report_error(RNG_E_INVAL, "%s: beta must be >= 0 (and not NaN)", me);
    const uint64_t half = (uint64_t)L * L / 2;
    if (n_streams < 1 || half % n_streams) return report_error(RNG_E_INVAL, "%s: n_streams must divide L*L/2", me);
    const uint64_t K = half / n_streams;
    if (!(K == 4 || K == 8 || K == 16 || K % 32 == 0))
        return report_error(RNG_E_INVAL, "%s: sites per stream and colour K = L*L/2/n_streams must be 4, 8, 16 or a multiple of 32", me);
    if (draws_done & 3ull) return report_error(RNG_E_INVAL, "%s: draws_done must be a multiple of 4 (whole Philox blocks)", me);
    if ((n_sweeps && 2 * K > UINT64_MAX / n_sweeps) || draws_done + 2 * K * n_sweeps < draws_done)
        return report_error(RNG_E_INVAL, "%s: draw counter would overflow", me);
    if (n_sweeps == 0) return RNG_OK;

    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return report_error(RNG_E_CUDA, "%s: no current CUDA device (this library has no CPU fallback)", me);
    }
    if (dev < 0 || dev >= kMaxDevices) return report_error(RNG_E_UNSUPPORTED, "%s: device ordinal %d not supported", me, dev);
    uint32_t *planes = nullptr;
    if (int rc = static_planes(dev, &planes)) return rc;

    // a handle-shaped description of the generator on the host stack: Philox owns no device memory
    rng_handle h{};
    h.device = dev;
    h.api_kind = RNG_PHILOX4X32_10;
    h.g.kind = RNG_PHILOX4X32_10;
    h.g.S = n_streams;
    h.g.first = 0;
    h.g.n_total = n_streams;
    h.g.seed = seed;
    h.g.draws_done = draws_done;
    h.g.k_one = 1u;
    h.g.k_zero = 0u;

    IsingTable tab;
    ising_accept_table(beta, nullptr, tab.T);
    if (!ising_ms_eligible(h, L, tab, K, draws_done))
        return report_error(RNG_E_UNSUPPORTED, "%s: this geometry has no multi-spin kernel", me);

    // Nothing in the planes has to start at zero: the pack kernel overwrites all 2 * L*L/64 words this call
    // reads before the first half-sweep, so whatever the previous call left behind is never seen.
    cudaStream_t st = (cudaStream_t)cuda_stream;
    uint64_t d = draws_done;
    CU_STATIC(launch_ising_ms_pack(d_spins, planes, L, st));
    for (uint32_t t = 0; t < n_sweeps; t++) {
        for (int c = 0; c < 2; c++) {
            CU_STATIC(launch_ising_ms_half_sweep(h, planes, L, tab, K, d, c, st));
            d += K;
        }
        if (d_energy_trace) CU_STATIC(launch_ising_ms_energy(planes, L, d_energy_trace + t, st)); // memsets its own output
    }
    CU_STATIC(launch_ising_ms_unpack(d_spins, planes, L, st));
    return RNG_OK;
}
