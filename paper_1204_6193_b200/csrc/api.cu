// api.cu -- the C-ABI of include/rng_b200.h: argument checking, handle ownership, launch
// sequencing.  No arithmetic of the method lives here except the host-side evaluation of
// the five-entry Metropolis table, which the paper's method itself places on the host
// ("precomputed acceptance table", BASELINE.json config 5).  There is NO CPU fallback:
// without a CUDA device every compute entry point returns RNG_E_CUDA.
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "internal.h"

using namespace rngb200;

namespace {
thread_local char g_err[512] = "";
std::atomic<uint64_t> g_launches{0};

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}
int cuda_fail(cudaError_t e, const char *what)
{
    return fail(e == cudaErrorMemoryAllocation ? RNG_E_NOMEM : RNG_E_CUDA, "%s: %s", what, cudaGetErrorString(e));
}
#define CU(call)                                                   \
    do {                                                           \
        cudaError_t e__ = (call);                                  \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call);      \
    } while (0)

bool aligned(const void *p, uintptr_t a) { return ((uintptr_t)p & (a - 1)) == 0; }

bool mul_overflows(uint64_t a, uint64_t b) { return b && a > UINT64_MAX / b; }

int ensure_staging(rng_handle *h, uint64_t bytes)
{
    if (h->staging_bytes >= bytes) return RNG_OK;
    if (h->staging) cudaFree(h->staging);
    h->staging = nullptr;
    h->staging_bytes = 0;
    CU(cudaMalloc(&h->staging, bytes));
    h->staging_bytes = bytes;
    return RNG_OK;
}
} // namespace

namespace rngb200 {
void count_launch(uint64_t n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
// for entry points that live in other files: leaves the message where rng_last_error() finds it, returns `code`
int report_error(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}
int sm_count(int device)
{
    static std::atomic<int> cache[64];
    if (device < 0 || device >= 64) return 148;
    int v = cache[device].load(std::memory_order_relaxed);
    if (v <= 0) {
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || v <= 0) {
            cudaGetLastError();
            v = 148;
        }
        cache[device].store(v, std::memory_order_relaxed);
    }
    return v;
}
} // namespace rngb200

namespace {
// a handle's buffers live on the device that was current at rng_create: every entry point that launches on them
// must be called with that device current (launch configuration and function attributes are per device too)
int check_device(const rng_handle *h, const char *name)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return fail(RNG_E_CUDA, "%s: no current CUDA device", name);
    }
    if (dev != h->device)
        return fail(RNG_E_INVAL, "%s: handle was created on device %d but device %d is current", name, h->device, dev);
    return RNG_OK;
}
#define CHECK_DEVICE(h, name)                  \
    do {                                       \
        int rc__ = check_device((h), (name));  \
        if (rc__) return rc__;                 \
    } while (0)
// a launch inside a multi-launch call failed: the launches before it are enqueued and will advance the generator
// state, so the handle's draw counter must say so before the error is returned
#define CU_AT(call, h, d)                               \
    do {                                                \
        cudaError_t e__ = (call);                       \
        if (e__ != cudaSuccess) {                       \
            (h)->g.draws_done = (d);                    \
            return cuda_fail(e__, #call);               \
        }                                               \
    } while (0)
} // namespace

extern "C" {

const char *rng_last_error(void) { return g_err; }
const char *rng_version(void) { return "rng_b200 0.1 sm_100a"; }
uint64_t rng_kernel_launches(void) { return g_launches.load(); }

uint64_t rng_state_bytes(int kind, uint64_t n)
{
    switch (kind) {
    case RNG_LCG64:
    case RNG_LCG64_LEAPFROG:
    case RNG_LCG64_BOTH:
    case RNG_MWC: return 8 * n;
    case RNG_XORWOW: return 24 * n;
    case RNG_MWC_MULTI: return 12 * n;
    case RNG_XS1024W:
    case RNG_XS1024W_SKIP:
    case RNG_LCG32:
    case RNG_LCG32_LEAPFROG: return 4 * n;
    case RNG_LFIB521: return 4ull * 521ull * (n / 256);
    case RNG_LFIB1279: return 4ull * 1279ull * (n / 256);
    default: return 0;
    }
}

int rng_create_shard(int kind, uint64_t n_total, uint64_t first, uint64_t n_local, uint64_t seed, rng_handle **out)
{
    if (!out) return fail(RNG_E_INVAL, "rng_create: out is NULL");
    *out = nullptr;
    if (kind < RNG_LCG64 || kind > RNG_MWC_MULTI) return fail(RNG_E_INVAL, "rng_create: unknown kind %d", kind);
    if (n_local < 1 || first + n_local < first || first + n_local > n_total)
        return fail(RNG_E_INVAL, "rng_create: stream range [%llu,+%llu) not inside [0,%llu)", (unsigned long long)first,
                    (unsigned long long)n_local, (unsigned long long)n_total);
    if ((kind == RNG_XS1024W || kind == RNG_XS1024W_SKIP) && ((first | n_local) & 31ull))
        return fail(RNG_E_INVAL, "rng_create: RNG_XS1024W needs whole 32-stream instances");
    if ((kind == RNG_LFIB521 || kind == RNG_LFIB1279) && ((first | n_local) & 255ull))
        return fail(RNG_E_INVAL, "rng_create: RNG_LFIB* needs whole 256-stream instances");
    if (n_local > (1ull << 38)) return fail(RNG_E_INVAL, "rng_create: too many streams");
    int dev = 0, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(RNG_E_CUDA, "rng_create: no CUDA device (this library has no CPU fallback)");
    }
    CU(cudaGetDevice(&dev));
    rng_handle *h = new (std::nothrow) rng_handle();
    if (!h) return fail(RNG_E_NOMEM, "rng_create: host allocation failed");
    memset(h, 0, sizeof *h);
    h->device = dev;
    h->api_kind = kind;
    h->g.kind = (kind == RNG_XS1024W_SKIP) ? RNG_XS1024W : kind; // same generator, other seeding
    h->g.S = n_local;
    h->g.first = first;
    h->g.n_total = n_total;
    h->g.seed = seed;
    h->g.draws_done = 0;
    h->g.k_one = 1u;
    h->g.k_zero = 0u;
    h->state_bytes = rng_state_bytes(kind, n_local);
    cudaError_t e = cudaSuccess;
    LcgTable *tab = nullptr;
    if (h->state_bytes) e = cudaMalloc(&h->g.state, h->state_bytes);
    if (e == cudaSuccess && (kind == RNG_LCG64 || kind == RNG_LCG64_LEAPFROG || kind == RNG_LCG32_LEAPFROG))
        e = cudaMalloc(&tab, sizeof(LcgTable));
    h->g.lcg = tab;
    if (e == cudaSuccess) e = cudaMalloc(&h->energy_scratch, 2 * sizeof(int64_t));
    if (e == cudaSuccess) {
        h->ticket = (uint64_t *)(h->energy_scratch + 1);
        e = cudaMemsetAsync(h->ticket, 0, sizeof(uint64_t), 0);
    }
    if (e == cudaSuccess)
        e = (kind == RNG_XS1024W_SKIP)                       ? launch_seed_xs1024_skip(h->g, h->device, 0)
            : (kind == RNG_LFIB521 || kind == RNG_LFIB1279) ? launch_seed_lfib(h->g, 0)
            : (kind == RNG_MWC_MULTI)                       ? launch_seed_mwc_multi(h->g, 0)
                                                            : launch_seed(h->g, tab, 0);
    if (e == cudaSuccess) e = cudaStreamSynchronize(0);
    if (e != cudaSuccess) {
        int rc = cuda_fail(e, "rng_create");
        rng_destroy(h);
        return rc;
    }
    *out = h;
    return RNG_OK;
}

int rng_create(int kind, uint64_t n_streams, uint64_t seed, rng_handle **out)
{
    return rng_create_shard(kind, n_streams, 0, n_streams, seed, out);
}

int rng_destroy(rng_handle *h)
{
    if (!h) return RNG_OK;
    if (h->g.state) cudaFree(h->g.state);
    if (h->g.lcg) cudaFree((void *)h->g.lcg);
    if (h->staging) cudaFree(h->staging);
    if (h->energy_scratch) cudaFree(h->energy_scratch);
    if (h->ms_planes) cudaFree(h->ms_planes);
    if (h->mh_mailbox) cudaFree(h->mh_mailbox);
    delete h;
    return RNG_OK;
}

static int fill_common(rng_handle *h, void *d_out, uint64_t n, bool f32, void *stream, const char *name)
{
    if (!h) return fail(RNG_E_INVAL, "%s: handle is NULL", name);
    if (n == 0) return RNG_OK;
    if (!d_out) return fail(RNG_E_INVAL, "%s: d_out is NULL", name);
    if (!aligned(d_out, 16)) return fail(RNG_E_INVAL, "%s: d_out must be 16-byte aligned", name);
    if (mul_overflows(h->g.S, n) || h->g.S * n > (1ull << 60)) return fail(RNG_E_INVAL, "%s: n_streams*n too large", name);
    if (h->g.draws_done + n < n) return fail(RNG_E_INVAL, "%s: draw counter would overflow", name);
    CHECK_DEVICE(h, name);
    CU(launch_fill(*h, d_out, n, f32, (cudaStream_t)stream));
    h->g.draws_done += n;
    return RNG_OK;
}

int rng_fill_u32(rng_handle *h, uint32_t *d_out, uint64_t n, void *stream)
{
    return fill_common(h, d_out, n, false, stream, "rng_fill_u32");
}
int rng_fill_f32(rng_handle *h, float *d_out, uint64_t n, void *stream)
{
    return fill_common(h, d_out, n, true, stream, "rng_fill_f32");
}

int rng_draw_reduce(rng_handle *h, uint32_t *d_out, uint64_t n, void *stream)
{
    if (!h) return fail(RNG_E_INVAL, "rng_draw_reduce: handle is NULL");
    if (!d_out) return fail(RNG_E_INVAL, "rng_draw_reduce: d_out is NULL");
    if (!aligned(d_out, 8)) return fail(RNG_E_INVAL, "rng_draw_reduce: d_out must be 8-byte aligned");
    if (h->g.draws_done + n < n) return fail(RNG_E_INVAL, "rng_draw_reduce: draw counter would overflow");
    CHECK_DEVICE(h, "rng_draw_reduce");
    CU(launch_draw_reduce(*h, d_out, n, (cudaStream_t)stream));
    h->g.draws_done += n;
    return RNG_OK;
}

int ising_accept_table(double beta, float P_out[5], uint32_t T_out[5])
{
    for (int i = 0; i < 5; i++) {
        const float P = (float)exp(-2.0 * beta * (double)(2 * i - 4)); // Metropolis min(1, e^{-beta dE}), dE = 2h
        if (P_out) P_out[i] = P;
        if (T_out) {
            const double x = ceil((double)P * 16777216.0); // exact: float times 2^24, then ceil
            T_out[i] = (x >= 16777216.0) ? 16777216u : (x > 0.0 ? (uint32_t)x : 0u);
        }
    }
    return RNG_OK;
}

int ising_sweep(rng_handle *h, int8_t *d_spins, uint32_t L, double beta, uint32_t n_sweeps, int64_t *d_trace,
                void *stream)
{
    if (!h) return fail(RNG_E_INVAL, "ising_sweep: handle is NULL");
    if (!d_spins) return fail(RNG_E_INVAL, "ising_sweep: d_spins is NULL");
    if (L < 4 || (L & 1u)) return fail(RNG_E_INVAL, "ising_sweep: L must be even and >= 4");
    if (!aligned(d_spins, 16)) return fail(RNG_E_INVAL, "ising_sweep: d_spins must be 16-byte aligned");
    if (!(beta == beta)) return fail(RNG_E_INVAL, "ising_sweep: beta is NaN");
    const uint64_t half = (uint64_t)L * L / 2;
    if (half % h->g.S) return fail(RNG_E_INVAL, "ising_sweep: n_streams must divide L*L/2");
    const uint64_t K = half / h->g.S;
    if (mul_overflows(2 * K, n_sweeps) || h->g.draws_done + 2 * K * n_sweeps < h->g.draws_done)
        return fail(RNG_E_INVAL, "ising_sweep: draw counter would overflow");
    CHECK_DEVICE(h, "ising_sweep");
    IsingTable tab;
    ising_accept_table(beta, nullptr, tab.T);
    cudaStream_t st = (cudaStream_t)stream;
    uint64_t d = h->g.draws_done;
    if (n_sweeps == 0) return RNG_OK;
    // variant "ising": 0 = automatic (multi-spin bit planes when the geometry allows and the pack/unpack
    // pays off, else the byte kernels), 1 = generic byte kernel only, 2 = byte kernels only, 3 = multi-spin
    // whenever eligible.  Every variant produces the same trajectory.
    const bool want_ms = h->var_ising == 3 || (h->var_ising == 0 && n_sweeps >= 2);
    if (want_ms && ising_ms_eligible(*h, L, tab, K, d)) {
        const uint64_t need = (uint64_t)L * L / 8; // two planes of L*L/64 words
        if (h->ms_planes_bytes < need) {
            if (h->ms_planes) cudaFree(h->ms_planes);
            h->ms_planes = nullptr;
            h->ms_planes_bytes = 0;
            CU(cudaMalloc((void **)&h->ms_planes, need));
            h->ms_planes_bytes = need;
        }
        CU(launch_ising_ms_pack(d_spins, h->ms_planes, L, st));
        for (uint32_t t = 0; t < n_sweeps; t++) {
            for (int c = 0; c < 2; c++) {
                CU_AT(launch_ising_ms_half_sweep(*h, h->ms_planes, L, tab, K, d, c, st), h, d);
                d += K;
            }
            if (d_trace) CU_AT(launch_ising_ms_energy(h->ms_planes, L, d_trace + t, st), h, d);
        }
        CU_AT(launch_ising_ms_unpack(d_spins, h->ms_planes, L, st), h, d);
        h->g.draws_done = d;
        return RNG_OK;
    }
    for (uint32_t t = 0; t < n_sweeps; t++) {
        for (int c = 0; c < 2; c++) {
            CU_AT(launch_ising_half_sweep(*h, d_spins, L, tab, K, d, c, st), h, d);
            d += K;
        }
        if (d_trace) CU_AT(launch_ising_energy(d_spins, L, d_trace + t, st), h, d);
    }
    h->g.draws_done = d;
    return RNG_OK;
}

int ising_sweep_multihit(rng_handle *h, int8_t *d_spins, uint32_t L, double beta, uint32_t n_sweeps, uint32_t tile,
                         uint32_t k_hits, int64_t *d_trace, void *stream)
{
    if (!h) return fail(RNG_E_INVAL, "ising_sweep_multihit: handle is NULL");
    if (!d_spins) return fail(RNG_E_INVAL, "ising_sweep_multihit: d_spins is NULL");
    if (!aligned(d_spins, 16)) return fail(RNG_E_INVAL, "ising_sweep_multihit: d_spins must be 16-byte aligned");
    if (!(beta == beta)) return fail(RNG_E_INVAL, "ising_sweep_multihit: beta is NaN");
    if (tile < 2 || (tile & 1u) || tile > 44u || L < 2 * tile || L % tile || ((L / tile) & 1u))
        return fail(RNG_E_INVAL, "ising_sweep_multihit: tile must be even, 2..44, divide L, with L/tile even");
    if (k_hits < 1) return fail(RNG_E_INVAL, "ising_sweep_multihit: k_hits must be >= 1");
    if (h->g.S != (uint64_t)L * L / 4) return fail(RNG_E_INVAL, "ising_sweep_multihit: needs n_streams == L*L/4");
    if ((h->g.kind == RNG_LFIB521 || h->g.kind == RNG_LFIB1279) && tile != 8u && tile != 16u)
        return fail(RNG_E_UNSUPPORTED, "ising_sweep_multihit: RNG_LFIB* shares its ring across a 256-thread CTA: tile 8 or 16 only");
    if (h->g.kind == RNG_XS1024W && (tile * tile / 2u) % 32u)
        return fail(RNG_E_INVAL, "ising_sweep_multihit: this kind needs whole warps per tile (tile a multiple of 8)");
    const uint64_t per_sweep = 4ull * k_hits;
    if (mul_overflows(per_sweep, n_sweeps) || h->g.draws_done + per_sweep * n_sweeps < h->g.draws_done)
        return fail(RNG_E_INVAL, "ising_sweep_multihit: draw counter would overflow");
    CHECK_DEVICE(h, "ising_sweep_multihit");
    IsingTable tab;
    ising_accept_table(beta, nullptr, tab.T);
    cudaStream_t st = (cudaStream_t)stream;
    uint64_t d = h->g.draws_done;
    if (n_sweeps == 0) return RNG_OK;
    // variant "ising": 0 = automatic (the whole call in ONE cooperative launch where that is faster: no energy trace
    // asked for, every tile resident, few hits -- PAPER.md:58's k = 1 regime without its launches and its per-visit
    // state traffic), 1 = always one launch per coarse colour, 4 = one launch whenever the call qualifies.
    // Same trajectory either way.
    if (!d_trace && h->var_ising != 1 && ising_multihit_coop_eligible(*h, L, tile, k_hits, n_sweeps, h->var_ising == 4)) {
        const uint64_t need = (uint64_t)(L / tile) * (L / tile) * 4ull * sizeof(unsigned long long);
        if (h->mh_mailbox_bytes < need) {
            if (h->mh_mailbox) cudaFree(h->mh_mailbox);
            h->mh_mailbox = nullptr;
            h->mh_mailbox_bytes = 0;
            CU(cudaMalloc((void **)&h->mh_mailbox, need));
            h->mh_mailbox_bytes = need;
        }
        const cudaError_t ce = launch_ising_multihit_coop(*h, d_spins, L, tab, tile, k_hits, n_sweeps, d, h->mh_mailbox, st);
        if (ce == cudaSuccess) {
            h->g.draws_done = d + per_sweep * n_sweeps;
            return RNG_OK;
        }
        // The one launch was refused (not every CTA can be resident: MPS or partition limits, fewer SMs than planned).
        // Nothing of it ran -- the zeroed mailbox is harmless -- so in automatic mode the call is served by the
        // per-colour launches below, as it was before the one-launch path existed; only variant 4 (forced) reports it.
        if (h->var_ising == 4) return cuda_fail(ce, "launch_ising_multihit_coop");
        cudaGetLastError();
    }
    for (uint32_t t = 0; t < n_sweeps; t++) {
        for (int c = 0; c < 2; c++) {
            CU_AT(launch_ising_multihit(*h, d_spins, L, tab, tile, k_hits, d, c, st), h, d);
            d += 2ull * k_hits;
        }
        if (d_trace) CU_AT(launch_ising_energy(d_spins, L, d_trace + t, st), h, d);
    }
    h->g.draws_done = d;
    return RNG_OK;
}

int ising_init_random(int8_t *d_spins, uint32_t L, uint64_t seed, void *stream)
{
    if (!d_spins || L < 2 || !aligned(d_spins, 16)) return fail(RNG_E_INVAL, "ising_init_random: bad arguments");
    CU(launch_ising_init_random(d_spins, L, seed, (cudaStream_t)stream));
    return RNG_OK;
}

int ising_energy(const int8_t *d_spins, uint32_t L, int64_t *d_out, void *stream)
{
    if (!d_spins || !d_out || L < 2 || !aligned(d_out, 8)) return fail(RNG_E_INVAL, "ising_energy: bad arguments");
    CU(launch_ising_energy(d_spins, L, d_out, (cudaStream_t)stream));
    return RNG_OK;
}

// ---- host-buffer entry points -------------------------------------------------------
static int fill_host_common(rng_handle *h, void *h_out, uint64_t n, bool f32, void *stream, const char *name)
{
    if (!h) return fail(RNG_E_INVAL, "%s: handle is NULL", name);
    if (n == 0) return RNG_OK;
    if (!h_out) return fail(RNG_E_INVAL, "%s: h_out is NULL", name);
    if (mul_overflows(h->g.S, n) || h->g.S * n > (1ull << 58)) return fail(RNG_E_INVAL, "%s: n_streams*n too large", name);
    const uint64_t bytes = h->g.S * n * 4;
    CHECK_DEVICE(h, name);
    int rc = ensure_staging(h, bytes);
    if (rc) return rc;
    rc = fill_common(h, h->staging, n, f32, stream, name);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h_out, h->staging, bytes, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    return RNG_OK;
}
int rng_fill_u32_host(rng_handle *h, uint32_t *h_out, uint64_t n, void *stream)
{
    return fill_host_common(h, h_out, n, false, stream, "rng_fill_u32_host");
}
int rng_fill_f32_host(rng_handle *h, float *h_out, uint64_t n, void *stream)
{
    return fill_host_common(h, h_out, n, true, stream, "rng_fill_f32_host");
}
int rng_draw_reduce_host(rng_handle *h, uint32_t *h_out, uint64_t n, void *stream)
{
    if (!h || !h_out) return fail(RNG_E_INVAL, "rng_draw_reduce_host: NULL argument");
    const uint64_t bytes = h->g.S * 8;
    CHECK_DEVICE(h, "rng_draw_reduce_host");
    int rc = ensure_staging(h, bytes);
    if (rc) return rc;
    rc = rng_draw_reduce(h, (uint32_t *)h->staging, n, stream);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h_out, h->staging, bytes, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    return RNG_OK;
}
int ising_sweep_host(rng_handle *h, int8_t *h_spins, uint32_t L, double beta, uint32_t n_sweeps, int64_t *h_trace,
                     void *stream)
{
    if (!h || !h_spins) return fail(RNG_E_INVAL, "ising_sweep_host: NULL argument");
    if (L < 4 || (L & 1u)) return fail(RNG_E_INVAL, "ising_sweep_host: L must be even and >= 4");
    const uint64_t N = (uint64_t)L * L;
    const uint64_t sp_bytes = (N + 15) & ~15ull, tr_bytes = h_trace ? 8ull * n_sweeps : 0;
    CHECK_DEVICE(h, "ising_sweep_host");
    int rc = ensure_staging(h, sp_bytes + tr_bytes);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    int8_t *d_sp = (int8_t *)h->staging;
    int64_t *d_tr = h_trace ? (int64_t *)((char *)h->staging + sp_bytes) : nullptr;
    CU(cudaMemcpyAsync(d_sp, h_spins, N, cudaMemcpyHostToDevice, st));
    rc = ising_sweep(h, d_sp, L, beta, n_sweeps, d_tr, stream);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h_spins, d_sp, N, cudaMemcpyDeviceToHost, st));
    if (h_trace) CU(cudaMemcpyAsync(h_trace, d_tr, tr_bytes, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return RNG_OK;
}

// ---- state access --------------------------------------------------------------------
uint64_t rng_draws_done(const rng_handle *h) { return h ? h->g.draws_done : 0; }
int rng_set_draws_done(rng_handle *h, uint64_t d)
{
    if (!h) return fail(RNG_E_INVAL, "rng_set_draws_done: handle is NULL");
    h->g.draws_done = d;
    return RNG_OK;
}

int rng_get_state(rng_handle *h, void *h_buf, uint64_t bytes)
{
    if (!h) return fail(RNG_E_INVAL, "rng_get_state: handle is NULL");
    if (bytes != h->state_bytes) return fail(RNG_E_INVAL, "rng_get_state: expected %llu bytes", (unsigned long long)h->state_bytes);
    if (!bytes) return RNG_OK;
    if (!h_buf) return fail(RNG_E_INVAL, "rng_get_state: h_buf is NULL");
    CHECK_DEVICE(h, "rng_get_state");
    CU(cudaDeviceSynchronize());
    const int wps = h->g.kind == RNG_XORWOW ? 6 : h->g.kind == RNG_MWC_MULTI ? 3 : 0; // words per stream of the SoA kinds
    if (wps) { // device layout w[k*S+s] -> canonical [s][k]
        uint32_t *tmp = new (std::nothrow) uint32_t[h->g.S * wps]; // nothing may throw across the C boundary
        if (!tmp) return fail(RNG_E_NOMEM, "rng_get_state: host allocation of %llu bytes failed", (unsigned long long)bytes);
        const cudaError_t e = cudaMemcpy(tmp, h->g.state, bytes, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) {
            delete[] tmp;
            return cuda_fail(e, "rng_get_state: cudaMemcpy");
        }
        uint32_t *o = (uint32_t *)h_buf;
        for (uint64_t s = 0; s < h->g.S; s++)
            for (int k = 0; k < wps; k++) o[wps * s + k] = tmp[k * h->g.S + s];
        delete[] tmp;
    } else {
        CU(cudaMemcpy(h_buf, h->g.state, bytes, cudaMemcpyDeviceToHost));
    }
    return RNG_OK;
}

int rng_set_state(rng_handle *h, const void *h_buf, uint64_t bytes)
{
    if (!h) return fail(RNG_E_INVAL, "rng_set_state: handle is NULL");
    if (bytes != h->state_bytes) return fail(RNG_E_INVAL, "rng_set_state: expected %llu bytes", (unsigned long long)h->state_bytes);
    if (!bytes) return RNG_OK;
    if (!h_buf) return fail(RNG_E_INVAL, "rng_set_state: h_buf is NULL");
    CHECK_DEVICE(h, "rng_set_state");
    CU(cudaDeviceSynchronize());
    const int wps = h->g.kind == RNG_XORWOW ? 6 : h->g.kind == RNG_MWC_MULTI ? 3 : 0;
    if (wps) {
        uint32_t *tmp = new (std::nothrow) uint32_t[h->g.S * wps];
        if (!tmp) return fail(RNG_E_NOMEM, "rng_set_state: host allocation of %llu bytes failed", (unsigned long long)bytes);
        const uint32_t *in = (const uint32_t *)h_buf;
        for (uint64_t s = 0; s < h->g.S; s++)
            for (int k = 0; k < wps; k++) tmp[k * h->g.S + s] = in[wps * s + k];
        const cudaError_t e = cudaMemcpy(h->g.state, tmp, bytes, cudaMemcpyHostToDevice);
        delete[] tmp;
        if (e != cudaSuccess) return cuda_fail(e, "rng_set_state: cudaMemcpy");
    } else {
        CU(cudaMemcpy(h->g.state, h_buf, bytes, cudaMemcpyHostToDevice));
    }
    return RNG_OK;
}

int rng_set_variant(rng_handle *h, const char *name, int value)
{
    if (!h || !name || value < 0) return fail(RNG_E_INVAL, "rng_set_variant: bad arguments");
    if (!strcmp(name, "xs1024")) h->var_xs1024 = value;
    else if (!strcmp(name, "ising")) h->var_ising = value;
    else if (!strcmp(name, "store")) h->var_store = value;
    else if (!strcmp(name, "lcg")) h->var_lcg = value;
    else if (!strcmp(name, "xsfill")) h->var_xsfill = value;
    else if (!strcmp(name, "cvt")) h->var_cvt = value;
    else return fail(RNG_E_INVAL, "rng_set_variant: unknown name '%s'", name);
    return RNG_OK;
}

} // extern "C"
