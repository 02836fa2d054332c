/*
 * rng_b200.h -- C-ABI boundary of the B200-native (sm_100a) implementation of
 * the hot path of Manssen, Weigel & Hartmann, "Random number generators for
 * massively parallel simulations on GPU" (arXiv:1204.6193):
 *
 *     many independent per-thread pseudo-random streams, seeded and advanced in
 *     parallel, their output either written in bulk to HBM or
 *     drawn in-register by a consumer kernel, the consumer
 *     being the checkerboard Metropolis sweep of the 2D Ising model the paper
 *     uses as its application test.
 *
 * Citations are lines of /root/reference/PAPER.md ("PAPER.md:<line>") or a
 * reading listed in DESIGN.md section 3 ("R-<id>").
 *
 * General conventions
 * -------------------
 *  - Every function returns RNG_OK (0) or a negative error code; nothing throws,
 *    aborts or prints.  rng_last_error() returns a thread-local message for the
 *    last failing call of the calling thread.
 *  - Pointers named d_* are DEVICE pointers owned by the caller (e.g. PyTorch
 *    tensors), 16-byte aligned unless stated, on the device that was current
 *    when the handle was created; every call that takes a handle must be made
 *    with that device current (RNG_E_INVAL otherwise: the handle's state, its
 *    staging buffers and its launch geometry belong to that device).  Calls on
 *    ONE handle must not overlap (different handles may run on different
 *    streams concurrently).  Pointers named h_* are HOST pointers owned by
 *    the caller (pinned memory makes the copies asynchronous, pageable works).
 *    The library never allocates or frees caller buffers.
 *  - `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default
 *    stream).  Device-pointer calls only enqueue work and return without
 *    synchronising.  Host-pointer calls (`*_host`) return after the result is
 *    in the host buffer.
 *  - A handle owns its generator state (device memory).  All streams of a handle
 *    advance in lockstep: every call consumes the same number of draws from
 *    every stream, and successive calls CONTINUE the streams:
 *    fill(n) followed by fill(m) produces exactly what fill(n+m) would.
 *  - Canonical output layout is stream-major:  out[s*n + j] = draw j (of this
 *    call) of local stream s  (BASELINE.json config 1: "per stream to a flat
 *    array").
 *  - A call that issues several launches (ising_sweep, ising_sweep_multihit) and
 *    fails at one of them leaves draws_done at the draws already enqueued, so
 *    the handle's position stays equal to its device state.
 *  - No CPU fallback exists: without a CUDA device every call that needs one
 *    fails with RNG_E_CUDA.
 */
#ifndef RNG_B200_H
#define RNG_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rng_handle rng_handle; /* opaque */

/* Generator kinds.  Stream s below is the GLOBAL stream id (first + local index);
 * SM_seed[k] is the k-th (0-based) output of splitmix64 started at `seed` (R-S1). */
enum {
    /* x <- a x + c mod 2^64, a = 2862933555777941757, c = 1442695040888963407
     * (eq.(1), :46); draw j = 32 most significant bits of x_j
     * (R-A3: output, then advance); x_0 of stream s = SM_seed[s]
     * ("random" seeding). */
    RNG_LCG64 = 0,
    /* the paper's sub-stream method (eq.(2),(3)): ONE global
     * sequence X_0 = SM_seed[0], stream s draw j = hi32(X_{s + j*n_total}). */
    RNG_LCG64_LEAPFROG = 1,
    /* Marsaglia's XORWOW (recurrence of Ref.[30], R-B1):
     * t=x^(x>>2); x=y; y=z; z=w; w=v; v=(v^(v<<4))^(t^(t<<1)); d+=362437;
     * return d+v.  Seeding: (x,y),(z,w),(v,d) = (lo32,hi32) of SM_seed[3s],
     * SM_seed[3s+1], SM_seed[3s+2]; if x|y|z|w|v == 0 then v = 1 (R-B2, R-B3). */
    RNG_XORWOW = 2,
    /* Philox4x32-10 (constants of Ref.[20], R-C1).  Key =
     * s XOR seed (64 bit, low word = k0); counter = (lo32(b), hi32(b), 0, 0) with
     * b = floor(j/4) the 4-word block index over the handle's lifetime; draw j
     * is word j mod 4 of that block (BASELINE.json config 2, R-C2).  Stateless. */
    RNG_PHILOX4X32_10 = 3,
    /* The paper's XORShift1024/Weyl generator (eq.(8), :177,
     * :201-225 Listing 1, :232-240).  One 1024-bit instance per WARP: streams
     * 32g..32g+31 are the 32 words of instance g, word 0 most significant
     * (R-D1, R-D4).  Update X ^= X<<329; X ^= X>>347; X ^= X<<344 (zeros shift
     * in); output of the n-th update since creation: (y ^ (y>>16)) + x_word with
     * y = n*362437 mod 2^32 (R-D6).  Seeding ("sloppy" variant, PAPER.md:230,
     * R-D7): words 2k, 2k+1 of instance g = lo32, hi32 of SM_seed[16g+k]; an
     * all-zero instance gets word 31 = 1.  n_streams and first must be
     * multiples of 32. */
    RNG_XS1024W = 4,
    /* Philox4x32 with 7 rounds (PAPER.md:269 Table 2, :300: "the fastest Crush-resistant"
     * variant; same S-box, constants, key schedule and stream mapping as kind 3). */
    RNG_PHILOX4X32_7 = 5,
    /* the 32-bit LCG of PAPER.md:33 eq.(1) with a = 1664525, c = 1013904223, m = 2^32
     * (Table 2 "LCG32"): draw j = x_j, the whole word (u = x/m, PAPER.md:35;
     * output, then advance); x_0 of stream s = lo32(SM_seed[s]).  Period 2^32: the paper's
     * deliberately bad example (fails SmallCrush), here for its Table-2 row. */
    RNG_LCG32 = 6,
    /* kind 4's generator seeded the way the paper itself seeds it: every
     * instance starts from ONE common state X_0 and instance g (global number, streams
     * 32g..32g+31) skips g * 2^137 updates: X_g = X_0 M^(g 2^137), M the 1024x1024 GF(2) matrix
     * of one update.  The sub-streams of 2^137 numbers are consecutive blocks of one sequence
     * and cannot overlap.  X_0 = kind 4's instance 0 (SM_seed[0..15], R-D7b).  Update, Weyl
     * term (the same for all instances: footnote 4), output, layout, state
     * access and every entry point are exactly kind 4's. */
    RNG_XS1024W_SKIP = 7,
    /* kind 0's generator and seeds "using the whole state to produce two 32-bit numbers"
     * (doubles the nominal rate, lowers the quality): draw 2i = 32 most
     * significant bits of x_i, draw 2i+1 = its 32 least significant bits, then the state
     * advances (R-F2).  State access as kind 0 (after an odd number of draws the state is
     * still x_i; the parity of draws_done says which half comes next). */
    RNG_LCG64_BOTH = 8,
    /* The paper's second generator with state shared by the threads of a block: the additive
     * lagged Fibonacci generator on floats, u_n = u_{n-r} + u_{n-s} (mod 1), single precision
     * (eq.(5)), lags (r,s) = (521,353) and (1279,861).
     * R-G1..G3: an INSTANCE (one ring buffer) serves 256 consecutive streams (n_streams and
     * first must be multiples of 256); its numbers v_0, v_1, ... are dealt round-robin, stream
     * t of the instance gets v_{256 j + t} as draw j.  Seeds: u_i of instance g, i < r, is
     * (w >> 9) 2^-23 with w the 32-bit word g r + i of the splitmix64 word sequence (word 2k =
     * lo32, 2k+1 = hi32 of SM_seed[k]); an instance without an odd multiple of 2^-23 gets
     * that bit on u_0.  All values are 23-bit fractions, every addition is exact.  fill_f32
     * writes the numbers themselves; as 32-bit integers they are (v 2^23) << 9, so the fixed
     * map (u >> 8) 2^-24 gives v back.  State: per instance its last r numbers, oldest first,
     * as float bit patterns.  ising_sweep runs on the byte kernel, ising_sweep_multihit with tile 8 or 16
     * (a CTA = one instance hosts 256 / (tile*tile/2) tiles). */
    RNG_LFIB521 = 9,
    RNG_LFIB1279 = 10,
    /* kind 1's sub-stream method for the 32-bit LCG of kind 6: ONE global sequence
     * X_0 = lo32(SM_seed[0]), stream s draw j = X_{s + j*n_total} (the whole word).  This is the paper's
     * Table 1 row "LCG32", its example of a generator that fails the application test. */
    RNG_LCG32_LEAPFROG = 11,
    /* Multiply-with-carry: x <- a x + c mod 2^32, c <- floor((a x + c) / 2^32), with the
     * paper's multiplier a = 4294967118 for every stream (Table 1 row "MWC, same a"); the draw is
     * x_n (output, then advance).  R-M1: (x_0, c_0) = (lo32, hi32 mod a) of SM_seed[s]; the fixed points (0,0)
     * and (2^32-1, a-1) are moved to (1,0) and (2^32-1, a-2).  State: n_local x {x, c} u32. */
    RNG_MWC = 12,
    /* kind 12 with ONE MULTIPLIER PER STREAM (Table 1 row "MWC, different a"): global stream s
     * uses multiplier number s, the (s+1)-th largest a < 2^32 for which a 2^32 - 1 is a safe prime (number 0 is
     * the paper's 4294967118); rng_create finds them on the device (trial division + Miller-Rabin, bases 2..37).
     * Seeds as kind 12 with the stream's own a.  State: n_local x {x, c, a} u32 ("64+32 = 96 bits"). */
    RNG_MWC_MULTI = 13
};

enum {
    RNG_OK = 0,
    RNG_E_INVAL = -1,       /* bad argument (null, misaligned, size constraint)   */
    RNG_E_NOMEM = -2,       /* host or device allocation failed                   */
    RNG_E_CUDA = -3,        /* CUDA runtime error, or no device                   */
    RNG_E_UNSUPPORTED = -4  /* valid request the library does not implement       */
};

/* ---- a1: seeding / stream setup --------------
 * rng_create: streams [0, n_streams) of n_streams.  Runs the seeding kernel on
 * the current device (legacy default stream, synchronised before returning).
 * rng_create_shard: local streams are the global streams [first, first+n_local)
 * out of n_total (for one-process-per-GPU sharding; n_total only matters for
 * RNG_LCG64_LEAPFROG, where it is the stride of the global sequence).
 * Errors: RNG_E_INVAL (n == 0, range overflow, XS1024W not in whole instances,
 * unknown kind, out == NULL), RNG_E_NOMEM, RNG_E_CUDA. */
int rng_create(int kind, uint64_t n_streams, uint64_t seed, rng_handle **out);
int rng_create_shard(int kind, uint64_t n_total, uint64_t first, uint64_t n_local,
                     uint64_t seed, rng_handle **out);
/* frees the state; NULL is allowed */
int rng_destroy(rng_handle *h);

/* ---- a2-a5,a7: fill mode -------------------------------------------------------
 * d_out[s*n + j] = draw (draws_done + j) of local stream s, s < n_local, j < n;
 * then draws_done += n.  n == 0 is a no-op.  d_out must hold n_local*n elements
 * and be 16-byte aligned (else RNG_E_INVAL).  Any n is accepted; n % 4 == 0 (and,
 * for Philox, draws_done % 4 == 0) takes the 128-bit-store path. */
int rng_fill_u32(rng_handle *h, uint32_t *d_out, uint64_t n, void *cuda_stream);
/* same stream pushed through the fixed map f = (float)(u >> 8) * 2^-24, exact,
 * in [0, 1 - 2^-24]  (BASELINE.json; the paper's u = x/m is PAPER.md:35, R-A4) */
int rng_fill_f32(rng_handle *h, float *d_out, uint64_t n, void *cuda_stream);

/* ---- a6: in-register draw mode -------------------------------------------------
 * Each stream draws n numbers that never leave the register file and reduces
 * them: d_out[2s] = XOR_j u_{s,j}, d_out[2s+1] = SUM_j u_{s,j} mod 2^32.
 * d_out holds 2*n_local uint32, 8-byte aligned.  draws_done += n.
 * (This is the mode of the paper's peak numbers.) */
int rng_draw_reduce(rng_handle *h, uint32_t *d_out, uint64_t n, void *cuda_stream);

/* ---- a8: consumer: checkerboard Metropolis sweeps of the 2D Ising model --------
 * (BASELINE.json config 5; R-E1..E8.)
 * d_spins: int8 +1/-1, row-major L x L, periodic; L even, >= 4.  Colour of (x,y)
 * is (x+y)&1; a sweep is the colour-0 half-sweep then the colour-1 half-sweep.
 * Sites of one colour are numbered q = y*(L/2) + xh with x = 2*xh + ((y+c)&1).
 * With S = n_local streams, K = (L*L/2)/S (S must divide L*L/2): stream s owns
 * q in [sK,(s+1)K) of both colours, visits them in increasing q and spends ONE
 * draw on each, accepted or not:  h = spin * (sum of its 4 neighbours);
 * flip iff (float)(r>>8)*2^-24 < P[(h+4)/2], P[i] = (float)exp(-2.0*beta*(2i-4))
 * evaluated in double on the host and rounded to float (strict <).
 * Equivalent to: per half-sweep, fill K draws per stream, then apply.
 * draws_done += 2*K*n_sweeps.  d_energy_trace: NULL, or int64[n_sweeps] (device)
 * receiving E = -sum_<ij> s_i s_j after every sweep.  Every kind is supported. */
int ising_sweep(rng_handle *h, int8_t *d_spins, uint32_t L, double beta, uint32_t n_sweeps,
                int64_t *d_energy_trace, void *cuda_stream);

/* ---- a8': the paper's own consumer: double checkerboard with multi-hit updates -------
 * (Table 1's k = 1 and k = 100 columns; reading R-E9.)
 * The lattice is cut into tile x tile tiles (tile even, 2..44, tile | L, L/tile even);
 * tile (tx,ty) has coarse colour (tx+ty)&1.  A sweep = coarse colour 0, then 1.  For one
 * coarse colour every tile of that colour receives k_hits hits; a hit = all its sites of fine
 * colour 0 ((x+y)&1 == 0), then all of fine colour 1, Metropolis rule and table as ising_sweep.
 * Streams: n_local must equal L*L/4.  Tiles of one coarse colour are numbered
 * p = ty*(L/tile/2) + txh, tx = 2*txh + ((ty+C)&1); thread t < tile*tile/2 owns, for c = 0, 1,
 * the site y_l = t/(tile/2), x_l = 2*(t%(tile/2)) + ((y_l+c)&1) of the tile; stream
 * s = p*tile*tile/2 + t serves tile p of both coarse colours and spends its draws in the order
 * (coarse colour, hit, fine colour): 4*k_hits per sweep, 2*k_hits per generator state load.
 * RNG_XS1024W / _SKIP need tile % 8 == 0; RNG_LFIB* (ring shared by a 256-thread CTA) tile 8 or 16, else
 * RNG_E_UNSUPPORTED.  d_energy_trace as in ising_sweep.
 * draws_done += 4*k_hits*n_sweeps.  Errors: RNG_E_INVAL (geometry, stream count), RNG_E_CUDA. */
int ising_sweep_multihit(rng_handle *h, int8_t *d_spins, uint32_t L, double beta, uint32_t n_sweeps,
                         uint32_t tile, uint32_t k_hits, int64_t *d_energy_trace, void *cuda_stream);

/* ---- a8 without allocation: for callers that cannot call cudaMalloc ---------------
 * ising_sweep needs a handle (rng_create allocates) and, on its multi-spin path, allocates the
 * two bit planes it works on.  That shuts out callers who cannot obtain device memory when they
 * want to sweep: a simulation sharing the GPU with a framework whose caching allocator already
 * holds all of HBM, a latency-critical loop that cannot take the device-wide synchronisation
 * cudaMalloc/cudaFree imply, a process whose memory budget was fixed when it started.  This entry
 * point serves them.  It calls no cudaMalloc, cudaFree or allocating library routine, ever:
 *  - the generator is Philox4x32-10 (kind 3), which stores no state, so there is no handle; the
 *    caller carries the stream position: pass draws_done (a multiple of 4; 0 for fresh streams) and
 *    pass draws_done + 2*K*n_sweeps to the next call, K = (L*L/2)/n_streams;
 *  - the bit planes live in a fixed array inside the library image (RNG_ISING_STATIC_MAX_L^2/8 =
 *    2 MiB).  Every GPU that loads the library holds that array until the process exits, used or
 *    not.  L > RNG_ISING_STATIC_MAX_L is refused with RNG_E_INVAL (the scratch never grows).
 * Result: d_spins (and d_energy_trace) are bit-identical to ising_sweep on a handle from
 * rng_create(RNG_PHILOX4X32_10, n_streams, seed) whose draws_done is the value passed here;
 * site numbering, acceptance rule and trace are ising_sweep's (see above).  Only the multi-spin
 * geometries are served: L a multiple of 64, 64 <= L <= RNG_ISING_STATIC_MAX_L; n_streams divides
 * L*L/2 with K = 4, 8, 16 or a multiple of 32; beta >= 0 (else RNG_E_INVAL / RNG_E_UNSUPPORTED).
 * Things to know:
 *  - the first call on each device looks up the array's device address (once per device, with
 *    that device current) and may make the runtime load the library's kernels there; make that
 *    first call during set-up, before any stream capture.  n_sweeps = 1 on a scratch lattice will do.
 *  - all calls on one device share the one array, and it keeps what the last call left.  Nothing
 *    in it has to start at zero (each call rewrites every word it later reads), but two calls that
 *    overlap on the GPU -- different streams, or different host threads -- race on it and corrupt
 *    each other's lattices.  Issue them on one stream, or order them yourself.
 *  - d_spins / d_energy_trace are the caller's device buffers, as for ising_sweep; the call only
 *    enqueues work.  After RNG_E_CUDA the lattice contents are unspecified. */
#define RNG_ISING_STATIC_MAX_L 4096u
int ising_sweep_philox_static(uint64_t n_streams, uint64_t seed, uint64_t draws_done, int8_t *d_spins, uint32_t L,
                              double beta, uint32_t n_sweeps, int64_t *d_energy_trace, void *cuda_stream);

/* helpers (not hot path) */
/* spin i = +1 if bit (i & 63) of SM_seed[i >> 6] is set, else -1 */
int ising_init_random(int8_t *d_spins, uint32_t L, uint64_t seed, void *cuda_stream);
/* *d_out = E = -sum over bonds s_i s_j, each bond once, periodic */
int ising_energy(const int8_t *d_spins, uint32_t L, int64_t *d_out, void *cuda_stream);
/* the acceptance table the sweep uses, as integers T[i] = min(2^24, ceil(P[i]*2^24)):
 * (r>>8) < T[i]  <=>  (float)(r>>8)*2^-24 < P[i]  exactly.  P_out / T_out may be NULL. */
int ising_accept_table(double beta, float P_out[5], uint32_t T_out[5]);

/* ---- host-buffer entry points (end-to-end path) -------------------------------
 * Same results as the calls above, but the caller's buffers are HOST memory:
 * the library stages through device memory it owns (grown on demand, freed by
 * rng_destroy), runs the kernel, copies the result to the host on the same stream
 * and returns when the host buffer is complete (the copy over PCIe dominates: the
 * 4 GiB of config 2 are generated in 0.7 ms and copied in 75 ms). */
int rng_fill_u32_host(rng_handle *h, uint32_t *h_out, uint64_t n, void *cuda_stream);
int rng_fill_f32_host(rng_handle *h, float *h_out, uint64_t n, void *cuda_stream);
int rng_draw_reduce_host(rng_handle *h, uint32_t *h_out, uint64_t n, void *cuda_stream);
/* h_spins is copied to the device, swept, and copied back; h_energy_trace may be NULL */
int ising_sweep_host(rng_handle *h, int8_t *h_spins, uint32_t L, double beta, uint32_t n_sweeps,
                     int64_t *h_energy_trace, void *cuda_stream);

/* ---- state access (checkpoint / resume; the state is stored to
 * global memory after every kernel and reloaded by the next) --------------------
 * Canonical order, independent of the device layout:
 *   LCG64 / LEAPFROG: n_local x u64 (current x of each stream)
 *   XORWOW: n_local x {x,y,z,w,v,d} u32, stream-major
 *   PHILOX (both): 0 bytes;  XS1024W and XS1024W_SKIP: n_local x u32 (word s%32 of instance s/32)
 *   LCG32 / LCG32_LEAPFROG: n_local x u32 (current x of each stream)
 *   LCG64_BOTH: n_local x u64 (current x; which half comes next is draws_done & 1)
 *   LFIB521 / LFIB1279: (n_local/256) x r floats, an instance's last r numbers, oldest first
 *   MWC: n_local x u64 (c << 32 | x);  MWC_MULTI: n_local x {x, c, a} u32, stream-major
 * rng_get_state/rng_set_state synchronise the device; bytes must equal
 * rng_state_bytes(kind, n_local).  draws_done is read / set separately. */
uint64_t rng_state_bytes(int kind, uint64_t n_streams);
int rng_get_state(rng_handle *h, void *h_buf, uint64_t bytes);
int rng_set_state(rng_handle *h, const void *h_buf, uint64_t bytes);
uint64_t rng_draws_done(const rng_handle *h);
/* Sets the per-stream draw counter WITHOUT touching the device state.  For the counter-based kinds
 * (PHILOX) the counter IS the position: any value repositions the streams.  For every stateful kind
 * the counter must describe the device state or the two fall apart silently -- the Weyl index of
 * XS1024W (term n of PAPER.md:236 is derived from draws_done), the half of the state LCG64_BOTH hands
 * out next (draws_done & 1), and every "draws_done" a later checkpoint records.  So for those kinds
 * call it only together with rng_set_state, with the draws_done that was read when that state was
 * saved (checkpoint / resume); the library cannot check this and does not try. */
int rng_set_draws_done(rng_handle *h, uint64_t draws_done);

/* ---- TEST AND MEASUREMENT INTERFACE: not part of the product boundary --------
 * Selects which of several bit-identical kernel variants a handle launches, so that tests can compare
 * them with one another and bench runs can time them: name in {"xs1024", "xsfill", "ising", "store",
 * "lcg", "cvt"}, value = variant index (0 = default, what every other caller gets and what bench.py
 * times).  No result of any other entry point depends on it; applications have no reason to call it
 * and it may change between versions.  See DESIGN.md section 6.  Unknown name/value: RNG_E_INVAL. */
int rng_set_variant(rng_handle *h, const char *name, int value);

/* number of kernels launched by this library in the calling process so far */
uint64_t rng_kernel_launches(void);
const char *rng_last_error(void);
/* "rng_b200 <version> sm_100a" */
const char *rng_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RNG_B200_H */
