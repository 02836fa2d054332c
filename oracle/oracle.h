/*
 * oracle.h -- CPU ORACLE for arxiv 1204.6193 (Manssen, Weigel, Hartmann).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow,
 * obviously-correct restatement of what the hot path computes, written from
 * /root/reference/PAPER.md (cited as PAPER.md:<line>) and, where the paper is
 * silent, from the readings listed in DESIGN.md section 3 (cited as R-<id>).
 * It shares no code, header, table or constant generator with the CUDA path
 * under paper_1204_6193_b200/csrc/.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.
 * One place where oracle and kernel necessarily follow the same ALGORITHM is the
 * primality test of the per-stream MWC multipliers (a kind outside SURVEY.md
 * section 8): the paper prescribes Miller-Rabin and both sides use
 * it, each in its own code.  Its pin therefore uses neither: tests/test_oracle_mwc.py
 * accepts a prime only with a Pratt / Pocklington certificate and a composite only
 * with a witness, and the scan below is the plain sequential one of the paper.
 *
 * Everything is integer arithmetic mod 2^32 / 2^64, so "precision" is exact;
 * the only floating point is the Ising acceptance table (double exp, rounded
 * to float) and the fixed u32 -> f32 map (u >> 8) * 2^-24, which is exact.
 *
 * Pin status (tests/test_oracle_*.py, all "-m 'not gpu'"): every function
 * below is pinned to something other than itself -- see DESIGN.md section 4.
 * Nothing here is "parity unpinned".
 */
#ifndef ORACLE_1204_6193_H
#define ORACLE_1204_6193_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* generator kinds (numbering chosen to match the paper's order of sections) */
enum {
    ORC_LCG64          = 0, /* PAPER.md:33 eq.(1), :46 constants, random seeds  */
    ORC_LCG64_LEAPFROG = 1, /* PAPER.md:39-46 eq.(2),(3): one global sequence   */
    ORC_XORWOW         = 2, /* PAPER.md:169, :236 (recurrence: Ref.[30], R-B1)  */
    ORC_PHILOX4X32_10  = 3, /* PAPER.md:284-296 (constants: Ref.[20], R-C1)     */
    ORC_XS1024W        = 4, /* PAPER.md:166 eq.(8), :177, :201-225, :232-240    */
    ORC_PHILOX4X32_7   = 5, /* the 7-round variant          */
    ORC_LCG32          = 6, /* PAPER.md:33 eq.(1), :46: a=1664525, c=1013904223,
                               m=2^32; draw j = x_j (all 32 bits), x_0 = lo32(SM_seed[s]) */
    ORC_XS1024W_SKIP   = 7, /* kind 4 seeded as PAPER.md:228 does: all instances from one
                               state, instance g skipped ahead by g * 2^137 updates     */
    ORC_LCG64_BOTH     = 8, /* LCG64 "using the whole state to produce two
                               32-bit numbers": draw 2i = hi32(x_i), draw 2i+1 = lo32(x_i) */
    ORC_LFIB521        = 9, /* PAPER.md:105-124 eq.(5): u_n = u_{n-r} + u_{n-s} mod 1 in float,   */
    ORC_LFIB1279       = 10, /* (r,s) = (521,353) / (1279,861); ring shared by 256 streams       */
    ORC_LCG32_LEAPFROG = 11, /* kind 1's sub-stream method for the 32-bit LCG (Table 1 row "LCG32") */
    ORC_MWC            = 12, /* multiply-with-carry, m = 2^32, a = 4294967118 for all streams */
    ORC_MWC_MULTI      = 13  /* one safe-prime multiplier per stream, working down from 4294967118 */
};

/* ---- elementary pieces, exported so that the tests can pin them ---------- */

/* k-th (0-based) output of splitmix64 started at state `seed` (R-S1). */
uint64_t orc_splitmix64(uint64_t seed, uint64_t k);

/* one step of eq.(1) with m = 2^64 */
uint64_t orc_lcg64_step(uint64_t x);
uint32_t orc_lcg32_step(uint32_t x);

/* eq.(2): the affine map x -> A x + C equal to n steps of eq.(1), evaluated by
 * the CLOSED FORM  A = a^n,  C = c (a^n - 1)/(a - 1)  (mod 2^64)  in 128-bit
 * integers (R-A1, R-A2) -- not by composing maps. */
void orc_lcg64_jump(uint64_t n, uint64_t *A, uint64_t *C);

/* Philox4x32 with R rounds: ctr[4], key[2] -> out[4] */
void orc_philox4x32(int R, const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* one XORWOW draw on st = {x,y,z,w,v,d}: advance, then return d+v (R-B1) */
uint32_t orc_xorwow_next(uint32_t st[6]);

/* one update X <- X M of the 1024-bit XORShift, eq.(8) with (a,b,c) =
 * (329,347,344); X[0] is the MOST significant word (R-D1). */
void orc_xs1024_update(uint32_t X[32]);

/* skip-ahead: M as a bit matrix (row r = image of the unit vector
 * "word r/32, bit r%32" under one update), X A, A B, and M^(2^k) by k squarings.
 * Matrices are [1024][32] uint32, row-major. */
void orc_xs1024_matrix(uint32_t *M);
void orc_xs1024_vecmat(const uint32_t X[32], const uint32_t *A, uint32_t out[32]);
void orc_xs1024_matmul(const uint32_t *A, const uint32_t *B, uint32_t *out);
void orc_xs1024_matpow2(unsigned k, uint32_t *out);

/* is a 2^32 - 1 a safe prime; multipliers number first .. first+count-1 counted down from 2^32 - 1 */
int orc_is_prime64(uint64_t n);
int orc_mwc_is_multiplier(uint32_t a);
int orc_mwc_multipliers(uint64_t first, uint64_t count, uint32_t *out);
/* one multiply-with-carry step on st = {x, c} */
void orc_mwc_step(uint32_t st[2]);

/* eq.(5): one float addition mod 1 */
float orc_lfib_add(float a, float b);

/* fixed output map u32 -> [0,1) float:  (u >> 8) * 2^-24   (BASELINE.json) */
float orc_u32_to_f32(uint32_t u);

/* ---- the stream object: same call sequence as the C-ABI under test ------- */

typedef struct orc_rng orc_rng;

/* Streams [first, first + n_local) out of n_total.  n_total matters for the
 * LEAPFROG kind (stride of the global sequence) and nothing else.
 * Returns NULL on invalid arguments. */
orc_rng *orc_create(int kind, uint64_t n_total, uint64_t first, uint64_t n_local, uint64_t seed);
void     orc_destroy(orc_rng *);
uint64_t orc_draws_done(const orc_rng *);
/* Philox kinds only (the counter IS the position); others: returns -1 */
int      orc_set_draws_done(orc_rng *, uint64_t draws_done);

/* out[s*n + j] = draw (draws_done + j) of local stream s; then draws_done += n */
void orc_fill_u32(orc_rng *, uint32_t *out, uint64_t n);
void orc_fill_f32(orc_rng *, float *out, uint64_t n);
/* out[2s] = XOR_j u_{s,j};  out[2s+1] = SUM_j u_{s,j} mod 2^32 */
void orc_draw_reduce(orc_rng *, uint32_t *out, uint64_t n);

/* raw state words in the documented canonical order (per kind):
 *   LCG64 / LEAPFROG: n_local x u64 (x of each stream, LEAPFROG: X_{s + t*S})
 *   XORWOW: n_local x 6 x u32 {x,y,z,w,v,d}, stream-major
 *   PHILOX: nothing (0 words)
 *   XS1024W: n_local x u32 (word `lane` of instance s/32 at index s)
 *   LFIB: per instance (256 streams) the last r numbers, oldest first, as float bits
 *   MWC: n_local x {x, c} u32;  MWC_MULTI: n_local x {x, c, a} u32 */
uint64_t orc_state_words32(const orc_rng *);
void     orc_get_state(const orc_rng *, uint32_t *out);

/* ---- Ising consumer (BASELINE.json config 5; R-E*) ------ */

/* P[i] = (float) exp(-2 beta (2 i - 4)), i = 0..4  (i = number of ALIGNED
 * neighbours = (h+4)/2 with h = s * sum of the four neighbours) */
void orc_ising_accept_table(double beta, float P[5]);
/* spin i = +1 if bit (i & 63) of splitmix64(seed, i >> 6) is set, else -1 */
void orc_ising_init_random(int8_t *spins, uint32_t L, uint64_t seed);
/* E = - sum over bonds s_i s_j, each bond once, periodic */
int64_t orc_ising_energy(const int8_t *spins, uint32_t L);
/* n_sweeps checkerboard Metropolis sweeps, drawing from `rng` (n_local streams
 * must divide L*L/2).  energy_trace may be NULL, else [n_sweeps].
 * returns 0, or -1 on invalid arguments. */
int orc_ising_sweep(orc_rng *, int8_t *spins, uint32_t L, double beta,
                    uint32_t n_sweeps, int64_t *energy_trace);

/* The paper's own consumer (R-E9): double checkerboard of T x T tiles
 * with k_hits multi-hit updates per tile visit; n_local must be L*L/4 (one stream per
 * thread of the paper's kernel); T even, T | L, L/T even.  A sweep updates every site
 * k_hits times and spends 4*k_hits draws per stream.  returns 0, or -1 on bad arguments. */
int orc_ising_sweep_multihit(orc_rng *, int8_t *spins, uint32_t L, double beta, uint32_t n_sweeps,
                             uint32_t T, uint32_t k_hits, int64_t *energy_trace);

/* number of OpenMP threads the loops above will use (1 if built without) */
int orc_threads(void);
void orc_set_threads(int n);

#ifdef __cplusplus
}
#endif
#endif
