/*
 * oracle.c -- CPU ORACLE (test infrastructure only; see oracle.h header).
 *
 * Plain C99, one translation unit, libc + libm only.  Written from PAPER.md
 * step by step in the paper's order and notation; no blocking, fusion or
 * reordering.  The only concession to run time is `#pragma omp parallel for`
 * over independent streams (the streams are independent by construction,
 * PAPER.md:19-21); delete the pragmas and nothing else changes.
 *
 * Citations: PAPER.md:<line>; R-<id> = reading listed in DESIGN.md section 3.
 */
#include "oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------ */
/* splitmix64 -- stands in for "seed each instance with another RNG"         */
/* (PAPER.md:46, :124, :230).  Not in the paper; named by BASELINE.json.     */
/* R-S1: state advances by the golden-ratio increment, output is the mixed   */
/* state; k-th output (0-based) from start state `seed` is random access.    */
/* ------------------------------------------------------------------------ */
uint64_t orc_splitmix64(uint64_t seed, uint64_t k)
{
    uint64_t z = seed + (k + 1u) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

/* ------------------------------------------------------------------------ */
/* A. LCG64   x_{n+1} = a x_n + c (mod 2^64)            PAPER.md:33 eq.(1)   */
/*    a = 2862933555777941757, c = 1442695040888963407         */
/*    output = the 32 most significant bits         */
/*    R-A3: draw j of a stream is hi32(x_j), j from 0 (output, then advance) */
/* ------------------------------------------------------------------------ */
#define LCG_A 2862933555777941757ull
#define LCG_C 1442695040888963407ull

uint64_t orc_lcg64_step(uint64_t x) { return LCG_A * x + LCG_C; }

/* eq.(2),(3).  Eq.(3) as printed (sum from i=1 to t of a^i c)
 * contradicts eq.(1) at t=1; R-A1 reads it as c * sum_{i=0}^{t-1} a^i
 * = c (a^t - 1)/(a - 1).  (a - 1) = 4 q with q odd is not invertible mod 2^64
 * (R-A2), so: a^t is taken mod 2^128 (only its low 66 bits are used), the
 * division by 4 is exact, and the division by the odd q is a multiplication
 * by q^{-1} mod 2^64. */
void orc_lcg64_jump(uint64_t n, uint64_t *A, uint64_t *C)
{
    unsigned __int128 p = 1, b = LCG_A; /* p = a^n mod 2^128 */
    uint64_t e = n;
    while (e) {
        if (e & 1) p *= b;
        b *= b;
        e >>= 1;
    }
    unsigned __int128 mask66 = (((unsigned __int128)1) << 66) - 1;
    unsigned __int128 num = (p - 1) & mask66;      /* a^n - 1 mod 2^66, divisible by 4 */
    uint64_t g4 = (uint64_t)(num >> 2);            /* (a^n - 1)/4 mod 2^64 */
    uint64_t q = (LCG_A - 1) / 4;                  /* odd */
    uint64_t qi = q;                               /* Newton: qi <- qi (2 - q qi) */
    for (int i = 0; i < 6; i++) qi *= 2 - q * qi;
    *A = (uint64_t)p;
    *C = LCG_C * (g4 * qi);
}

/* ------------------------------------------------------------------------ */
/* C. Philox4x32_R        */
/*   S-box on a pair (L,R) with multiplier M and key word k:  */
/*       L' = mullo(R, M)          R' = mulhi(R, M) xor k xor L              */
/*   N = 4 words: two S-boxes per round with different multipliers, words    */
/*   permuted between rounds.  R-C1: multipliers, pairing,    */
/*   permutation and key schedule are those of Ref.[20]:                     */
/*   S-box A on (L,R) = (c1,c2) with M1 and key word k0, S-box B on (L,R) =  */
/*   (c3,c0) with M0 and key word k1; after the S-boxes the block is         */
/*   (R'_A, L'_A, R'_B, L'_B); key += (W0,W1) after each round.              */
/* ------------------------------------------------------------------------ */
static uint32_t mulhi32(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a * b) >> 32); }
static uint32_t mullo32(uint32_t a, uint32_t b) { return (uint32_t)((uint64_t)a * b); }

void orc_philox4x32(int R, const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < R; r++) {
        /* S-box A on (L,R) = (c1,c2), multiplier M1, key word k0 */
        uint32_t LA = mullo32(c2, M1);
        uint32_t RA = mulhi32(c2, M1) ^ k0 ^ c1;
        /* S-box B on (L,R) = (c3,c0), multiplier M0, key word k1 */
        uint32_t LB = mullo32(c0, M0);
        uint32_t RB = mulhi32(c0, M0) ^ k1 ^ c3;
        /* P-box between rounds */
        c0 = RA; c1 = LA; c2 = RB; c3 = LB;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------------ */
/* B. XORWOW (Marsaglia, Ref.[30]; "w = 160 xorshift +   */
/*   32-bit Weyl, c = 362437", 192 bits of state).  R-B1: recurrence is      */
/*   Ref.[30]'s xorwow with shifts (2,1,4); advance, then output d + v.      */
/* ------------------------------------------------------------------------ */
uint32_t orc_xorwow_next(uint32_t st[6])
{
    uint32_t x = st[0], y = st[1], z = st[2], w = st[3], v = st[4], d = st[5];
    uint32_t t = x ^ (x >> 2);
    x = y; y = z; z = w; w = v;
    v = (v ^ (v << 4)) ^ (t ^ (t << 1));
    d = d + 362437u;
    st[0] = x; st[1] = y; st[2] = z; st[3] = w; st[4] = v; st[5] = d;
    return d + v;
}

/* ------------------------------------------------------------------------ */
/* D. XORShift1024 + Weyl, the paper's generator.                            */
/*   eq.(8):  X <- X (I + L^a)(I + R^b)(I + L^c), w = 1024,     */
/*   (a,b,c) = (329,347,344) PAPER.md:177; "x ^ (x << a)" PAPER.md:164.      */
/*   Bits shifted past either end are lost, zeros enter (zero padding,       */
/*   PAPER.md:175-177).  R-D1: word held by thread/lane i is X[i], lane 0 =  */
/*   most significant word (this is what makes Listing 1,  */
/*   and eq.(8) the same map).  Written here as whole-number shifts on a     */
/*   32-word array, for any shift amount -- not in Listing 1's per-lane form.*/
/* ------------------------------------------------------------------------ */
static void shl1024(const uint32_t X[32], unsigned a, uint32_t out[32])
{
    unsigned ws = a / 32, bs = a % 32;
    for (unsigned i = 0; i < 32; i++) {
        uint32_t hi = (i + ws < 32) ? X[i + ws] : 0u;         /* more significant source */
        uint32_t lo = (i + ws + 1 < 32) ? X[i + ws + 1] : 0u; /* less significant source */
        out[i] = bs ? ((hi << bs) | (lo >> (32 - bs))) : hi;
    }
}
static void shr1024(const uint32_t X[32], unsigned b, uint32_t out[32])
{
    unsigned ws = b / 32, bs = b % 32;
    for (unsigned i = 0; i < 32; i++) {
        uint32_t lo = (i >= ws) ? X[i - ws] : 0u;
        uint32_t hi = (i >= ws + 1) ? X[i - ws - 1] : 0u;
        out[i] = bs ? ((lo >> bs) | (hi << (32 - bs))) : lo;
    }
}
void orc_xs1024_update(uint32_t X[32])
{
    uint32_t T[32];
    shl1024(X, 329, T); for (int i = 0; i < 32; i++) X[i] ^= T[i];
    shr1024(X, 347, T); for (int i = 0; i < 32; i++) X[i] ^= T[i];
    shl1024(X, 344, T); for (int i = 0; i < 32; i++) X[i] ^= T[i];
}
/* ---- skip-ahead of the XORShift1024 ---------------------------
 * The update is X <- X M over GF(2) (eq.(8)).  The paper seeds the
 * instances by "multiplying the state with the precomputed 2^137-th power of the
 * recursion matrix M".  Written out: M as 1024 rows of 1024 bits, row r = image
 * of the unit vector e_r (word r/32, bit r%32 of that word) under ONE update;
 * a vector-matrix product X A = XOR of the rows A[r] over the set bits r of X;
 * a matrix product (A B)[r] = A[r] B; powers by repeated squaring. */
void orc_xs1024_matrix(uint32_t *M /* [1024][32] */)
{
    for (int r = 0; r < 1024; r++) {
        uint32_t *row = M + 32 * r;
        memset(row, 0, 32 * sizeof(uint32_t));
        row[r / 32] = 1u << (r % 32);
        orc_xs1024_update(row);
    }
}
void orc_xs1024_vecmat(const uint32_t X[32], const uint32_t *A, uint32_t out[32])
{
    uint32_t acc[32] = {0};
    for (int r = 0; r < 1024; r++)
        if ((X[r / 32] >> (r % 32)) & 1u)
            for (int i = 0; i < 32; i++) acc[i] ^= A[32 * r + i];
    memcpy(out, acc, sizeof acc);
}
void orc_xs1024_matmul(const uint32_t *A, const uint32_t *B, uint32_t *out /* may not alias */)
{
#pragma omp parallel for schedule(static)
    for (int r = 0; r < 1024; r++) orc_xs1024_vecmat(A + 32 * r, B, out + 32 * r);
}
/* out = M^(2^k) by k squarings */
void orc_xs1024_matpow2(unsigned k, uint32_t *out /* [1024][32] */)
{
    uint32_t *T = (uint32_t *)malloc(1024 * 32 * sizeof(uint32_t));
    orc_xs1024_matrix(out);
    for (unsigned i = 0; i < k; i++) {
        orc_xs1024_matmul(out, out, T);
        memcpy(out, T, 1024 * 32 * sizeof(uint32_t));
    }
    free(T);
}

/* Weyl part, eq.(9): y_n = y_0 + n c mod 2^32, c = 362437;
 * R-D6: y_0 = 0 for every instance (footnote 4), n = number of
 * updates since creation.  Output (gamma = w/2 = 16):
 *     out_i = (y_n (I + R^16)) + x_i  =  (y_n ^ (y_n >> 16)) + x_i  mod 2^32 */
static uint32_t xs1024_weyl_term(uint64_t n_updates)
{
    uint32_t y = (uint32_t)n_updates * 362437u;
    return y ^ (y >> 16);
}

/* ------------------------------------------------------------------------ */
float orc_u32_to_f32(uint32_t u) { return (float)(u >> 8) * 0x1p-24f; }

/* ------------------------------------------------------------------------ */
/* stream object                                                             */
/* ------------------------------------------------------------------------ */
struct orc_rng {
    int kind;
    uint64_t n_total, first, n_local, seed;
    uint64_t draws_done;  /* per stream, all streams in lockstep */
    uint64_t *lcg;        /* LCG64: x of each local stream */
    uint64_t leap_X;      /* LEAPFROG: X_{draws_done * n_total} of the global sequence */
    uint32_t leap_X32;    /* LCG32_LEAPFROG: the same for the 32-bit LCG */
    uint32_t *mwc;        /* MWC: [n_local][2] = {x, c};  MWC_MULTI: [n_local][3] = {x, c, a} */
    uint32_t *xw;         /* XORWOW: [n_local][6] */
    uint32_t *xs;         /* XS1024W: [n_local/32][32], word i of instance g at 32 g + i */
    uint32_t *lcg32;      /* LCG32: x of each local stream */
    float *lf;            /* LFIB: [n_local/256][r], the last r numbers of each instance, oldest first */
};

/* ---- lagged Fibonacci, PAPER.md:105-124 ---------------------------------------------
 * eq.(5):  u_n = u_{n-r} + u_{n-s} (mod 1)  "by using floating-point arithmetic",
 * with (r,s) = (521,353) and (1279,861).  Single precision:  t = a + b; if
 * (t >= 1) t -= 1.  R-G1: the seeds are 23-bit fractions, so that every sum is exact in
 * float (a sum in [1,2) has spacing 2^-23) and the float recurrence IS addition mod 1.
 * The ring buffer is shared by the threads of a block, which produce s numbers at a
 * time: R-G2: an INSTANCE serves T = 256 streams (threads), T <= s; the
 * instance's numbers v_0, v_1, ... (v_m = u_{r+m}) are dealt round-robin: stream t of
 * the instance gets v_{jT+t} as its draw j.  R-G3: u_i of instance g, i < r, is
 * (w >> 9) 2^-23 with w the 32-bit word number g r + i of the splitmix64 word sequence
 * (word 2k = lo32, 2k+1 = hi32 of SM_seed[k]); if no u_i of an instance is an odd
 * multiple of 2^-23 its u_0 gets that bit (an all-even seed would halve the period [19]).
 * As 32-bit integers the draws are (v 2^23) << 9, so that the fixed map gives v back. */
#define ORC_LFIB_T 256
static int lfib_lags(int kind, int *r, int *s)
{
    if (kind == ORC_LFIB521) { *r = 521; *s = 353; return 1; }
    if (kind == ORC_LFIB1279) { *r = 1279; *s = 861; return 1; }
    return 0;
}
float orc_lfib_add(float a, float b)
{
    volatile float t = a + b; /* one IEEE single-precision addition, no wider intermediate */
    if (t >= 1.0f) t = t - 1.0f;
    return t;
}
static uint32_t splitmix_word32(uint64_t seed, uint64_t w)
{
    uint64_t z = orc_splitmix64(seed, w / 2);
    return (w & 1) ? (uint32_t)(z >> 32) : (uint32_t)z;
}

/* Multiply-with-carry:  x_{n+1} = a x_n + c_n mod m,  c_{n+1} = floor((a x_n + c_n)/m),
 * m = 2^32, a = 4294967118 ("a standard choice for a single generator instance"; Table 1 row
 * "MWC, same a": every stream uses this multiplier, only the seeds differ). */
#define ORC_MWC_A 4294967118ull
static void mwc_step_a(uint32_t st[2], uint32_t a)
{
    uint64_t t = (uint64_t)a * (uint64_t)st[0] + (uint64_t)st[1];
    st[0] = (uint32_t)t;
    st[1] = (uint32_t)(t >> 32);
}
void orc_mwc_step(uint32_t st[2])
{
    uint64_t t = ORC_MWC_A * (uint64_t)st[0] + (uint64_t)st[1];
    st[0] = (uint32_t)t;         /* x_{n+1} */
    st[1] = (uint32_t)(t >> 32); /* c_{n+1} */
}

/* ---- per-stream MWC multipliers, PAPER.md:97 -----------------------------------------
 * "it is possible to systematically generate multipliers by finding the largest safe prime am-1 with a less
 * than 2^32 (which is just the a = 4294967118 above) and then systematically working one's way down from there
 * towards smaller multipliers.  To check for primality one uses probabilistic tests such as the Rabin-Miller
 * algorithm".  Written out: multiplier number k (k = 0, 1, ...) is the (k+1)-th largest a < 2^32 for which both
 * p = a 2^32 - 1 and (p - 1)/2 are prime.  Primality: trial division by the primes below 60, then Miller-Rabin
 * with the twelve bases 2..37, which is a PROOF for numbers below 3.3e24 (all candidates are below 2^64). */
static uint64_t mulmod64(uint64_t a, uint64_t b, uint64_t n) { return (uint64_t)((unsigned __int128)a * b % n); }
static uint64_t powmod64(uint64_t a, uint64_t e, uint64_t n)
{
    uint64_t r = 1;
    a %= n;
    while (e) {
        if (e & 1) r = mulmod64(r, a, n);
        a = mulmod64(a, a, n);
        e >>= 1;
    }
    return r;
}
int orc_is_prime64(uint64_t n)
{
    static const uint64_t small[] = {2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37, 41, 43, 47, 53, 59};
    static const uint64_t bases[] = {2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37};
    if (n < 2) return 0;
    for (unsigned i = 0; i < sizeof small / sizeof *small; i++)
        if (n % small[i] == 0) return n == small[i];
    uint64_t d = n - 1;
    int r = 0;
    while ((d & 1) == 0) { d >>= 1; r++; }
    for (unsigned i = 0; i < sizeof bases / sizeof *bases; i++) {
        uint64_t x = powmod64(bases[i], d, n);
        if (x == 1 || x == n - 1) continue;
        int composite = 1;
        for (int k = 1; k < r; k++) {
            x = mulmod64(x, x, n);
            if (x == n - 1) { composite = 0; break; }
        }
        if (composite) return 0;
    }
    return 1;
}
int orc_mwc_is_multiplier(uint32_t a)
{
    uint64_t p = ((uint64_t)a << 32) - 1; /* a m - 1 */
    return a > 0 && orc_is_prime64((p - 1) / 2) && orc_is_prime64(p);
}
/* out[i] = multiplier number first + i, scanning down from 2^32 - 1.  returns 0, or -1 if the candidates run out.
 * PAPER.md:97 as it reads: start at the top and work down one candidate at a time, counting those that qualify
 * (plain sequential order, no chunking: slow -- about 1300 candidates per multiplier -- and meant to be).
 * The list found so far is remembered for the life of the process, so that a later call continues the same scan
 * where the last one stopped instead of starting again at the top (a memo of results; the order of work is the same). */
static uint32_t *mwc_found;           /* multipliers number 0 .. mwc_n_found-1 */
static uint64_t mwc_n_found, mwc_cap;
static uint64_t mwc_next = 0xffffffffull; /* the next candidate a to look at */
int orc_mwc_multipliers(uint64_t first, uint64_t count, uint32_t *out)
{
    const uint64_t need = first + count;
    if (need > mwc_cap) {
        uint64_t cap = mwc_cap ? mwc_cap : 1024;
        while (cap < need) cap *= 2;
        uint32_t *p = (uint32_t *)realloc(mwc_found, cap * sizeof *p);
        if (!p) return -1;
        mwc_found = p;
        mwc_cap = cap;
    }
    for (; mwc_n_found < need && mwc_next >= 1; mwc_next--)
        if (orc_mwc_is_multiplier((uint32_t)mwc_next)) mwc_found[mwc_n_found++] = (uint32_t)mwc_next;
    if (mwc_n_found < need) return -1;
    memcpy(out, mwc_found + first, count * sizeof *out);
    return 0;
}

/* G1: 32-bit LCG, eq.(1) with the constants of PAPER.md:46 */
uint32_t orc_lcg32_step(uint32_t x) { return 1664525u * x + 1013904223u; }

orc_rng *orc_create(int kind, uint64_t n_total, uint64_t first, uint64_t n_local, uint64_t seed)
{
    if (n_local < 1 || first + n_local > n_total || first + n_local < first) return NULL;
    if (kind < ORC_LCG64 || kind > ORC_MWC_MULTI) return NULL;
    if ((kind == ORC_LFIB521 || kind == ORC_LFIB1279) && (first % ORC_LFIB_T || n_local % ORC_LFIB_T)) return NULL;
    if ((kind == ORC_XS1024W || kind == ORC_XS1024W_SKIP) && (first % 32 || n_local % 32)) return NULL;
    orc_rng *r = (orc_rng *)calloc(1, sizeof *r);
    if (!r) return NULL;
    r->kind = kind; r->n_total = n_total; r->first = first; r->n_local = n_local; r->seed = seed;
    switch (kind) {
    case ORC_LCG64_BOTH: /* same generator and seeds; only the output rule differs */
    case ORC_LCG64: /* random seeding: x_0^(s) = SM_seed[s] */
        r->lcg = (uint64_t *)malloc(n_local * sizeof(uint64_t));
        for (uint64_t s = 0; s < n_local; s++) r->lcg[s] = orc_splitmix64(seed, first + s);
        break;
    case ORC_LCG64_LEAPFROG: /* sub-streams of ONE sequence: X_0 = SM_seed[0] */
        r->leap_X = orc_splitmix64(seed, 0);
        break;
    case ORC_MWC: /* R-M1: (x_0, c_0) = (lo32, hi32 mod a) of SM_seed[s]; the two fixed points (0,0) and
                   * (m-1, a-1) of the map are moved to (1,0) and (m-1, a-2) */
        r->mwc = (uint32_t *)malloc(n_local * 2 * sizeof(uint32_t));
        for (uint64_t s = 0; s < n_local; s++) {
            uint64_t z = orc_splitmix64(seed, first + s);
            uint32_t x = (uint32_t)z, cc = (uint32_t)((z >> 32) % ORC_MWC_A);
            if (x == 0 && cc == 0) x = 1;
            if (x == 0xffffffffu && cc == (uint32_t)(ORC_MWC_A - 1)) cc = (uint32_t)(ORC_MWC_A - 2);
            r->mwc[2 * s] = x;
            r->mwc[2 * s + 1] = cc;
        }
        break;
    case ORC_MWC_MULTI: { /* Table 1 row "MWC, different a": stream s (global id) uses multiplier number s; seeds as
                           * ORC_MWC with its own a: (lo32, hi32 mod a_s), fixed points (0,0), (m-1, a_s-1) moved */
        uint32_t *mult = (uint32_t *)malloc(n_local * sizeof(uint32_t));
        if (orc_mwc_multipliers(first, n_local, mult) != 0) { free(mult); free(r); return NULL; }
        r->mwc = (uint32_t *)malloc(n_local * 3 * sizeof(uint32_t));
        for (uint64_t s = 0; s < n_local; s++) {
            uint64_t z = orc_splitmix64(seed, first + s);
            uint32_t a = mult[s], x = (uint32_t)z, cc = (uint32_t)(z >> 32) % a;
            if (x == 0 && cc == 0) x = 1;
            if (x == 0xffffffffu && cc == a - 1) cc = a - 2;
            r->mwc[3 * s] = x;
            r->mwc[3 * s + 1] = cc;
            r->mwc[3 * s + 2] = a;
        }
        free(mult);
        break;
    }
    case ORC_LCG32_LEAPFROG: /* the same for the 32-bit LCG (Table 1 row "LCG32"): X_0 = lo32(SM_seed[0]) */
        r->leap_X32 = (uint32_t)orc_splitmix64(seed, 0);
        break;
    case ORC_XORWOW: /* R-B2: (x,y),(z,w),(v,d) = (lo,hi) of SM_seed[3s], [3s+1], [3s+2] */
        r->xw = (uint32_t *)malloc(n_local * 6 * sizeof(uint32_t));
        for (uint64_t s = 0; s < n_local; s++) {
            uint32_t *st = r->xw + 6 * s;
            for (int p = 0; p < 3; p++) {
                uint64_t z = orc_splitmix64(seed, 3 * (first + s) + p);
                st[2 * p] = (uint32_t)z;
                st[2 * p + 1] = (uint32_t)(z >> 32);
            }
            if ((st[0] | st[1] | st[2] | st[3] | st[4]) == 0) st[4] = 1; /* R-B3 fixed point */
        }
        break;
    case ORC_PHILOX4X32_10: /* no state: key and counter are intrinsic */
    case ORC_PHILOX4X32_7:
        break;
    case ORC_LCG32: /* random seeding */
        r->lcg32 = (uint32_t *)malloc(n_local * sizeof(uint32_t));
        for (uint64_t s = 0; s < n_local; s++) r->lcg32[s] = (uint32_t)orc_splitmix64(seed, first + s);
        break;
    case ORC_XS1024W: /* "sloppy" random seeding; R-D7 */
        r->xs = (uint32_t *)malloc(n_local * sizeof(uint32_t));
        for (uint64_t g = 0; g < n_local / 32; g++) {
            uint64_t gg = first / 32 + g; /* global instance number */
            uint32_t *X = r->xs + 32 * g, any = 0;
            for (int k = 0; k < 16; k++) {
                uint64_t z = orc_splitmix64(seed, 16 * gg + k);
                X[2 * k] = (uint32_t)z;
                X[2 * k + 1] = (uint32_t)(z >> 32);
                any |= X[2 * k] | X[2 * k + 1];
            }
            if (!any) X[31] = 1;
        }
        break;
    case ORC_LFIB521:
    case ORC_LFIB1279: { /* random seeding of the ring buffers, PAPER.md:122 ("it appears safe to just seed") */
        int lr, ls;
        lfib_lags(kind, &lr, &ls);
        r->lf = (float *)malloc(n_local / ORC_LFIB_T * (uint64_t)lr * sizeof(float));
        for (uint64_t g = 0; g < n_local / ORC_LFIB_T; g++) {
            uint64_t gg = first / ORC_LFIB_T + g;
            float *h = r->lf + g * (uint64_t)lr;
            int odd = 0;
            for (int i = 0; i < lr; i++) {
                uint32_t k = splitmix_word32(seed, gg * (uint64_t)lr + (uint64_t)i) >> 9;
                odd |= (int)(k & 1u);
                h[i] = (float)k * 0x1p-23f;
            }
            if (!odd) h[0] += 0x1p-23f; /* k even, so k+1 < 2^23: still a 23-bit fraction */
        }
        break;
    }
    case ORC_XS1024W_SKIP: {
        /* every instance starts from the SAME state and skips g * 2^137 updates,
         * g = global instance number, by multiplying with J = M^(2^137) once per instance.
         * R-D7b: the paper does not say which common state; it is instance 0's state under
         * the random seeding above (SM_seed[0..15]). */
        uint32_t *J = (uint32_t *)malloc(1024 * 32 * sizeof(uint32_t));
        uint32_t X[32], any = 0;
        orc_xs1024_matpow2(137, J);
        for (int k = 0; k < 16; k++) {
            uint64_t z = orc_splitmix64(seed, (uint64_t)k);
            X[2 * k] = (uint32_t)z;
            X[2 * k + 1] = (uint32_t)(z >> 32);
            any |= X[2 * k] | X[2 * k + 1];
        }
        if (!any) X[31] = 1;
        r->xs = (uint32_t *)malloc(n_local * sizeof(uint32_t));
        for (uint64_t gg = 0; gg < (first + n_local) / 32; gg++) { /* successively, as the paper does */
            if (gg >= first / 32) memcpy(r->xs + 32 * (gg - first / 32), X, sizeof X);
            orc_xs1024_vecmat(X, J, X);
        }
        free(J);
        break;
    }
    }
    return r;
}

void orc_destroy(orc_rng *r)
{
    if (!r) return;
    free(r->lcg); free(r->xw); free(r->xs); free(r->lcg32); free(r->lf); free(r->mwc); free(r);
}

uint64_t orc_draws_done(const orc_rng *r) { return r->draws_done; }

/* Reposition a COUNTER-BASED stream: Philox has no state but (key, counter) and the
 * counter is the draw index (R-C2), so any position is reachable at once.
 * Stateful kinds cannot be repositioned this way: -1. */
int orc_set_draws_done(orc_rng *r, uint64_t draws_done)
{
    if (r->kind != ORC_PHILOX4X32_10 && r->kind != ORC_PHILOX4X32_7) return -1;
    r->draws_done = draws_done;
    return 0;
}

/* Philox stream mapping (BASELINE.json config 2, R-C2): key = stream id XOR
 * seed (64 bit, k0 = low word); counter = index of the 4-word block,
 * (lo32(b), hi32(b), 0, 0); draw j is word (j mod 4) of block floor(j/4). */
static uint32_t philox_draw(int rounds, uint64_t stream_id, uint64_t seed, uint64_t j)
{
    uint64_t K = stream_id ^ seed, b = j / 4;
    uint32_t key[2] = {(uint32_t)K, (uint32_t)(K >> 32)};
    uint32_t ctr[4] = {(uint32_t)b, (uint32_t)(b >> 32), 0u, 0u};
    uint32_t o[4];
    orc_philox4x32(rounds, ctr, key, o);
    return o[j % 4];
}

void orc_fill_u32(orc_rng *r, uint32_t *out, uint64_t n)
{
    const uint64_t S = r->n_local;
    switch (r->kind) {
    case ORC_LCG64:
#pragma omp parallel for schedule(static)
        for (uint64_t s = 0; s < S; s++) {
            uint64_t x = r->lcg[s];
            for (uint64_t j = 0; j < n; j++) {
                out[s * n + j] = (uint32_t)(x >> 32); /* 32 most significant bits */
                x = orc_lcg64_step(x);
            }
            r->lcg[s] = x;
        }
        break;
    case ORC_LCG64_BOTH:
        /* "on using the whole state to produce two 32-bit numbers, the nominal
         * performance would double (but ... the quality ... would be reduced)".  R-F2: a state x_i
         * yields draw 2i = its 32 most significant bits, draw 2i+1 = its 32 least significant bits;
         * the state advances after the second one.  draws_done is common to all streams, so its
         * parity says which half comes next. */
#pragma omp parallel for schedule(static)
        for (uint64_t s = 0; s < S; s++) {
            uint64_t x = r->lcg[s];
            for (uint64_t j = 0; j < n; j++) {
                if (((r->draws_done + j) & 1) == 0) {
                    out[s * n + j] = (uint32_t)(x >> 32);
                } else {
                    out[s * n + j] = (uint32_t)x;
                    x = orc_lcg64_step(x);
                }
            }
            r->lcg[s] = x;
        }
        break;
    case ORC_LCG64_LEAPFROG: {
        /* "all threads generate numbers out of the same global
         * sequence (1)": element m of the global sequence is draw floor(m/S)
         * of stream m mod S, S = number of streams (R-A5).  Walk the global
         * sequence once, in order. */
        uint64_t X = r->leap_X;
        for (uint64_t j = 0; j < n; j++)
            for (uint64_t m = 0; m < r->n_total; m++) {
                if (m >= r->first && m < r->first + S) out[(m - r->first) * n + j] = (uint32_t)(X >> 32);
                X = orc_lcg64_step(X);
            }
        r->leap_X = X;
        break;
    }
    case ORC_MWC:
#pragma omp parallel for schedule(static)
        for (uint64_t s = 0; s < S; s++)
            for (uint64_t j = 0; j < n; j++) {
                out[s * n + j] = r->mwc[2 * s]; /* the draw is x_n (output, then advance: R-A3) */
                orc_mwc_step(r->mwc + 2 * s);
            }
        break;
    case ORC_MWC_MULTI:
#pragma omp parallel for schedule(static)
        for (uint64_t s = 0; s < S; s++)
            for (uint64_t j = 0; j < n; j++) {
                out[s * n + j] = r->mwc[3 * s];
                mwc_step_a(r->mwc + 3 * s, r->mwc[3 * s + 2]);
            }
        break;
    case ORC_LCG32_LEAPFROG: {
        /* as ORC_LCG64_LEAPFROG: walk the ONE global 32-bit sequence in order; the whole word is the draw */
        uint32_t X = r->leap_X32;
        for (uint64_t j = 0; j < n; j++)
            for (uint64_t m = 0; m < r->n_total; m++) {
                if (m >= r->first && m < r->first + S) out[(m - r->first) * n + j] = X;
                X = orc_lcg32_step(X);
            }
        r->leap_X32 = X;
        break;
    }
    case ORC_XORWOW:
#pragma omp parallel for schedule(static)
        for (uint64_t s = 0; s < S; s++)
            for (uint64_t j = 0; j < n; j++) out[s * n + j] = orc_xorwow_next(r->xw + 6 * s);
        break;
    case ORC_PHILOX4X32_10:
    case ORC_PHILOX4X32_7: {
        const int rounds = r->kind == ORC_PHILOX4X32_7 ? 7 : 10;
#pragma omp parallel for schedule(static)
        for (uint64_t s = 0; s < S; s++)
            for (uint64_t j = 0; j < n; j++)
                out[s * n + j] = philox_draw(rounds, r->first + s, r->seed, r->draws_done + j);
        break;
    }
    case ORC_LCG32:
#pragma omp parallel for schedule(static)
        for (uint64_t s = 0; s < S; s++) {
            uint32_t x = r->lcg32[s];
            for (uint64_t j = 0; j < n; j++) {
                out[s * n + j] = x; /* u_n = x_n / m: the whole word is the output */
                x = orc_lcg32_step(x);
            }
            r->lcg32[s] = x;
        }
        break;
    case ORC_LFIB521:
    case ORC_LFIB1279: {
        int lr, ls;
        lfib_lags(r->kind, &lr, &ls);
#pragma omp parallel for schedule(static)
        for (uint64_t g = 0; g < S / ORC_LFIB_T; g++) {
            /* the instance's sequence, one number after the other: hist = u_{n-r} .. u_{n-1} */
            float *hist = r->lf + g * (uint64_t)lr;
            float *u = (float *)malloc(((uint64_t)lr + n * ORC_LFIB_T) * sizeof(float));
            memcpy(u, hist, (size_t)lr * sizeof(float));
            for (uint64_t m = 0; m < n * ORC_LFIB_T; m++) {
                uint64_t i = (uint64_t)lr + m;                 /* u[i] = u[i-r] + u[i-s] mod 1, eq.(5) */
                u[i] = orc_lfib_add(u[i - (uint64_t)lr], u[i - (uint64_t)ls]);
                /* v_m is draw m / T of stream m % T of this instance (R-G2) */
                out[(g * ORC_LFIB_T + m % ORC_LFIB_T) * n + m / ORC_LFIB_T] = (uint32_t)(u[i] * 0x1p23f) << 9;
            }
            memcpy(hist, u + n * ORC_LFIB_T, (size_t)lr * sizeof(float));
            free(u);
        }
        break;
    }
    case ORC_XS1024W:
    case ORC_XS1024W_SKIP:
        /* stream s = word (s mod 32) of instance floor(s/32)  (R-D4) */
#pragma omp parallel for schedule(static)
        for (uint64_t g = 0; g < S / 32; g++) {
            uint32_t *X = r->xs + 32 * g;
            for (uint64_t j = 0; j < n; j++) {
                orc_xs1024_update(X);
                uint32_t wy = xs1024_weyl_term(r->draws_done + j + 1);
                for (uint64_t i = 0; i < 32; i++) out[(32 * g + i) * n + j] = wy + X[i];
            }
        }
        break;
    }
    r->draws_done += n;
}

void orc_fill_f32(orc_rng *r, float *out, uint64_t n)
{
    /* the float stream IS the integer stream pushed through the fixed map */
    uint32_t *u = (uint32_t *)out;
    orc_fill_u32(r, u, n);
    for (uint64_t i = 0; i < r->n_local * n; i++) {
        float f = orc_u32_to_f32(u[i]);
        out[i] = f;
    }
}

void orc_draw_reduce(orc_rng *r, uint32_t *out, uint64_t n)
{
    /* definition: reduce the rows of what fill would have written.  Done in
     * slabs of at most 4096 draws so the scratch array stays small. */
    const uint64_t S = r->n_local, slab = 4096;
    for (uint64_t s = 0; s < S; s++) { out[2 * s] = 0; out[2 * s + 1] = 0; }
    uint32_t *tmp = (uint32_t *)malloc(S * (n < slab ? (n ? n : 1) : slab) * sizeof(uint32_t));
    for (uint64_t done = 0; done < n;) {
        uint64_t m = (n - done < slab) ? n - done : slab;
        orc_fill_u32(r, tmp, m);
        for (uint64_t s = 0; s < S; s++)
            for (uint64_t j = 0; j < m; j++) {
                out[2 * s] ^= tmp[s * m + j];
                out[2 * s + 1] += tmp[s * m + j];
            }
        done += m;
    }
    free(tmp);
}

uint64_t orc_state_words32(const orc_rng *r)
{
    switch (r->kind) {
    case ORC_LCG64: case ORC_LCG64_BOTH: case ORC_LCG64_LEAPFROG: case ORC_MWC: return 2 * r->n_local;
    case ORC_XORWOW: return 6 * r->n_local;
    case ORC_XS1024W: case ORC_XS1024W_SKIP: return r->n_local;
    case ORC_LCG32: case ORC_LCG32_LEAPFROG: return r->n_local;
    case ORC_MWC_MULTI: return 3 * r->n_local;
    case ORC_LFIB521: return r->n_local / ORC_LFIB_T * 521;
    case ORC_LFIB1279: return r->n_local / ORC_LFIB_T * 1279;
    default: return 0;
    }
}

void orc_get_state(const orc_rng *r, uint32_t *out)
{
    switch (r->kind) {
    case ORC_LCG64: case ORC_LCG64_BOTH: memcpy(out, r->lcg, r->n_local * 8); break;
    case ORC_LCG64_LEAPFROG: {
        uint64_t X = r->leap_X; /* X_{t S}; stream s sits at X_{t S + s} */
        for (uint64_t m = 0; m < r->first + r->n_local; m++) {
            if (m >= r->first) memcpy(out + 2 * (m - r->first), &X, 8);
            X = orc_lcg64_step(X);
        }
        break;
    }
    case ORC_LCG32_LEAPFROG: {
        uint32_t X = r->leap_X32;
        for (uint64_t m = 0; m < r->first + r->n_local; m++) {
            if (m >= r->first) out[m - r->first] = X;
            X = orc_lcg32_step(X);
        }
        break;
    }
    case ORC_MWC: memcpy(out, r->mwc, r->n_local * 8); break;
    case ORC_MWC_MULTI: memcpy(out, r->mwc, r->n_local * 12); break;
    case ORC_XORWOW: memcpy(out, r->xw, r->n_local * 24); break;
    case ORC_XS1024W: case ORC_XS1024W_SKIP: memcpy(out, r->xs, r->n_local * 4); break;
    case ORC_LCG32: memcpy(out, r->lcg32, r->n_local * 4); break;
    case ORC_LFIB521: case ORC_LFIB1279: memcpy(out, r->lf, orc_state_words32(r) * 4); break; /* float bit patterns */
    default: break;
    }
}

/* ------------------------------------------------------------------------ */
/* E. Ising consumer.  Zero-field nearest-neighbour ferromagnet on the       */
/*   periodic square lattice, Metropolis, checkerboard.        */
/*   BASELINE.json config 5 fixes: int8 +/-1 spins, plain checkerboard, one  */
/*   uniform per site update, acceptance table exp(-2 beta h).  R-E2: h =    */
/*   s_i * (sum of 4 neighbours), Delta E = 2 h, accept with min(1,e^{-2bh}).*/
/* ------------------------------------------------------------------------ */
void orc_ising_accept_table(double beta, float P[5])
{
    for (int i = 0; i < 5; i++) P[i] = (float)exp(-2.0 * beta * (double)(2 * i - 4));
}

void orc_ising_init_random(int8_t *spins, uint32_t L, uint64_t seed)
{
    uint64_t N = (uint64_t)L * L;
    for (uint64_t i = 0; i < N; i++)
        spins[i] = ((orc_splitmix64(seed, i >> 6) >> (i & 63)) & 1) ? 1 : -1;
}

int64_t orc_ising_energy(const int8_t *sp, uint32_t L)
{
    int64_t E = 0;
    for (uint32_t y = 0; y < L; y++)
        for (uint32_t x = 0; x < L; x++) {
            int s = sp[(uint64_t)y * L + x];
            int right = sp[(uint64_t)y * L + (x + 1) % L];
            int down = sp[(uint64_t)((y + 1) % L) * L + x];
            E -= s * (right + down); /* each bond once */
        }
    return E;
}

int orc_ising_sweep(orc_rng *r, int8_t *sp, uint32_t L, double beta, uint32_t n_sweeps, int64_t *trace)
{
    if (!r || L < 4 || (L & 1)) return -1;
    const uint64_t half = (uint64_t)L * L / 2, S = r->n_local, hw = L / 2;
    if (half % S) return -1;
    const uint64_t K = half / S; /* sites per stream per colour (R-E8) */
    float P[5];
    orc_ising_accept_table(beta, P);
    uint32_t *draws = (uint32_t *)malloc(half * sizeof(uint32_t));
    if (!draws) return -1;
    for (uint32_t t = 0; t < n_sweeps; t++) {
        for (uint32_t c = 0; c < 2; c++) {
            /* "ising_sweep == fill, then apply": stream s owns sites
             * q in [sK,(s+1)K) of this colour, visited in increasing q, and
             * site q consumes the stream's next draw -- which is exactly the
             * stream-major layout draws[s*K + k] = draws[q]. */
            orc_fill_u32(r, draws, K);
            /* all sites of one colour are independent: their neighbours have
             * the other colour and are not touched in this half-sweep */
#pragma omp parallel for schedule(static)
            for (uint64_t q = 0; q < half; q++) {
                uint64_t y = q / hw, xh = q % hw;
                uint64_t x = 2 * xh + ((y + c) & 1);   /* colour of (x,y) = (x+y)&1 */
                int s = sp[y * L + x];
                int nn = sp[y * L + (x + 1) % L] + sp[y * L + (x + L - 1) % L]
                       + sp[((y + 1) % L) * L + x] + sp[((y + L - 1) % L) * L + x];
                int h = s * nn;                         /* in {-4,-2,0,2,4} */
                float u = orc_u32_to_f32(draws[q]);     /* a draw is ALWAYS consumed (R-E3) */
                if (u < P[(h + 4) / 2]) sp[y * L + x] = (int8_t)(-s); /* strict < (R-E3) */
            }
        }
        if (trace) trace[t] = orc_ising_energy(sp, L);
    }
    free(draws);
    return 0;
}

int orc_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---- the paper's own consumer: double checkerboard with multi-hit updates --------
 * PAPER.md:56 ("a double checkerboard decomposition"), :58 ("updating the spins of a
 * tile once (k = 1) ... two random numbers are produced per state load ... multi-hit
 * updates (k = 100), 200 random numbers"); the kernel itself is in Refs.[13,25], so the
 * order below is reading R-E9:
 *   the lattice is cut into T x T tiles (T even, L/T even); tile (tx,ty) has COARSE colour
 *   (tx+ty)&1.  One sweep = coarse colour 0, then coarse colour 1.  For one coarse colour,
 *   every tile of that colour (they are independent: all sites around a tile belong to
 *   tiles of the other coarse colour, which rest) receives k HITS; a hit = update all sites
 *   of fine colour 0 of the tile, then all of fine colour 1 (fine colour = (x+y)&1, the
 *   usual checkerboard), each by the Metropolis rule of orc_ising_sweep.
 * Streams (one per thread of the paper's kernel: 1024^2 sites <-> 262144 threads,
 * PAPER.md:54): S = L*L/4.  Tiles of one coarse colour are numbered p = ty*(L/T/2) + txh,
 * tx = 2*txh + ((ty+C)&1); thread t < T*T/2 of a tile owns the fine-colour-c site
 * y_l = t/(T/2), x_l = 2*(t%(T/2)) + ((y_l+c)&1) for c = 0 and 1 (a horizontal domino);
 * stream s = p*(T*T/2) + t serves tile p of BOTH coarse colours.  Per sweep a stream
 * spends 4k draws in the order (C, hit, c): draw ((2*sweep + C)*k + hit)*2 + c.  */
int orc_ising_sweep_multihit(orc_rng *r, int8_t *sp, uint32_t L, double beta, uint32_t n_sweeps,
                             uint32_t T, uint32_t k_hits, int64_t *trace)
{
    if (!r || T < 2 || (T & 1) || L % T || ((L / T) & 1) || k_hits < 1) return -1;
    const uint64_t S = r->n_local, tpt = (uint64_t)T * T / 2; /* threads per tile */
    if (S != (uint64_t)L * L / 4) return -1;
    const uint32_t ntx = L / T, nth = ntx / 2;
    float P[5];
    orc_ising_accept_table(beta, P);
    uint32_t *draws = (uint32_t *)malloc(S * 2 * sizeof(uint32_t));
    if (!draws) return -1;
    for (uint32_t sw = 0; sw < n_sweeps; sw++) {
        for (uint32_t C = 0; C < 2; C++)
            for (uint32_t hit = 0; hit < k_hits; hit++) {
                orc_fill_u32(r, draws, 2); /* draws[2 s + c]: the stream's next two numbers */
                for (uint32_t c = 0; c < 2; c++) {
#pragma omp parallel for schedule(static)
                    for (uint64_t s = 0; s < S; s++) {
                        uint64_t p = s / tpt, t = s % tpt;
                        uint32_t ty = (uint32_t)(p / nth), txh = (uint32_t)(p % nth);
                        uint32_t tx = 2 * txh + ((ty + C) & 1);
                        uint32_t yl = (uint32_t)(t / (T / 2)), xl = 2 * (uint32_t)(t % (T / 2)) + ((yl + c) & 1);
                        uint64_t x = (uint64_t)tx * T + xl, y = (uint64_t)ty * T + yl;
                        int sc = sp[y * L + x];
                        int nn = sp[y * L + (x + 1) % L] + sp[y * L + (x + L - 1) % L]
                               + sp[((y + 1) % L) * L + x] + sp[((y + L - 1) % L) * L + x];
                        int h = sc * nn;
                        float u = orc_u32_to_f32(draws[2 * s + c]);
                        if (u < P[(h + 4) / 2]) sp[y * L + x] = (int8_t)(-sc);
                    }
                }
            }
        if (trace) trace[sw] = orc_ising_energy(sp, L);
    }
    free(draws);
    return 0;
}
