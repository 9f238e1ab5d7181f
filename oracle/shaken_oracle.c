/*
 * shaken_oracle.c -- ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).
 *
 * A plain, slow, single-threaded CPU statement of the shaken dynamics of
 * D'Autilia, Andrianaivo, Troiani, "Parallel simulation of two-dimensional
 * Ising models using Probabilistic Cellular Automata" (arXiv 1908.07341),
 * written from PAPER.md only.  It shares no code, header, table or constant
 * generator with the CUDA library under paper_1908_07341_b200/csrc and
 * neither imports the other.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may call it.
 *
 * What it computes (paper passages):
 *   lattice, neighbours     eq. (3)-(4)
 *   Hamiltonian H(s,t)      eq. (5)
 *   local fields            eq. (14)
 *   half-step at odd times  eq. (15)      PAPER.md:162-167   (tau  <- sigma, down/left field,  Alg. 2 :371-377)
 *   half-step at even times eq. (16)      PAPER.md:169-172   (sigma <- tau,  up/right field,   Alg. 1 :354-361)
 *   sampling rule           PAPER.md:174  P(zeta) = exp(zeta h) / (2 cosh h);  "if rand() < p" Alg. 3 :413,:433
 *   magnetisation           eq. (17)
 *
 * Readings of silent points: x=(i,j) -> column c=i, row r=j,
 * site = r*L + c; up = r+1, right = c+1, down = r-1, left = c-1 (mod L).
 * rand() is a counter-based Philox4x32-10 word (the paper used cuRAND's default
 * generator; BASELINE.json's north_star fixes Philox keyed by seed, chain, step,
 * half, site); "rand() < p" is taken on the 32-bit integer scale: r < T,
 * T = round(2^32 p) clamped to [1, 2^32-1].
 *
 * Pins (tests/test_oracle_*.py): Philox against cuRAND's host generator,
 * thresholds against exact big-float arithmetic, J=q=0 (spin = top bit of the
 * random word), J=0 closed-form contraction tanh(q), exact 2^9-state
 * transition matrix on the 3x3 torus built from eq. (15)-(16), detailed
 * balance w.r.t. pi_s = Z_sigma/Z, the two forms of eq. (5),
 * monotone coupling, observables by brute force; coupling groups and coalescence times
 * against pairs of uncoupled single-chain runs and the J = 0 closed form.
 * The site->counter mapping itself is a convention: parity unpinned beyond
 * self-consistency (by design).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------ */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): the public      */
/* algorithm restated.  Ten rounds; the key is bumped between rounds. */
/* ------------------------------------------------------------------ */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* The random word of one site in one half-step.
 * g = 2*t + half (t = 0-based full-step index), counter = (site>>2, chain, g lo, g hi),
 * key = (seed lo, seed hi), word (site & 3). */
static uint32_t rnd_word(uint64_t seed, uint32_t chain, uint64_t g, uint64_t site)
{
    uint32_t ctr[4] = { (uint32_t)(site >> 2), chain, (uint32_t)g, (uint32_t)(g >> 32) };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t out[4];
    oracle_philox4x32_10(ctr, key, out);
    return out[site & 3];
}

/* Random word of the init stream: counter = (site>>2, chain, which, 0xFFFFFFFF),
 * which = 0 for sigma, 1 for tau. */
static uint32_t init_word(uint64_t seed, uint32_t chain, uint32_t which, uint64_t site)
{
    uint32_t ctr[4] = { (uint32_t)(site >> 2), chain, which, 0xFFFFFFFFu };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t out[4];
    oracle_philox4x32_10(ctr, key, out);
    return out[site & 3];
}

/* ------------------------------------------------------------------ */
/* Heat-bath thresholds.  P(+ | h) = e^h / (2 cosh h) = 1/(1+e^{-2h}) */
/* (Alg. 3 line 3).  Integer scale: T = round(2^32 P),   */
/* computed for |h| and mirrored so that T(h) + T(-h) = 2^32 exactly.  */
/* ------------------------------------------------------------------ */
static uint32_t F_nonneg(double a)
{
    double p = 1.0 / (1.0 + exp(-2.0 * a));
    double v = floor(ldexp(p, 32) + 0.5);
    if (v < 2147483648.0) v = 2147483648.0;
    if (v > 4294967295.0) v = 4294967295.0;
    return (uint32_t)v;
}

uint32_t oracle_threshold(double h)
{
    if (h >= 0.0) return F_nonneg(h);
    return (uint32_t)(4294967296.0 - (double)F_nonneg(-h));
}

/* T[2k+c]: k = number of +1 among the two J-neighbours, c = [same-site spin == +1];
 * field (eq. 14) h = J*(2k-2) + q*(2c-1). */
void oracle_thresholds(double J, double q, uint32_t T[6])
{
    for (int k = 0; k < 3; ++k)
        for (int c = 0; c < 2; ++c) {
            double h = (double)(2 * k - 2) * J + (double)(2 * c - 1) * q;
            T[2 * k + c] = oracle_threshold(h);
        }
}

/* ------------------------------------------------------------------ */
/* Context                                                            */
/* ------------------------------------------------------------------ */
typedef struct oracle_ctx {
    int64_t L;
    int64_t n_chains;
    uint64_t seed;
    int8_t *sigma;      /* [chain][r][c] */
    int8_t *tau;        /* [chain][r][c] */
    uint64_t step;      /* number of full steps done (global index t) */
    int64_t *records;   /* [record][chain][6] */
    int64_t n_records;
    int64_t cap_records;
    int complement;     /* test hook: replace every random word r by 2^32-1-r */
    int64_t group;      /* coupling: chains c with equal c / group evolve "with the same update function and the same
                         * sequence of random numbers": all draw the words of chain (c / group) * group */
    int64_t *coal;      /* [n_chains / group] coalescence time T = min{n : X_n = Y_n} in full steps,
                         * -1 while the sigma layers of the group still differ */
} oracle_ctx;

enum { ORACLE_OK = 0, ORACLE_EINVAL = -1, ORACLE_ENOMEM = -2 };

int oracle_create(oracle_ctx **out, int64_t L, int64_t n_chains, uint64_t seed)
{
    if (!out || L < 1 || n_chains < 1 || L > 65536) return ORACLE_EINVAL;
    oracle_ctx *o = (oracle_ctx *)calloc(1, sizeof(*o));
    if (!o) return ORACLE_ENOMEM;
    o->L = L; o->n_chains = n_chains; o->seed = seed;
    size_t n = (size_t)n_chains * (size_t)L * (size_t)L;
    o->sigma = (int8_t *)malloc(n);
    o->tau = (int8_t *)malloc(n);
    if (!o->sigma || !o->tau) { free(o->sigma); free(o->tau); free(o); return ORACLE_ENOMEM; }
    memset(o->sigma, 1, n);
    memset(o->tau, 1, n);
    o->group = 1;
    *out = o;
    return ORACLE_OK;
}

/* Coupled chains.  group >= 1 must divide n_chains; group = 1 uncouples.  Forgets coalescence times. */
int oracle_set_coupling(oracle_ctx *o, int64_t group)
{
    if (!o || group < 1 || o->n_chains % group != 0) return ORACLE_EINVAL;
    free(o->coal);
    o->coal = NULL;
    o->group = group;
    if (group > 1) {
        int64_t ng = o->n_chains / group;
        o->coal = (int64_t *)malloc((size_t)ng * sizeof(int64_t));
        if (!o->coal) return ORACLE_ENOMEM;
        for (int64_t i = 0; i < ng; ++i) o->coal[i] = -1;
    }
    return ORACLE_OK;
}

/* Coalescence times of the groups, -1 = not yet; returns the number of groups written (0 when uncoupled). */
int64_t oracle_coalescence(const oracle_ctx *o, int64_t *out, int64_t max_groups)
{
    if (!o || max_groups < 0) return ORACLE_EINVAL;
    if (o->group <= 1) return 0;
    int64_t ng = o->n_chains / o->group, n = ng < max_groups ? ng : max_groups;
    for (int64_t i = 0; i < n; ++i) out[i] = o->coal[i];
    return n;
}

void oracle_destroy(oracle_ctx *o)
{
    if (!o) return;
    free(o->sigma); free(o->tau); free(o->records); free(o->coal); free(o);
}

/* mode +1: all +1; -1: all -1; 0: iid +-1 from the init stream (spin = +1 iff word < 2^31);
 * 2 ("sandwich"): the first chain of every coupling group all +1 (sigma^top), the others all -1 (sigma^bot). */
int oracle_init(oracle_ctx *o, int mode)
{
    if (!o || (mode != 1 && mode != -1 && mode != 0 && mode != 2)) return ORACLE_EINVAL;
    int64_t L = o->L;
    uint64_t nsite = (uint64_t)L * (uint64_t)L;
    for (int64_t ch = 0; ch < o->n_chains; ++ch)
        for (uint64_t x = 0; x < nsite; ++x) {
            int8_t s, t;
            if (mode == 0) {
                s = init_word(o->seed, (uint32_t)ch, 0u, x) < 0x80000000u ? 1 : -1;
                t = init_word(o->seed, (uint32_t)ch, 1u, x) < 0x80000000u ? 1 : -1;
            } else if (mode == 2) {
                s = t = (int8_t)(ch % o->group == 0 ? 1 : -1);
            } else {
                s = t = (int8_t)mode;
            }
            o->sigma[(uint64_t)ch * nsite + x] = s;
            o->tau[(uint64_t)ch * nsite + x] = t;
        }
    o->step = 0;
    o->n_records = 0;
    if (o->coal)
        for (int64_t i = 0; i < o->n_chains / o->group; ++i) o->coal[i] = -1;
    return ORACLE_OK;
}

void oracle_set_complement(oracle_ctx *o, int on) { o->complement = on ? 1 : 0; }

static inline int64_t wrap(int64_t a, int64_t L) { a %= L; return a < 0 ? a + L : a; }

/* The six int64 sums of one chain on the pair (sigma, tau):
 * M_sigma, M_tau, E_J = sum_x sigma_x (tau_up + tau_right), E_q = sum_x sigma_x tau_x   (eq. 5, first form)
 * C_x = sum_x sigma_x sigma_right, C_y = sum_x sigma_x sigma_up   (square-lattice bonds of the sigma layer). */
void oracle_measure(const int8_t *sigma, const int8_t *tau, int64_t L, int64_t out[6])
{
    int64_t Ms = 0, Mt = 0, EJ = 0, Eq = 0, Cx = 0, Cy = 0;
    for (int64_t r = 0; r < L; ++r)
        for (int64_t c = 0; c < L; ++c) {
            int64_t s = sigma[r * L + c], t = tau[r * L + c];
            int64_t up = wrap(r + 1, L), right = wrap(c + 1, L);
            Ms += s;
            Mt += t;
            EJ += s * ((int64_t)tau[up * L + c] + (int64_t)tau[r * L + right]);
            Eq += s * t;
            Cx += s * (int64_t)sigma[r * L + right];
            Cy += s * (int64_t)sigma[up * L + c];
        }
    out[0] = Ms; out[1] = Mt; out[2] = EJ; out[3] = Eq; out[4] = Cx; out[5] = Cy;
}

/* One half-step of one chain, rows r0 .. r0+nrows-1 of the target only (the whole lattice when r0 = 0,
 * nrows = L).  half = 0: tau <- heat bath on the down/left field of sigma (eq. 15); half = 1: sigma <- heat
 * bath on the up/right field of tau (eq. 16).  src (L x L) is read; dst_rows points at row r0 of the target. */
static void half_step_rows(int64_t L, uint64_t seed, int complement, int64_t ch, const uint32_t T[6], int half,
                           const int8_t *src, int8_t *dst_rows, uint64_t t, int64_t r0, int64_t nrows)
{
    int64_t d = half == 0 ? -1 : +1;
    uint64_t g = 2u * t + (uint64_t)half;
    for (int64_t r = r0; r < r0 + nrows; ++r)
        for (int64_t c = 0; c < L; ++c) {
            int8_t vert = src[wrap(r + d, L) * L + c];      /* down (half 0) / up (half 1)    */
            int8_t horz = src[r * L + wrap(c + d, L)];      /* left (half 0) / right (half 1) */
            int8_t self = src[r * L + c];
            int k = (vert == 1) + (horz == 1);
            int idx = 2 * k + (self == 1);
            uint32_t rw = rnd_word(seed, (uint32_t)ch, g, (uint64_t)(r * L + c));
            if (complement) rw = ~rw;
            dst_rows[(r - r0) * L + c] = rw < T[idx] ? 1 : -1;
        }
}

static void half_step(const oracle_ctx *o, int64_t ch, const uint32_t T[6], int half,
                      const int8_t *src, int8_t *dst, uint64_t t)
{
    half_step_rows(o->L, o->seed, o->complement, ch, T, half, src, dst, t, 0, o->L);
}

/* Context-free form for full-size spot checks: rows r0 .. r0+nrows-1 of one half-step of chain `chain` at
 * full-step index t, from a caller-supplied source sublattice (L x L, +-1).  Same per-site statement as above. */
int oracle_half_step_rows(const int8_t *src, int8_t *dst_rows, int64_t L, uint64_t seed, int64_t chain,
                          double J, double q, uint64_t t, int half, int64_t r0, int64_t nrows)
{
    if (!src || !dst_rows || L < 1 || (half != 0 && half != 1) || r0 < 0 || nrows < 0 || r0 + nrows > L)
        return ORACLE_EINVAL;
    uint32_t T[6];
    oracle_thresholds(J, q, T);
    half_step_rows(L, seed, 0, chain, T, half, src, dst_rows, t, r0, nrows);
    return ORACLE_OK;
}

static int push_record(oracle_ctx *o)
{
    if (o->n_records == o->cap_records) {
        int64_t cap = o->cap_records ? 2 * o->cap_records : 64;
        int64_t *p = (int64_t *)realloc(o->records, (size_t)cap * (size_t)o->n_chains * 6 * sizeof(int64_t));
        if (!p) return ORACLE_ENOMEM;
        o->records = p; o->cap_records = cap;
    }
    size_t nsite = (size_t)o->L * (size_t)o->L;
    for (int64_t ch = 0; ch < o->n_chains; ++ch)
        oracle_measure(o->sigma + (size_t)ch * nsite, o->tau + (size_t)ch * nsite, o->L,
                       o->records + ((size_t)o->n_records * (size_t)o->n_chains + (size_t)ch) * 6);
    o->n_records++;
    return ORACLE_OK;
}

/* Advance every chain by n_steps full steps with per-chain couplings J[ch], q[ch].
 * A record is appended after each full step whose 1-based global index is a multiple of obs_every. */
int oracle_run_grid(oracle_ctx *o, const double *J, const double *q, int64_t n_steps, int64_t obs_every)
{
    if (!o || !J || !q || n_steps < 0 || obs_every < 0) return ORACLE_EINVAL;
    for (int64_t ch = 0; ch < o->n_chains; ++ch)
        if (!isfinite(J[ch]) || !isfinite(q[ch])) return ORACLE_EINVAL;
    size_t nsite = (size_t)o->L * (size_t)o->L;
    uint32_t *T = (uint32_t *)malloc((size_t)o->n_chains * 6 * sizeof(uint32_t));
    if (!T) return ORACLE_ENOMEM;
    for (int64_t ch = 0; ch < o->n_chains; ++ch) oracle_thresholds(J[ch], q[ch], T + 6 * ch);
    for (int64_t s = 0; s < n_steps; ++s) {
        for (int64_t ch = 0; ch < o->n_chains; ++ch) {
            int8_t *sg = o->sigma + (size_t)ch * nsite, *ta = o->tau + (size_t)ch * nsite;
            int64_t rng_chain = (ch / o->group) * o->group;      /* the same random numbers within a group */
            half_step(o, rng_chain, T + 6 * ch, 0, sg, ta, o->step);
            half_step(o, rng_chain, T + 6 * ch, 1, ta, sg, o->step);
        }
        o->step++;
        if (o->coal)                                             /* T = min{n : X_n = Y_n} on the sigma layer */
            for (int64_t gi = 0; gi < o->n_chains / o->group; ++gi) {
                if (o->coal[gi] >= 0) continue;
                const int8_t *first = o->sigma + (size_t)(gi * o->group) * nsite;
                int same = 1;
                for (int64_t m = 1; m < o->group && same; ++m)
                    same = memcmp(first, first + (size_t)m * nsite, nsite) == 0;
                if (same) o->coal[gi] = (int64_t)o->step;
            }
        if (obs_every > 0 && o->step % (uint64_t)obs_every == 0) {
            int rc = push_record(o);
            if (rc) { free(T); return rc; }
        }
    }
    free(T);
    return ORACLE_OK;
}

int oracle_run(oracle_ctx *o, double J, double q, int64_t n_steps, int64_t obs_every)
{
    if (!o) return ORACLE_EINVAL;
    double *Ja = (double *)malloc((size_t)o->n_chains * sizeof(double));
    double *qa = (double *)malloc((size_t)o->n_chains * sizeof(double));
    if (!Ja || !qa) { free(Ja); free(qa); return ORACLE_ENOMEM; }
    for (int64_t ch = 0; ch < o->n_chains; ++ch) { Ja[ch] = J; qa[ch] = q; }
    int rc = oracle_run_grid(o, Ja, qa, n_steps, obs_every);
    free(Ja); free(qa);
    return rc;
}

/* ------------------------------------------------------------------ */
/* Alternate parallel heat bath on the SQUARE lattice:  */
/* "a parallel version of the heat bath dynamics that updates,         */
/* alternatively, the spins on the odd and the even sites of the       */
/* lattice", whose equilibrium measure is the Gibbs measure of the     */
/* square-lattice Ising model with coupling J.  One spin field (the    */
/* sigma array; tau is not touched), L even.  Site (r, c) has colour   */
/* (r + c) & 1; half-step `half` of full step t redraws every site of  */
/* colour `half` by heat bath on h = J * (sum of its four neighbours): */
/* +1 iff rnd < A[k], k = number of +1 neighbours, h = J (2k - 4).     */
/* The sites of one colour, numbered m = 0, 1, ... in row-major order  */
/* (m = (r L + c) >> 1), draw the words the shaken half-step g = 2t +  */
/* half gives sites 0, 1, ...: word m & 3 of counter (m >> 2, chain,   */
/* g lo, g hi).                                                        */
/* ------------------------------------------------------------------ */
void oracle_alt_thresholds(double J, uint32_t A[5])
{
    for (int k = 0; k < 5; ++k) A[k] = oracle_threshold((double)(2 * k - 4) * J);
}

/* Rows r0 .. r0+nrows-1 of the lattice after one half-step; src (L x L) is the lattice before it. */
static void alt_half_step_rows(int64_t L, uint64_t seed, int complement, int64_t ch, const uint32_t A[5], int half,
                               const int8_t *src, int8_t *dst_rows, uint64_t t, int64_t r0, int64_t nrows)
{
    uint64_t g = 2u * t + (uint64_t)half;
    for (int64_t r = r0; r < r0 + nrows; ++r)
        for (int64_t c = 0; c < L; ++c) {
            int8_t out = src[r * L + c];
            if (((r + c) & 1) == half) {
                int k = (src[wrap(r + 1, L) * L + c] == 1) + (src[wrap(r - 1, L) * L + c] == 1) +
                        (src[r * L + wrap(c + 1, L)] == 1) + (src[r * L + wrap(c - 1, L)] == 1);
                uint32_t rw = rnd_word(seed, (uint32_t)ch, g, (uint64_t)(r * L + c) >> 1);
                if (complement) rw = ~rw;
                out = rw < A[k] ? 1 : -1;
            }
            dst_rows[(r - r0) * L + c] = out;
        }
}

int oracle_alt_half_step_rows(const int8_t *src, int8_t *dst_rows, int64_t L, uint64_t seed, int64_t chain,
                              double J, uint64_t t, int half, int64_t r0, int64_t nrows)
{
    if (!src || !dst_rows || L < 2 || (L & 1) || (half != 0 && half != 1) || r0 < 0 || nrows < 0 || r0 + nrows > L)
        return ORACLE_EINVAL;
    uint32_t A[5];
    oracle_alt_thresholds(J, A);
    alt_half_step_rows(L, seed, 0, chain, A, half, src, dst_rows, t, r0, nrows);
    return ORACLE_OK;
}

/* n_steps full steps (even sites, then odd sites) of every chain with per-chain coupling J[ch].  Coupling groups and
 * coalescence times as in oracle_run_grid.  A record after a step holds (M, 0, 0, 0, C_x, C_y) of the sigma array:
 * H(sigma) = -J (C_x + C_y). */
int oracle_run_alternate(oracle_ctx *o, const double *J, int64_t n_steps, int64_t obs_every)
{
    if (!o || !J || n_steps < 0 || obs_every < 0 || (o->L & 1)) return ORACLE_EINVAL;
    for (int64_t ch = 0; ch < o->n_chains; ++ch)
        if (!isfinite(J[ch])) return ORACLE_EINVAL;
    size_t nsite = (size_t)o->L * (size_t)o->L;
    int8_t *tmp = (int8_t *)malloc(nsite);
    if (!tmp) return ORACLE_ENOMEM;
    for (int64_t s = 0; s < n_steps; ++s) {
        for (int64_t ch = 0; ch < o->n_chains; ++ch) {
            int8_t *sg = o->sigma + (size_t)ch * nsite;
            int64_t rng_chain = (ch / o->group) * o->group;
            uint32_t A[5];
            oracle_alt_thresholds(J[ch], A);
            for (int half = 0; half < 2; ++half) {
                alt_half_step_rows(o->L, o->seed, o->complement, rng_chain, A, half, sg, tmp, o->step, 0, o->L);
                memcpy(sg, tmp, nsite);
            }
        }
        o->step++;
        if (o->coal)
            for (int64_t gi = 0; gi < o->n_chains / o->group; ++gi) {
                if (o->coal[gi] >= 0) continue;
                const int8_t *first = o->sigma + (size_t)(gi * o->group) * nsite;
                int same = 1;
                for (int64_t m = 1; m < o->group && same; ++m)
                    same = memcmp(first, first + (size_t)m * nsite, nsite) == 0;
                if (same) o->coal[gi] = (int64_t)o->step;
            }
        if (obs_every > 0 && o->step % (uint64_t)obs_every == 0) {
            int rc = push_record(o);
            if (rc) { free(tmp); return rc; }
            int64_t *rec = o->records + (size_t)(o->n_records - 1) * (size_t)o->n_chains * 6;
            for (int64_t ch = 0; ch < o->n_chains; ++ch) rec[ch * 6 + 1] = rec[ch * 6 + 2] = rec[ch * 6 + 3] = 0;
        }
    }
    free(tmp);
    return ORACLE_OK;
}

/* Copy min(n_records, max_records) records, layout [record][chain][6]; returns the count. */
int64_t oracle_observables(const oracle_ctx *o, int64_t *out, int64_t max_records)
{
    if (!o || max_records < 0) return ORACLE_EINVAL;
    int64_t n = o->n_records < max_records ? o->n_records : max_records;
    if (n > 0) {
        if (!out) return ORACLE_EINVAL;
        memcpy(out, o->records, (size_t)n * (size_t)o->n_chains * 6 * sizeof(int64_t));
    }
    return n;
}

int64_t oracle_num_records(const oracle_ctx *o) { return o ? o->n_records : ORACLE_EINVAL; }

/* which = 0: sigma, 1: tau; host buffer of n_chains*L*L int8 (+1/-1). */
int oracle_get_spins(const oracle_ctx *o, int which, int8_t *host)
{
    if (!o || !host || (which != 0 && which != 1)) return ORACLE_EINVAL;
    size_t n = (size_t)o->n_chains * (size_t)o->L * (size_t)o->L;
    memcpy(host, which == 0 ? o->sigma : o->tau, n);
    return ORACLE_OK;
}

int oracle_set_spins(oracle_ctx *o, int which, const int8_t *host)
{
    if (!o || !host || (which != 0 && which != 1)) return ORACLE_EINVAL;
    size_t n = (size_t)o->n_chains * (size_t)o->L * (size_t)o->L;
    for (size_t i = 0; i < n; ++i)
        if (host[i] != 1 && host[i] != -1) return ORACLE_EINVAL;
    memcpy(which == 0 ? o->sigma : o->tau, host, n);
    return ORACLE_OK;
}

/* Diagonal spin-spin correlations of the sigma layer (Table 1), as translation-averaged integer sums
 * over the torus.  With x = (i, j) -> column i, row j:
 *   SW-NE  pi(sigma_{0,0} sigma_{l,l}):  out[..][0] = sum_{r,c} sigma[r][c]   * sigma[r+l][c+l]
 *   NW-SE  pi(sigma_{0,l} sigma_{l,0}):  out[..][1] = sum_{r,c} sigma[r+l][c] * sigma[r][c+l]        (indices mod L)
 * out layout [chain][n_ell][2]. */
int oracle_diag_correlations(const oracle_ctx *o, const int64_t *ells, int64_t n_ell, int64_t *out)
{
    if (!o || !ells || !out || n_ell < 0) return ORACLE_EINVAL;
    int64_t L = o->L;
    size_t nsite = (size_t)L * (size_t)L;
    for (int64_t ch = 0; ch < o->n_chains; ++ch) {
        const int8_t *sg = o->sigma + (size_t)ch * nsite;
        for (int64_t e = 0; e < n_ell; ++e) {
            int64_t l = ells[e], swne = 0, nwse = 0;
            for (int64_t r = 0; r < L; ++r)
                for (int64_t c = 0; c < L; ++c) {
                    int64_t r2 = wrap(r + l, L), c2 = wrap(c + l, L);
                    swne += (int64_t)sg[r * L + c] * (int64_t)sg[r2 * L + c2];
                    nwse += (int64_t)sg[r2 * L + c] * (int64_t)sg[r * L + c2];
                }
            out[((size_t)ch * (size_t)n_ell + (size_t)e) * 2 + 0] = swne;
            out[((size_t)ch * (size_t)n_ell + (size_t)e) * 2 + 1] = nwse;
        }
    }
    return ORACLE_OK;
}

uint64_t oracle_get_step(const oracle_ctx *o) { return o ? o->step : 0; }
int oracle_set_step(oracle_ctx *o, uint64_t step) { if (!o) return ORACLE_EINVAL; o->step = step; return ORACLE_OK; }
