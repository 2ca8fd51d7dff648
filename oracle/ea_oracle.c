/*
 * ea_oracle.c -- CPU ORACLE for the checkerboard Metropolis sweep of the 3D +-J
 * Edwards-Anderson model and its popcount observables.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code
 * with the CUDA path (paper_1411_5512_b200/csrc): the two sides implement the same
 * WRITTEN stream definition ("Contract") independently.
 *
 * Style: plain, slow, obviously correct.  One spin per byte (+1 / -1), one bond per
 * byte (+1 / -1), scalar per-site Metropolis in the paper's order.  No bit tricks, no
 * blocking, no fusion.  The only concession to speed is "#pragma omp parallel for" over
 * the 64 independent samples (lanes), which never interact.
 *
 * Citations are PAPER.md:<line> (Manssen & Hartmann, arXiv:1411.5512) plus the
 * section / equation the line falls in; "C-xx" are the readings listed in DESIGN.md
 * section 2 (taken from SURVEY.md section 8(c)) where the paper is silent.
 *
 * Pins (tests/test_oracle_pins.py, all "-m 'not gpu'"): Philox known-answer vectors,
 * thresholds closed form, single-site acceptance, L=2 Boltzmann statistics by brute
 * force, energy bookkeeping, T=0 monotonicity, p=1 ground state, T=inf alternation,
 * exact gauge equivalence, order independence, lane independence, observables against
 * numpy (roll / FFT) restatements; full-vector C_4 against the 3-D FFT and closed-form
 * anisotropic fields (P14); heat-bath thresholds, detailed-balance ratio and the L = 2
 * transition matrix (P16).  The fp64 post-processing (C_4 curve, integral estimator,
 * P15) lives in oracle/__init__.py.  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_LANES 64 /* PAPER.md:90-92 (III): 64 samples per 64-bit multispin word */

typedef struct oracle_sim {
    int L;          /* side length, even, >= 2  (II)                      */
    int64_t N;      /* L^3 sites                                                        */
    int n_replicas; /* 1: 64 independent samples; 2: 32 disorders x 2 replicas (:33)    */
    double p, T;    /* bond fraction and temperature (Eq. 9, :77)         */
    uint64_t seed;
    uint64_t t;      /* completed sweeps since the random start           */
    uint64_t thr[3]; /* integer acceptance thresholds for n_u = 0,1,2 (C-A4)            */
    int dynamics;       /* 0: Metropolis (Eq. 9, the paper's); 1: heat bath (C-HB)          */
    uint64_t thr_hb[7]; /* heat-bath thresholds for n_u = 0..6 (C-HB)                       */
    int8_t *S;       /* S[lane*N + site]            = +-1                               */
    int8_t *J;       /* J[(lane*3 + d)*N + site]    = +-1, forward bond site->site+e_d  */
    int8_t *snap;    /* n_slots snapshots of S                                           */
    uint64_t *snap_t;
    int *snap_set;
    int n_slots;
    int64_t dE_accum[ORACLE_LANES]; /* sum of accepted Delta E per lane (pin P4)         */
    int order;       /* 0 ascending, 1 descending, 2 pseudo-shuffled (pin P9)            */
    uint32_t *r_lo, *r_hi; /* scratch: per-site random numbers of the current half-sweep */
} oracle_sim;

/* ------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  The paper's own generator is an
 * unspecified 1024-bit xorshift (ref. 42); BASELINE north_star replaces it
 * by a counter-based generator.  Reading C-A6.
 * ---------------------------------------------------------------------------------- */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = M0 * (uint64_t)c0; /* 32x32 -> 64 bit products */
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1; /* Weyl key schedule, bumped after every round */
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Stream tags, 4th counter word (C-A6). */
enum { TAG_UPDATE_PARITY0 = 0, TAG_UPDATE_PARITY1 = 1, TAG_INIT_SPINS = 2, TAG_BONDS = 3 };

static void stream_block(const oracle_sim *s, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t tag,
                         uint32_t out[4])
{
    uint32_t ctr[4] = { c0, c1, c2, tag };
    uint32_t key[2] = { (uint32_t)(s->seed & 0xffffffffu), (uint32_t)(s->seed >> 32) };
    oracle_philox4x32_10(ctr, key, out);
}

/* ------------------------------------------------------------------------------------
 * Acceptance thresholds.  Eq. 9: p_accept = min(1, exp(-(2/T) sum_j J_ij S_i S_j)).
 * With n_u unsatisfied bonds among the 6, sum_j J_ij S_i S_j = 6 - 2 n_u, so for
 * n_u = 0,1,2 the exponent is -(2/T)(6 - 2 n_u) = -4 (3 - n_u) / T; for n_u >= 3 the
 * probability is 1.  "Precalculated flipping probabilities" become the
 * integers thr[n_u] = floor(2^32 * exp(-4 (3 - n_u) / T) + 0.5); a uniform 32-bit r
 * accepts iff r < thr  (C-A4, C-S5).  T = 0 -> 0, T = +inf -> 2^32 (always).
 * ---------------------------------------------------------------------------------- */
void oracle_thresholds(double T, uint64_t thr[3])
{
    for (int n_u = 0; n_u < 3; ++n_u) {
        double prob = exp(-(4.0 * (double)(3 - n_u)) / T);
        thr[n_u] = (uint64_t)floor(4294967296.0 * prob + 0.5);
    }
}

/* Heat-bath variant (NOT the paper's dynamics, which is Metropolis) -- reading
 * C-HB: a spin is flipped with probability 1 / (1 + exp(Delta E / T)), Delta E = 2 sum_j J_ij S_i S_j = 12 - 4 n_u,
 * for every n_u = 0..6 (no "always flip" shortcut; Delta E = 0 gives exactly 1/2 at any T, T = 0 gives 0, 1/2, 1).
 * thr_hb[n_u] = floor(2^32 P + 0.5), compared with the same 32-bit numbers by the same strict "<". */
void oracle_thresholds_heatbath(double T, uint64_t thr[7])
{
    for (int n_u = 0; n_u < 7; ++n_u) {
        double dE = 12.0 - 4.0 * (double)n_u;
        double w = dE == 0.0 ? 1.0 : exp(dE / T); /* 0/0 at T = 0 is the Delta E = 0 case: weight 1 */
        double prob = 1.0 / (1.0 + w);
        thr[n_u] = (uint64_t)floor(4294967296.0 * prob + 0.5);
    }
}

int oracle_accept_heatbath(const uint64_t thr[7], int local_sum, uint32_t r)
{
    int n_u = (6 - local_sum) / 2; /* 0..6 */
    return (uint64_t)r < thr[n_u];
}

/* P(J = +1) = p as an integer threshold on a 32-bit uniform (C-A9). */
uint64_t oracle_bond_threshold(double p) { return (uint64_t)floor(4294967296.0 * p + 0.5); }

/* Eq. 9 decision for one spin: local_sum = sum_j J_ij S_i S_j in {-6,-4,...,6}. */
int oracle_accept(const uint64_t thr[3], int local_sum, uint32_t r)
{
    if (local_sum <= 0) return 1;    /* Delta E = 2*local_sum <= 0: min(1, e^{>=0}) = 1, incl. Delta E = 0 (C-S6) */
    int n_u = (6 - local_sum) / 2;   /* 0, 1 or 2 */
    return (uint64_t)r < thr[n_u];
}

/* ------------------------------------------------------------------------------------
 * Lattice (C-A1): site = x + L*(y + L*z), periodic in all directions.
 * Bond (d, site) couples site and site + e_d; only forward bonds are stored (:88).
 * ---------------------------------------------------------------------------------- */
static inline int64_t site_of(int L, int x, int y, int z) { return (int64_t)x + (int64_t)L * ((int64_t)y + (int64_t)L * z); }
static inline int wrap(int a, int L) { return (a % L + L) % L; }

/* The site r steps from `site` along axis d (r may be negative), periodic. */
int64_t oracle_shift(int L, int64_t site, int d, int r)
{
    int x = (int)(site % L), y = (int)((site / L) % L), z = (int)(site / ((int64_t)L * L));
    if (d == 0) x = wrap(x + r, L);
    if (d == 1) y = wrap(y + r, L);
    if (d == 2) z = wrap(z + r, L);
    return site_of(L, x, y, z);
}

int64_t oracle_neighbour(int L, int64_t site, int d, int sign) { return oracle_shift(L, site, d, sign); }

/* One periodic step from coordinate a (sign = +1 or -1). */
static inline int step(int a, int sign, int L)
{
    int b = a + sign;
    if (b == L) b = 0;
    if (b < 0) b = L - 1;
    return b;
}

/* sum_j J_ij S_i S_j over the 6 bonds at site (x, y, z), sample `lane` (Eq. 9 / Eq. 1). */
static int local_sum_xyz(const oracle_sim *s, int lane, int x, int y, int z)
{
    const int L = s->L;
    const int64_t N = s->N;
    const int8_t *S = s->S + (int64_t)lane * N;
    const int8_t *J = s->J + (int64_t)lane * 3 * N; /* J[d*N + site] */
    const int64_t site = site_of(L, x, y, z);
    const int64_t xp = site_of(L, step(x, +1, L), y, z), xm = site_of(L, step(x, -1, L), y, z);
    const int64_t yp = site_of(L, x, step(y, +1, L), z), ym = site_of(L, x, step(y, -1, L), z);
    const int64_t zp = site_of(L, x, y, step(z, +1, L)), zm = site_of(L, x, y, step(z, -1, L));
    int sum = 0;
    sum += J[0 * N + site] * S[site] * S[xp]; /* own forward bonds ...                  */
    sum += J[1 * N + site] * S[site] * S[yp];
    sum += J[2 * N + site] * S[site] * S[zp];
    sum += J[0 * N + xm] * S[site] * S[xm];   /* ... and the backward neighbours' ones  */
    sum += J[1 * N + ym] * S[site] * S[ym];
    sum += J[2 * N + zm] * S[site] * S[zm];
    return sum;
}

int oracle_local_sum(const oracle_sim *s, int lane, int64_t site)
{
    const int L = s->L;
    return local_sum_xyz(s, lane, (int)(site % L), (int)((site / L) % L), (int)(site / ((int64_t)L * L)));
}

/* ------------------------------------------------------------------------------------
 * Setup (C-A8, C-A9).  Random start = quench from T = inf; bonds iid from
 * P(J) = p delta(J-1) + (1-p) delta(J+1).  Bit/sign encoding of the packed
 * formats: bit 1 <-> -1 (C-A2).
 * ---------------------------------------------------------------------------------- */
static void init_spins(oracle_sim *s)
{
    for (int64_t site = 0; site < s->N; ++site) {
        uint32_t out[4];
        stream_block(s, (uint32_t)site, 0u, 0u, TAG_INIT_SPINS, out);
        for (int lane = 0; lane < ORACLE_LANES; ++lane) {
            uint32_t word = lane < 32 ? out[0] : out[1];
            int bit = (word >> (lane & 31)) & 1u;
            s->S[(int64_t)lane * s->N + site] = bit ? -1 : +1;
        }
    }
}

static void init_bonds(oracle_sim *s)
{
    uint64_t P = oracle_bond_threshold(s->p);
    int drawn = s->n_replicas == 2 ? 32 : 64;
    for (int64_t site = 0; site < s->N; ++site)
        for (int d = 0; d < 3; ++d)
            for (int lane = 0; lane < drawn; ++lane) {
                uint32_t out[4];
                stream_block(s, (uint32_t)site, (uint32_t)(16 * d + (lane >> 2)), 0u, TAG_BONDS, out);
                uint32_t v = out[lane & 3];
                int8_t Jv = ((uint64_t)v < P) ? +1 : -1;
                s->J[((int64_t)lane * 3 + d) * s->N + site] = Jv;
                if (s->n_replicas == 2) /* replica b+32 has "the same bond configuration" */
                    s->J[((int64_t)(lane + 32) * 3 + d) * s->N + site] = Jv;
            }
}

oracle_sim *oracle_create(int L, double p, double T, int n_replicas, uint64_t seed, int n_slots)
{
    if (L < 2 || (L & 1) || (n_replicas != 1 && n_replicas != 2) || n_slots < 0) return NULL;
    if (!(p >= 0.0 && p <= 1.0) || !(T >= 0.0)) return NULL;
    oracle_sim *s = (oracle_sim *)calloc(1, sizeof(oracle_sim));
    s->L = L; s->N = (int64_t)L * L * L; s->n_replicas = n_replicas;
    s->p = p; s->T = T; s->seed = seed; s->t = 0; s->n_slots = n_slots;
    oracle_thresholds(T, s->thr);
    s->dynamics = 0;
    oracle_thresholds_heatbath(T, s->thr_hb);
    s->S = (int8_t *)malloc((size_t)ORACLE_LANES * s->N);
    s->J = (int8_t *)malloc((size_t)ORACLE_LANES * 3 * s->N);
    s->snap = n_slots ? (int8_t *)malloc((size_t)n_slots * ORACLE_LANES * s->N) : NULL;
    s->snap_t = (uint64_t *)calloc(n_slots ? n_slots : 1, sizeof(uint64_t));
    s->snap_set = (int *)calloc(n_slots ? n_slots : 1, sizeof(int));
    s->r_lo = (uint32_t *)malloc((size_t)s->N * sizeof(uint32_t));
    s->r_hi = (uint32_t *)malloc((size_t)s->N * sizeof(uint32_t));
    init_spins(s);
    init_bonds(s);
    return s;
}

void oracle_destroy(oracle_sim *s)
{
    if (!s) return;
    free(s->S); free(s->J); free(s->snap); free(s->snap_t); free(s->snap_set); free(s->r_lo); free(s->r_hi);
    free(s);
}

void oracle_set_temperature(oracle_sim *s, double T) { s->T = T; oracle_thresholds(T, s->thr); oracle_thresholds_heatbath(T, s->thr_hb); }
int oracle_set_dynamics(oracle_sim *s, int dynamics) { if (dynamics != 0 && dynamics != 1) return 1; s->dynamics = dynamics; return 0; }
void oracle_get_thresholds(const oracle_sim *s, uint64_t thr[3]) { memcpy(thr, s->thr, sizeof(s->thr)); }
uint64_t oracle_get_time(const oracle_sim *s) { return s->t; }
void oracle_set_time(oracle_sim *s, uint64_t t) { s->t = t; }
void oracle_set_order(oracle_sim *s, int order) { s->order = order; }
void oracle_set_threads(int n)
{
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int oracle_get_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
int8_t *oracle_spin_bytes(oracle_sim *s) { return s->S; } /* [64][N]    +-1, for numpy pins */
int8_t *oracle_bond_bytes(oracle_sim *s) { return s->J; } /* [64][3][N] +-1                 */
const int64_t *oracle_dE_accum(const oracle_sim *s) { return s->dE_accum; }

/* ------------------------------------------------------------------------------------
 * One half-sweep: every site of one colour gets one Metropolis trial.
 * Random numbers (C-A6, C-A7): the same-colour sites of one x-row are x = s, s+2, s+4, ...;
 * number them j = x >> 1 = 0 .. L/2 - 1.  Sites j (even) and j + 1 form a pair and share ONE
 * Philox block per sweep, counter (site index of the pair's first site, t lo, t hi,
 * tag = parity): the first site takes out[0] (samples 0..31) and out[1] (samples 32..63),
 * the second takes out[2] and out[3].  (L/2 odd: the last site of a row is a pair of its
 * own; L = 2: every site is.)  All four words of a block are used, none twice.
 * "It is customary to save computational effort by using only one random number for
 * multiple samples"; the two replicas never share one.
 * Same-colour sites are never neighbours (L even), so the visiting order is immaterial;
 * `order` exists only so a test can demonstrate that.
 * ---------------------------------------------------------------------------------- */
static int64_t visit(const oracle_sim *s, int64_t k)
{
    if (s->order == 1) return s->N - 1 - k;
    if (s->order == 2) { /* a fixed bijection of [0, N): multiply by an odd number mod N if N is a power of two, else reverse pairs */
        if ((s->N & (s->N - 1)) == 0) return (k * 0x9E3779B1LL + 12345) & (s->N - 1);
        return k ^ 1;
    }
    return k;
}

/* One Metropolis trial of spin (x,y,z) of sample `lane` (Eq. 9); returns the energy change it caused. */
static int metropolis_trial(oracle_sim *s, int lane, int x, int y, int z)
{
    int64_t site = site_of(s->L, x, y, z);
    int8_t *S = s->S + (int64_t)lane * s->N;
    int local_sum = local_sum_xyz(s, lane, x, y, z);
    uint32_t r = lane < 32 ? s->r_lo[site] : s->r_hi[site]; /* C-A7 */
    if (!(s->dynamics == 0 ? oracle_accept(s->thr, local_sum, r) : oracle_accept_heatbath(s->thr_hb, local_sum, r))) return 0;
    S[site] = (int8_t)-S[site];
    return 2 * local_sum; /* Delta E of the flip = 2 sum_j J_ij S_i S_j (Eq. 1) */
}

void oracle_half_sweep(oracle_sim *s, int parity)
{
    const int L = s->L;
    const int64_t N = s->N;
    uint32_t tag = parity == 0 ? TAG_UPDATE_PARITY0 : TAG_UPDATE_PARITY1;
    for (int64_t site = 0; site < N; ++site) {
        int x = (int)(site % L), y = (int)((site / L) % L), z = (int)(site / ((int64_t)L * L));
        if (((x + y + z) & 1) != parity) continue;
        int j = x >> 1;                /* position among the same-colour sites of this x-row */
        int second = j & 1;            /* second site of its pair?                            */
        int64_t first_site = site_of(L, x - 2 * second, y, z);
        uint32_t out[4];
        stream_block(s, (uint32_t)first_site, (uint32_t)(s->t & 0xffffffffu), (uint32_t)(s->t >> 32), tag, out);
        s->r_lo[site] = out[2 * second];
        s->r_hi[site] = out[2 * second + 1];
    }
#pragma omp parallel for schedule(static) if (N >= 4096) /* tiny lattices: thread start-up costs more than the work */
    for (int lane = 0; lane < ORACLE_LANES; ++lane) {
        int64_t dE = 0;
        if (s->order == 0) { /* ascending site index */
            for (int z = 0; z < L; ++z)
                for (int y = 0; y < L; ++y)
                    for (int x = 0; x < L; ++x)
                        if (((x + y + z) & 1) == parity) dE += metropolis_trial(s, lane, x, y, z);
        } else { /* any other visiting order of the same colour (pin P9) */
            for (int64_t k = 0; k < N; ++k) {
                int64_t site = visit(s, k);
                int x = (int)(site % L), y = (int)((site / L) % L), z = (int)(site / ((int64_t)L * L));
                if (((x + y + z) & 1) == parity) dE += metropolis_trial(s, lane, x, y, z);
            }
        }
        s->dE_accum[lane] += dE;
    }
}

/* One sweep = "white fields" (parity 0, C-S2) then the other half = one time step. */
void oracle_sweep(oracle_sim *s, uint64_t n)
{
    for (uint64_t i = 0; i < n; ++i) {
        oracle_half_sweep(s, 0);
        oracle_half_sweep(s, 1);
        s->t += 1;
    }
}

/* ------------------------------------------------------------------------------------
 * Observables (C-A10): signed integer sums, per sample.
 * ---------------------------------------------------------------------------------- */

/* E_b = H(S) = - sum_<ij> J_ij S_i S_j over the 3N forward bonds (Eq. 1). */
void oracle_energy(const oracle_sim *s, int64_t E[ORACLE_LANES])
{
#pragma omp parallel for schedule(static)
    for (int lane = 0; lane < ORACLE_LANES; ++lane) {
        const int8_t *S = s->S + (int64_t)lane * s->N;
        const int8_t *J = s->J + (int64_t)lane * 3 * s->N;
        int64_t e = 0;
        for (int d = 0; d < 3; ++d)
            for (int64_t site = 0; site < s->N; ++site)
                e -= J[(int64_t)d * s->N + site] * S[site] * S[oracle_neighbour(s->L, site, d, +1)];
        E[lane] = e;
    }
}

/* M_b = sum_i S_i (C-S14). */
void oracle_magnetisation(const oracle_sim *s, int64_t M[ORACLE_LANES])
{
    for (int lane = 0; lane < ORACLE_LANES; ++lane) {
        int64_t m = 0;
        for (int64_t site = 0; site < s->N; ++site) m += s->S[(int64_t)lane * s->N + site];
        M[lane] = m;
    }
}

/* Keep S(t_w) (the paper stored whole configurations at the measure points). */
int oracle_snapshot(oracle_sim *s, int slot)
{
    if (slot < 0 || slot >= s->n_slots) return 1;
    memcpy(s->snap + (size_t)slot * ORACLE_LANES * s->N, s->S, (size_t)ORACLE_LANES * s->N);
    s->snap_t[slot] = s->t;
    s->snap_set[slot] = 1;
    return 0;
}

/* A_b = N * C(t, t_w) = sum_i S_i(t_w) S_i(t_w + t)  (Eq. 7). */
int oracle_autocorr(const oracle_sim *s, int slot, int64_t A[ORACLE_LANES])
{
    if (slot < 0 || slot >= s->n_slots || !s->snap_set[slot]) return 1;
    const int8_t *W = s->snap + (size_t)slot * ORACLE_LANES * s->N;
    for (int lane = 0; lane < ORACLE_LANES; ++lane) {
        int64_t a = 0;
        for (int64_t site = 0; site < s->N; ++site)
            a += W[(int64_t)lane * s->N + site] * s->S[(int64_t)lane * s->N + site];
        A[lane] = a;
    }
    return 0;
}

/* q_b = sum_i q_i,  q_i = S_i^(a) S_i^(b)  (Eq. 2): replica a = lane b, replica b = lane b+32. */
int oracle_overlap(const oracle_sim *s, int64_t q[32])
{
    if (s->n_replicas != 2) return 1;
    for (int b = 0; b < 32; ++b) {
        int64_t acc = 0;
        for (int64_t site = 0; site < s->N; ++site)
            acc += s->S[(int64_t)b * s->N + site] * s->S[(int64_t)(b + 32) * s->N + site];
        q[b] = acc;
    }
    return 0;
}

/* B_b(d, r) = N * C_4(r e_d, t_w) = sum_i q_i q_{i + r e_d}  (Eq. 3),
 * displacement along lattice axis d ("integer-valued distances ... along the lattice axes", :112; C-S8). */
int oracle_c4_one(const oracle_sim *s, int d, int r, int64_t B[32])
{
    if (s->n_replicas != 2 || d < 0 || d > 2 || r < 0 || r > s->L) return 1;
#pragma omp parallel for schedule(static)
    for (int b = 0; b < 32; ++b) {
        const int8_t *Sa = s->S + (int64_t)b * s->N;
        const int8_t *Sb = s->S + (int64_t)(b + 32) * s->N;
        int64_t acc = 0;
        for (int64_t site = 0; site < s->N; ++site) {
            int64_t other = oracle_shift(s->L, site, d, r); /* i + r e_d */
            int qi = Sa[site] * Sb[site];
            int qj = Sa[other] * Sb[other];
            acc += qi * qj;
        }
        B[b] = acc;
    }
    return 0;
}

/* All r = 0..r_max along the three axes: B[(d*(r_max+1) + r)*32 + b]. */
int oracle_c4(const oracle_sim *s, int r_max, int64_t *B)
{
    if (s->n_replicas != 2 || r_max < 0 || r_max > s->L / 2) return 1;
    for (int d = 0; d < 3; ++d)
        for (int r = 0; r <= r_max; ++r)
            if (oracle_c4_one(s, d, r, B + ((int64_t)d * (r_max + 1) + r) * 32)) return 1;
    return 0;
}

/* ------------------------------------------------------------------------------------
 * Full-vector four-point correlation.  Eq. 3: "With
 * i + r we denote a spin which has a spacial distance r from spin i" -- reading C-S8v: r is
 * any lattice vector (dx, dy, dz), periodic; the axis values above are the special case
 * the paper prefers for its fits, the full set is its "all r >= 3" reference (:112) and the
 * merged points of Fig. 2.
 *   B_b(r) = sum_i q_i q_{i+r},  q_i = S_i^(a) S_i^(b).
 * ---------------------------------------------------------------------------------- */
int oracle_c4_vector(const oracle_sim *s, int dx, int dy, int dz, int64_t B[32])
{
    if (s->n_replicas != 2) return 1;
    const int L = s->L;
#pragma omp parallel for schedule(static)
    for (int b = 0; b < 32; ++b) {
        const int8_t *Sa = s->S + (int64_t)b * s->N;
        const int8_t *Sb = s->S + (int64_t)(b + 32) * s->N;
        int64_t acc = 0;
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    int64_t i = site_of(L, x, y, z);
                    int64_t j = site_of(L, wrap(x + dx, L), wrap(y + dy, L), wrap(z + dz, L));
                    acc += (Sa[i] * Sb[i]) * (Sa[j] * Sb[j]);
                }
        B[b] = acc;
    }
    return 0;
}

/* Shell sums: every vector with |dx|, |dy|, |dz| <= r_max, collected by squared length
 * d2 = dx^2 + dy^2 + dz^2 = 0 .. 3 r_max^2:
 *   S[d2*32 + b] = sum_{|r|^2 = d2} B_b(r),   mult[d2] = number of those vectors
 * so that C_4(|r| = sqrt(d2)) = S / (mult N) is the average over all directions (Fig. 2).
 * No symmetry is used: r and -r are both visited.  r_max = L/2 visits +L/2 and -L/2 (the
 * same displacement on the torus) as two vectors; the average is unaffected. */
int oracle_c4_shells(const oracle_sim *s, int r_max, int64_t *S, int64_t *mult)
{
    if (s->n_replicas != 2 || r_max < 0 || r_max > s->L / 2) return 1;
    const int n_bins = 3 * r_max * r_max + 1;
    memset(S, 0, sizeof(int64_t) * 32 * (size_t)n_bins);
    memset(mult, 0, sizeof(int64_t) * (size_t)n_bins);
    for (int dz = -r_max; dz <= r_max; ++dz)
        for (int dy = -r_max; dy <= r_max; ++dy)
            for (int dx = -r_max; dx <= r_max; ++dx) {
                int64_t B[32];
                if (oracle_c4_vector(s, dx, dy, dz, B)) return 1;
                int d2 = dx * dx + dy * dy + dz * dz;
                for (int b = 0; b < 32; ++b) S[(int64_t)d2 * 32 + b] += B[b];
                mult[d2] += 1;
            }
    return 0;
}

/* ------------------------------------------------------------------------------------
 * Canonical packed I/O (C-A2): word[site] bit b = 1 <-> S_b = -1;
 * bond word[d*N + site] bit b = 1 <-> J_b = -1.  This is the exchange format of the
 * library boundary (include/ea.h), written out here independently.
 * ---------------------------------------------------------------------------------- */
void oracle_get_spins(const oracle_sim *s, uint64_t *words)
{
    for (int64_t site = 0; site < s->N; ++site) {
        uint64_t w = 0;
        for (int lane = 0; lane < ORACLE_LANES; ++lane)
            if (s->S[(int64_t)lane * s->N + site] < 0) w |= (uint64_t)1 << lane;
        words[site] = w;
    }
}

void oracle_set_spins(oracle_sim *s, const uint64_t *words)
{
    for (int64_t site = 0; site < s->N; ++site)
        for (int lane = 0; lane < ORACLE_LANES; ++lane)
            s->S[(int64_t)lane * s->N + site] = ((words[site] >> lane) & 1u) ? -1 : +1;
}

void oracle_get_bonds(const oracle_sim *s, uint64_t *words)
{
    for (int d = 0; d < 3; ++d)
        for (int64_t site = 0; site < s->N; ++site) {
            uint64_t w = 0;
            for (int lane = 0; lane < ORACLE_LANES; ++lane)
                if (s->J[((int64_t)lane * 3 + d) * s->N + site] < 0) w |= (uint64_t)1 << lane;
            words[(int64_t)d * s->N + site] = w;
        }
}

void oracle_set_bonds(oracle_sim *s, const uint64_t *words)
{
    for (int d = 0; d < 3; ++d)
        for (int64_t site = 0; site < s->N; ++site)
            for (int lane = 0; lane < ORACLE_LANES; ++lane)
                s->J[((int64_t)lane * 3 + d) * s->N + site] =
                    ((words[(int64_t)d * s->N + site] >> lane) & 1u) ? -1 : +1;
}

void oracle_get_snapshot(const oracle_sim *s, int slot, uint64_t *words)
{
    const int8_t *W = s->snap + (size_t)slot * ORACLE_LANES * s->N;
    for (int64_t site = 0; site < s->N; ++site) {
        uint64_t w = 0;
        for (int lane = 0; lane < ORACLE_LANES; ++lane)
            if (W[(int64_t)lane * s->N + site] < 0) w |= (uint64_t)1 << lane;
        words[site] = w;
    }
}
