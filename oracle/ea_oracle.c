/*
 * ea_oracle.c — plain, slow, sequential CPU oracle for the Monte Carlo hot path of
 * arXiv:1403.4560 (3D Edwards-Anderson spin glass in a field).
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.  It shares no code, header, table
 * generator or constant file with the CUDA path under paper_1403_4560_b200/csrc/.
 *
 * One oracle instance simulates ONE disorder sample `sample` with all of its
 * n_replicas x n_temps systems, one spin per `int`, sequential in-place updates.
 * Citations are "PAPER.md:<line>" (the paper text) or "DESIGN.md R<n>" (a reading of a
 * point the paper leaves open; every reading is listed in DESIGN.md §3).
 *
 * Followed step by step:
 *   Eq. 1  H = -sum_<ij> J_ij S_i S_j - h sum_i S_i
 *   bimodal J = +-1 equiprobable, periodic L^3 simple cubic
 *   overlap q(k) = (1/N) sum_j S^a_j S^b_j exp(i k.r_j)       PAPER.md:43 (Eq. 2)
 *   parallel tempering over N_T temperatures
 *   k_min=(2pi/L,0,0); k2=(2pi/L,2pi/L,0); point-group avg
 *
 * Pins (tests/test_oracle_*.py): Philox known answers; threshold-table worked example;
 * exact enumeration on 2x2x2 and 2x2x3; tracked energy == recomputed energy; gauge
 * covariance; (h,S)->(-h,-S) covariance; beta=0 and beta=inf limits; stripe closed form
 * and Parseval for q(k); dexp/dlog/dsincos vs libm; Gaussian moments; the draw <-> site
 * keying of sweep_once and the PT draw keying followed by hand (tests/test_oracle_keying.py).
 * Parity unpinned (conventions, not results): choice of random initial state, PT pair
 * schedule, measurement cadence — see DESIGN.md §3.
 *
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fno-fast-math -shared -fPIC (oracle/build.py)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define EA_PI 3.14159265358979323846
#define EA_PMJ 0
#define EA_GAUSS 1
#define EA_NK 12      /* non-zero wave vectors, R8 */
#define EA_REC 25     /* 1 + 2*EA_NK doubles per (slot, pair) measurement record */
#define EA_NMOM 66    /* accumulator doubles per slot, R9 */

/* ------------------------------------------------------------------ Philox4x32-10 */
/* Salmon et al., "Parallel random numbers: as easy as 1, 2, 3" (SC'11): 10 rounds,
 * multipliers 0xD2511F53 / 0xCD9E8D57, Weyl key increments 0x9E3779B9 / 0xBB67AE85. */
void ea_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Counter layout, R5/R6: c0=index, c1=time, c2=packed word w (or sample s),
 * c3 = (domain<<24)|(replica<<16)|slot; domain 1 couplings, 2 initial spins, 3 sweep, 4 PT.
 * key = (seed low 32 bits, seed high 32 bits). */
static void draw4(const uint32_t key[2], uint32_t index, uint32_t time, uint32_t word,
                  uint32_t domain, uint32_t replica, uint32_t slot, uint32_t out[4])
{
    uint32_t ctr[4];
    ctr[0] = index; ctr[1] = time; ctr[2] = word;
    ctr[3] = (domain << 24) | (replica << 16) | slot;
    ea_philox4x32_10(ctr, key, out);
}

/* ------------------------------------------------ deterministic elementary functions */
/* DESIGN.md R12: written sequences of IEEE-754 operations (every multiply and add rounded
 * separately; this file is compiled with -ffp-contract=off).  They define the method's
 * exponentials / Box-Muller transcendentals so that a second implementation can reproduce
 * them bit for bit; accuracy vs libm is pinned in tests/test_oracle_rng_math.py. */

/* 2^32 * exp(-y) rounded down, for y > 0; table[i] = exp(-i/256) from libm. */
static uint64_t dexp64_tab(const double *table, double y)
{
    if (!(y < 22.5)) return 0;                 /* 2^32 e^-22.5 < 1 */
    int i = (int)(y * 256.0);
    double f = y - (double)i * 0.00390625;     /* exact */
    double z = -f;
    double g = 0x1.6c16c16c16c17p-10;          /* 1/720 */
    g = g * z; g = g + 0x1.1111111111111p-7;   /* 1/120 */
    g = g * z; g = g + 0x1.5555555555555p-5;   /* 1/24 */
    g = g * z; g = g + 0x1.5555555555555p-3;   /* 1/6 */
    g = g * z; g = g + 0x1.0000000000000p-1;   /* 1/2 */
    g = g * z; g = g + 1.0;
    g = g * z; g = g + 1.0;
    double p = table[i] * g;
    return (uint64_t)(p * 4294967296.0);
}

/* fp32 analogue: step 1/64, degree 4; table[i] = (float)exp(-i/64). */
static uint64_t dexp32_tab(const float *table, float y)
{
    if (!(y < 22.5f)) return 0;
    int i = (int)(y * 64.0f);
    float f = y - (float)i * 0.015625f;        /* exact */
    float z = -f;
    float g = 0x1.555556p-5f;                  /* 1/24 */
    g = g * z; g = g + 0x1.555556p-3f;         /* 1/6 */
    g = g * z; g = g + 0.5f;
    g = g * z; g = g + 1.0f;
    g = g * z; g = g + 1.0f;
    float p = table[i] * g;
    return (uint64_t)(p * 4294967296.0f);
}

#define DEXP64_N 5761   /* i <= floor(22.5*256) = 5760 */
#define DEXP32_N 1441   /* i <= floor(22.5*64)  = 1440 */

static void fill_dexp_tables(double *t64, float *t32)
{
    for (int i = 0; i < DEXP64_N; ++i) t64[i] = exp(-(double)i / 256.0);
    for (int i = 0; i < DEXP32_N; ++i) t32[i] = (float)exp(-(double)i / 64.0);
}

/* natural log for 0 < u < 1 (normal doubles): u = m 2^e, m in (sqrt(1/2), sqrt 2],
 * ln m = 2 z (1 + w/3 + w^2/5 + ... + w^11/23), z = (m-1)/(m+1), w = z^2. */
static double dlog(double u)
{
    uint64_t bits;
    memcpy(&bits, &u, 8);
    int e = (int)((bits >> 52) & 0x7ff) - 1023;
    bits = (bits & 0x000fffffffffffffULL) | 0x3ff0000000000000ULL;
    double m;
    memcpy(&m, &bits, 8);                      /* m in [1,2) */
    if (m > 0x1.6a09e667f3bcdp+0) { m = m * 0.5; e = e + 1; }
    double z = (m - 1.0) / (m + 1.0);
    double w = z * z;
    double s = 0x1.642c8590b2164p-5;           /* 1/23 */
    s = s * w; s = s + 0x1.8618618618618p-5;   /* 1/21 */
    s = s * w; s = s + 0x1.af286bca1af28p-5;   /* 1/19 */
    s = s * w; s = s + 0x1.e1e1e1e1e1e1ep-5;   /* 1/17 */
    s = s * w; s = s + 0x1.1111111111111p-4;   /* 1/15 */
    s = s * w; s = s + 0x1.3b13b13b13b14p-4;   /* 1/13 */
    s = s * w; s = s + 0x1.745d1745d1746p-4;   /* 1/11 */
    s = s * w; s = s + 0x1.c71c71c71c71cp-4;   /* 1/9 */
    s = s * w; s = s + 0x1.2492492492492p-3;   /* 1/7 */
    s = s * w; s = s + 0x1.999999999999ap-3;   /* 1/5 */
    s = s * w; s = s + 0x1.5555555555555p-2;   /* 1/3 */
    s = s * w; s = s + 1.0;
    double lnm = (2.0 * z) * s;
    double le = (double)e * 0x1.62e42fefa39efp-1;  /* e ln 2 */
    return le + lnm;
}

/* cos(2 pi u), sin(2 pi u) for 0 <= u < 1: nearest quadrant kk, r = u - kk/4 in
 * [-1/8, 1/8], x = 2 pi r, Taylor to x^18 / x^17, exact quadrant rotation. */
static void dsincos2pi(double u, double *c_out, double *s_out)
{
    int kk = (int)(u * 4.0 + 0.5);             /* 0..4 */
    double r = u - (double)kk * 0.25;          /* exact */
    double x = 0x1.921fb54442d18p+2 * r;
    double x2 = x * x;
    double ps = 0x1.952c77030ad4ap-49;         /* 1/17! */
    ps = ps * x2; ps = ps + -0x1.ae7f3e733b81fp-41;
    ps = ps * x2; ps = ps + 0x1.6124613a86d09p-33;
    ps = ps * x2; ps = ps + -0x1.ae64567f544e4p-26;
    ps = ps * x2; ps = ps + 0x1.71de3a556c734p-19;
    ps = ps * x2; ps = ps + -0x1.a01a01a01a01ap-13;
    ps = ps * x2; ps = ps + 0x1.1111111111111p-7;
    ps = ps * x2; ps = ps + -0x1.5555555555555p-3;
    ps = ps * x2; ps = ps + 1.0;
    double sn = x * ps;
    double pc = -0x1.6827863b97d97p-53;        /* -1/18! */
    pc = pc * x2; pc = pc + 0x1.ae7f3e733b81fp-45;
    pc = pc * x2; pc = pc + -0x1.93974a8c07c9dp-37;
    pc = pc * x2; pc = pc + 0x1.1eed8eff8d898p-29;
    pc = pc * x2; pc = pc + -0x1.27e4fb7789f5cp-22;
    pc = pc * x2; pc = pc + 0x1.a01a01a01a01ap-16;
    pc = pc * x2; pc = pc + -0x1.6c16c16c16c17p-10;
    pc = pc * x2; pc = pc + 0x1.5555555555555p-5;
    pc = pc * x2; pc = pc + -0x1.0000000000000p-1;
    pc = pc * x2; pc = pc + 1.0;
    double cs = pc;
    switch (kk & 3) {
    case 0: *c_out = cs;  *s_out = sn;  break;
    case 1: *c_out = -sn; *s_out = cs;  break;
    case 2: *c_out = -cs; *s_out = -sn; break;
    default: *c_out = sn; *s_out = -cs; break;
    }
}

/* exported for the pins */
double ea_dlog(double u) { return dlog(u); }
void ea_dsincos2pi(double u, double *c, double *s) { dsincos2pi(u, c, s); }
uint64_t ea_dexp64(double y)
{
    static double t64[DEXP64_N]; static float t32[DEXP32_N]; static int init = 0;
    if (!init) { fill_dexp_tables(t64, t32); init = 1; }
    return dexp64_tab(t64, y);
}
uint64_t ea_dexp32(float y)
{
    static double t64[DEXP64_N]; static float t32[DEXP32_N]; static int init = 0;
    if (!init) { fill_dexp_tables(t64, t32); init = 1; }
    return dexp32_tab(t32, y);
}

/* --------------------------------------------------------------------- the oracle */
typedef struct ea_oracle {
    int Lx, Ly, Lz, N;
    double h;
    int R, NT, kind, sample;
    uint32_t key[2];
    uint32_t word;          /* c2 for sweep / disorder / init draws: sample>>5 (PMJ) or sample (GAUSS) */
    int lane;               /* sample & 31 (PMJ) */
    double *T, *beta;
    float *beta_f;
    uint64_t *thr;          /* [NT][7][2] */
    int *nbr;               /* [N][6]: +x,-x,+y,-y,+z,-z */
    int *colour;            /* [N] */
    int *Jpm;               /* [3][N], +-1 */
    float *Jg;              /* [3][N] */
    int64_t *Jfix;          /* [3][N] */
    int *S;                 /* [R][NT][N] */
    int64_t *U;             /* [R][NT] unsatisfied bonds (PMJ) or E_fix (GAUSS) */
    int32_t *M;             /* [R][NT] */
    uint64_t sweeps, exchanges;
    int64_t n_meas;
    double *acc;            /* [NT][EA_NMOM] */
    double *ck, *sk;        /* [EA_NK][N] cos/sin(k.r) */
    double t64[DEXP64_N];
    float t32[DEXP32_N];
    uint64_t n_pt_prop, n_pt_acc;
    /* diagnostics ("logarithm binning test", "distribution of the overlap parameter") */
    int pq_bins;            /* 0 = off */
    uint64_t *pq;           /* [NT][pq_bins] counts of the overlap q_ab(0), all pairs, all measurements */
    int n_windows;          /* 0 = off */
    double *accw;           /* [n_windows][NT][EA_NMOM]: the accumulators of R9 per window [2^k, 2^(k+1)) of the sweep counter */
    int64_t *n_meas_w;      /* [n_windows] */
} ea_oracle;

static const int KVEC[EA_NK][3] = {      /* in units of (2pi/Lx, 2pi/Ly, 2pi/Lz); R8 */
    {1, 0, 0}, {0, 1, 0}, {0, 0, 1},     /* k1 = k_min and permutations */
    {2, 0, 0}, {0, 2, 0}, {0, 0, 2},     /* BASELINE.json's k2 = (4pi/L,0,0)                 */
    {1, 1, 0}, {1, -1, 0}, {1, 0, 1}, {1, 0, -1}, {0, 1, 1}, {0, 1, -1}  /* paper's k2 */
};

static int *Sys(ea_oracle *o, int a, int t) { return o->S + ((size_t)a * o->NT + t) * o->N; }

/* J_(i,d) as a double (only for literal energy sums) */
static double Jval(const ea_oracle *o, int d, int i)
{
    return o->kind == EA_PMJ ? (double)o->Jpm[d * o->N + i] : (double)o->Jg[d * o->N + i];
}

/* recompute (U, M) of one system from scratch: Eq. 1 */
static void recompute(const ea_oracle *o, const int *S, int64_t *U, int32_t *M)
{
    int64_t u = 0; int32_t m = 0;
    for (int i = 0; i < o->N; ++i) {
        m += S[i];
        for (int d = 0; d < 3; ++d) {
            int j = o->nbr[i * 6 + 2 * d];
            if (o->kind == EA_PMJ) {
                if (o->Jpm[d * o->N + i] * S[i] * S[j] == -1) u += 1;
            } else {
                u -= o->Jfix[d * o->N + i] * (int64_t)(S[i] * S[j]);
            }
        }
    }
    *U = u; *M = m;
}

void ea_destroy(ea_oracle *o)
{
    if (!o) return;
    free(o->T); free(o->beta); free(o->beta_f); free(o->thr); free(o->nbr); free(o->colour);
    free(o->Jpm); free(o->Jg); free(o->Jfix); free(o->S); free(o->U); free(o->M);
    free(o->acc); free(o->ck); free(o->sk);
    free(o->pq); free(o->accw); free(o->n_meas_w);
    free(o);
}

ea_oracle *ea_create(int Lx, int Ly, int Lz, double h, int n_replicas, int n_temps,
                     const double *temps, int kind, uint64_t seed, int sample)
{
    if (Lx < 2 || Ly < 2 || Lz < 2 || (Lx & 1) || n_replicas < 1 || n_replicas > 4 || n_temps < 1 || !temps) return NULL;
    if (kind != EA_PMJ && kind != EA_GAUSS) return NULL;
    ea_oracle *o = (ea_oracle *)calloc(1, sizeof(ea_oracle));
    if (!o) return NULL;
    const int N = Lx * Ly * Lz;
    o->Lx = Lx; o->Ly = Ly; o->Lz = Lz; o->N = N; o->h = h;
    o->R = n_replicas; o->NT = n_temps; o->kind = kind; o->sample = sample;
    o->key[0] = (uint32_t)seed; o->key[1] = (uint32_t)(seed >> 32);
    o->word = kind == EA_PMJ ? (uint32_t)(sample >> 5) : (uint32_t)sample;
    o->lane = sample & 31;
    fill_dexp_tables(o->t64, o->t32);

    o->T = (double *)malloc(sizeof(double) * n_temps);
    o->beta = (double *)malloc(sizeof(double) * n_temps);
    o->beta_f = (float *)malloc(sizeof(float) * n_temps);
    o->thr = (uint64_t *)malloc(sizeof(uint64_t) * n_temps * 14);
    o->nbr = (int *)malloc(sizeof(int) * N * 6);
    o->colour = (int *)malloc(sizeof(int) * N);
    o->Jpm = (int *)calloc((size_t)3 * N, sizeof(int));
    o->Jg = (float *)calloc((size_t)3 * N, sizeof(float));
    o->Jfix = (int64_t *)calloc((size_t)3 * N, sizeof(int64_t));
    o->S = (int *)malloc(sizeof(int) * (size_t)n_replicas * n_temps * N);
    o->U = (int64_t *)malloc(sizeof(int64_t) * n_replicas * n_temps);
    o->M = (int32_t *)malloc(sizeof(int32_t) * n_replicas * n_temps);
    o->acc = (double *)calloc((size_t)n_temps * EA_NMOM, sizeof(double));
    o->ck = (double *)malloc(sizeof(double) * EA_NK * N);
    o->sk = (double *)malloc(sizeof(double) * EA_NK * N);

    /* lattice: site i = x + Lx*(y + Ly*z), periodic neighbours */
    for (int z = 0; z < Lz; ++z)
        for (int y = 0; y < Ly; ++y)
            for (int x = 0; x < Lx; ++x) {
                int i = x + Lx * (y + Ly * z);
                o->colour[i] = (x + y + z) & 1;
                o->nbr[i * 6 + 0] = ((x + 1) % Lx) + Lx * (y + Ly * z);
                o->nbr[i * 6 + 1] = ((x + Lx - 1) % Lx) + Lx * (y + Ly * z);
                o->nbr[i * 6 + 2] = x + Lx * (((y + 1) % Ly) + Ly * z);
                o->nbr[i * 6 + 3] = x + Lx * (((y + Ly - 1) % Ly) + Ly * z);
                o->nbr[i * 6 + 4] = x + Lx * (y + Ly * ((z + 1) % Lz));
                o->nbr[i * 6 + 5] = x + Lx * (y + Ly * ((z + Lz - 1) % Lz));
                for (int k = 0; k < EA_NK; ++k) {      /* phase of Eq. 2, +i, r from 0: DESIGN.md R7 */
                    double ph = 2.0 * EA_PI * ((double)(KVEC[k][0] * x) / (double)Lx +
                                              (double)(KVEC[k][1] * y) / (double)Ly +
                                              (double)(KVEC[k][2] * z) / (double)Lz);
                    o->ck[k * N + i] = cos(ph);
                    o->sk[k * N + i] = sin(ph);
                }
            }

    /* temperatures -> beta, Metropolis thresholds                     DESIGN.md R2, R4 */
    for (int t = 0; t < n_temps; ++t) {
        o->T[t] = temps[t];
        o->beta[t] = 1.0 / temps[t];
        o->beta_f[t] = (float)(1.0 / temps[t]);
        for (int nu = 0; nu <= 6; ++nu)
            for (int a = 0; a < 2; ++a) {
                double dE = (double)(12 - 4 * nu) + (a ? 2.0 * fabs(h) : -(2.0 * fabs(h)));
                uint64_t th;
                if (dE <= 0.0) th = 4294967296ULL;
                else {
                    double p = floor(exp(-o->beta[t] * dE) * 4294967296.0);
                    th = p >= 4294967296.0 ? 4294967296ULL : (uint64_t)p;
                }
                o->thr[(t * 7 + nu) * 2 + a] = th;
            }
    }

    /* disorder                                                         PAPER.md:39; R5 */
    for (int i = 0; i < N; ++i) {
        uint32_t r[4];
        draw4(o->key, (uint32_t)i, 0, o->word, 1, 0, 0, r);
        if (kind == EA_PMJ) {
            for (int d = 0; d < 3; ++d)
                o->Jpm[d * N + i] = ((r[d] >> o->lane) & 1u) ? -1 : +1;
        } else {
            double u[4], c, s;
            for (int k = 0; k < 4; ++k) u[k] = ((double)r[k] + 0.5) * 0x1p-32;
            double rho = sqrt(-2.0 * dlog(u[0]));
            dsincos2pi(u[1], &c, &s);
            o->Jg[0 * N + i] = (float)(rho * c);
            o->Jg[1 * N + i] = (float)(rho * s);
            rho = sqrt(-2.0 * dlog(u[2]));
            dsincos2pi(u[3], &c, &s);
            o->Jg[2 * N + i] = (float)(rho * c);
            for (int d = 0; d < 3; ++d)           /* DESIGN.md R14: fixed-point image, exact */
                o->Jfix[d * N + i] = (int64_t)((double)o->Jg[d * N + i] * 4294967296.0);
        }
    }

    /* initial spins: random                                            DESIGN.md R5 */
    for (int a = 0; a < n_replicas; ++a)
        for (int t = 0; t < n_temps; ++t) {
            int *S = Sys(o, a, t);
            for (int i = 0; i < N; ++i) {
                uint32_t r[4];
                draw4(o->key, (uint32_t)i, 0, o->word, 2, (uint32_t)a, (uint32_t)t, r);
                uint32_t bit = kind == EA_PMJ ? ((r[0] >> o->lane) & 1u) : (r[0] & 1u);
                S[i] = bit ? +1 : -1;
            }
            recompute(o, S, &o->U[a * n_temps + t], &o->M[a * n_temps + t]);
        }
    return o;
}

/* one checkerboard Metropolis sweep of every system                    DESIGN.md R2, R3, R6 */
static void sweep_once(ea_oracle *o)
{
    const int N = o->N;
    const uint32_t k = (uint32_t)o->sweeps;
    const float hf = (float)o->h;
    for (int a = 0; a < o->R; ++a)
        for (int t = 0; t < o->NT; ++t) {
            int *S = Sys(o, a, t);
            int64_t *U = &o->U[a * o->NT + t];
            int32_t *M = &o->M[a * o->NT + t];
            for (int c = 0; c < 2; ++c) {
                uint32_t n = 0;                   /* rank of the site inside its colour class */
                uint32_t r4[4] = {0, 0, 0, 0};
                for (int i = 0; i < N; ++i) {
                    if (o->colour[i] != c) continue;
                    if ((n & 3u) == 0)
                        draw4(o->key, n >> 2, 2u * k + (uint32_t)c, o->word, 3, (uint32_t)a, (uint32_t)t, r4);
                    const uint32_t r = r4[n & 3u];
                    ++n;
                    const int *nb = &o->nbr[i * 6];
                    int flip;
                    if (o->kind == EA_PMJ) {
                        int nu = 0;
                        for (int d = 0; d < 3; ++d) {
                            int jp = nb[2 * d], jm = nb[2 * d + 1];
                            if (o->Jpm[d * N + i] * S[i] * S[jp] == -1) ++nu;   /* bond (i,d)  */
                            if (o->Jpm[d * N + jm] * S[i] * S[jm] == -1) ++nu;  /* bond (jm,d) */
                        }
                        int al = (o->h < 0.0 ? -S[i] : S[i]) == 1;               /* field alignment */
                        flip = (uint64_t)r < o->thr[(t * 7 + nu) * 2 + al];
                        if (flip) { *U += 6 - 2 * nu; *M -= 2 * S[i]; S[i] = -S[i]; }
                    } else {                                                     /* DESIGN.md R13 */
                        float hl = 0.0f;
                        for (int d = 0; d < 3; ++d) {
                            int jp = nb[2 * d], jm = nb[2 * d + 1];
                            float Jp = o->Jg[d * N + i], Jm = o->Jg[d * N + jm];
                            hl = hl + (S[jp] > 0 ? Jp : -Jp);
                            hl = hl + (S[jm] > 0 ? Jm : -Jm);
                        }
                        hl = hl + hf;
                        float dE = S[i] > 0 ? 2.0f * hl : -(2.0f * hl);
                        if (dE <= 0.0f) flip = 1;
                        else flip = (uint64_t)r < dexp32_tab(o->t32, o->beta_f[t] * dE);
                        if (flip) {
                            int64_t de = 0;       /* exact fixed-point energy change */
                            for (int d = 0; d < 3; ++d) {
                                int jp = nb[2 * d], jm = nb[2 * d + 1];
                                de += 2 * o->Jfix[d * N + i] * (int64_t)(S[i] * S[jp]);
                                de += 2 * o->Jfix[d * N + jm] * (int64_t)(S[i] * S[jm]);
                            }
                            *U += de; *M -= 2 * S[i]; S[i] = -S[i];
                        }
                    }
                }
            }
        }
    o->sweeps += 1;
}

void ea_sweep(ea_oracle *o, int n) { for (int s = 0; s < n; ++s) sweep_once(o); }

/* total energy of slot (a,t) as the PT step sees it                    DESIGN.md R12, R14 */
static double energy_pt(const ea_oracle *o, int a, int t)
{
    int64_t U = o->U[a * o->NT + t];
    double hm = o->h * (double)o->M[a * o->NT + t];
    if (o->kind == EA_PMJ) return (double)(2 * U - 3 * (int64_t)o->N) - hm;
    return (double)U * 0x1p-32 - hm;
}

/* one parallel-tempering exchange step                                 PAPER.md:66; R12 */
void ea_pt_exchange(ea_oracle *o)
{
    const uint32_t e = (uint32_t)o->exchanges;
    int *tmp = (int *)malloc(sizeof(int) * o->N);
    for (int a = 0; a < o->R; ++a)
        for (int t = (int)(e & 1u); t + 1 < o->NT; t += 2) {
            double Et = energy_pt(o, a, t), Eu = energy_pt(o, a, t + 1);
            double x = (o->beta[t] - o->beta[t + 1]) * (Et - Eu);
            uint32_t r[4];
            draw4(o->key, 0, e, (uint32_t)o->sample, 4, (uint32_t)a, (uint32_t)t, r);
            int accept = (x >= 0.0) || ((uint64_t)r[0] < dexp64_tab(o->t64, -x));
            o->n_pt_prop += 1;
            if (accept) {
                o->n_pt_acc += 1;
                int *A = Sys(o, a, t), *B = Sys(o, a, t + 1);
                memcpy(tmp, A, sizeof(int) * o->N);
                memcpy(A, B, sizeof(int) * o->N);
                memcpy(B, tmp, sizeof(int) * o->N);
                int64_t u = o->U[a * o->NT + t]; o->U[a * o->NT + t] = o->U[a * o->NT + t + 1]; o->U[a * o->NT + t + 1] = u;
                int32_t m = o->M[a * o->NT + t]; o->M[a * o->NT + t] = o->M[a * o->NT + t + 1]; o->M[a * o->NT + t + 1] = m;
            }
        }
    free(tmp);
    o->exchanges += 1;
}

int ea_n_pairs(const ea_oracle *o) { return o->R * (o->R - 1) / 2; }

/* accumulators, R9 (one measurement of one slot added to A[EA_NMOM]):
 * [0..3]  sum over pairs of q, q^2, q^3, q^4  (q = q_ab(0))           -> Eq. 3
 * [4+5k+0..2] sum over pairs of Re q(Kk), Im q(Kk), |q(Kk)|^2          -> Eq. 4
 * [4+5k+3] sum over the unordered couples of pairs sharing exactly one replica of Re(q_p conj q_p')
 * [4+5k+4] sum over the disjoint pair-couples of Re(q_p conj q_p')
 * [64],[65] the same two cross sums for k = 0 */
static void add_moments(double *A, double rec[6][EA_REC], const int *pa, const int *pb, int P)
{
    for (int q = 0; q < P; ++q) {
        double v = rec[q][0];
        A[0] += v; A[1] += v * v; A[2] += v * v * v; A[3] += (v * v) * (v * v);
        for (int k = 0; k < EA_NK; ++k) {
            double re = rec[q][1 + 2 * k], im = rec[q][2 + 2 * k];
            A[4 + 5 * k + 0] += re;
            A[4 + 5 * k + 1] += im;
            A[4 + 5 * k + 2] += re * re + im * im;
        }
    }
    for (int q = 0; q < P; ++q)
        for (int q2 = q + 1; q2 < P; ++q2) {
            int shared = (pa[q] == pa[q2]) + (pa[q] == pb[q2]) + (pb[q] == pa[q2]) + (pb[q] == pb[q2]);
            int slot = shared == 1 ? 3 : 4;
            A[slot == 3 ? 64 : 65] += rec[q][0] * rec[q2][0];
            for (int k = 0; k < EA_NK; ++k)
                A[4 + 5 * k + slot] += rec[q][1 + 2 * k] * rec[q2][1 + 2 * k] +
                                       rec[q][2 + 2 * k] * rec[q2][2 + 2 * k];
        }
}

/* overlaps of all replica pairs at every slot: literal Eq. 2
 * out (may be NULL): [NT][n_pairs][25] = q(0), Re q(K0), Im q(K0), ..., Re q(K11), Im q(K11);
 * pair order (0,1),(0,2),(0,3),(1,2),(1,3),(2,3).  Always adds to the accumulators (R9). */
void ea_measure(ea_oracle *o, double *out)
{
    const int N = o->N, R = o->R, P = ea_n_pairs(o);
    double rec[6][EA_REC];
    int pa[6], pb[6];
    for (int t = 0; t < o->NT; ++t) {
        int p = 0;
        for (int a = 0; a < R; ++a)
            for (int b = a + 1; b < R; ++b) {
                if (p >= 6) break;
                const int *Sa = Sys(o, a, t), *Sb = Sys(o, b, t);
                double q0 = 0.0;
                for (int j = 0; j < N; ++j) q0 += (double)(Sa[j] * Sb[j]);
                rec[p][0] = q0 / (double)N;
                for (int k = 0; k < EA_NK; ++k) {
                    double re = 0.0, im = 0.0;
                    for (int j = 0; j < N; ++j) {
                        double sg = (double)(Sa[j] * Sb[j]);
                        re += sg * o->ck[k * N + j];
                        im += sg * o->sk[k * N + j];
                    }
                    rec[p][1 + 2 * k] = re / (double)N;
                    rec[p][2 + 2 * k] = im / (double)N;
                }
                pa[p] = a; pb[p] = b;
                ++p;
            }
        if (out)
            for (int q = 0; q < P; ++q)
                memcpy(out + ((size_t)t * P + q) * EA_REC, rec[q], sizeof(double) * EA_REC);

        /* P(q): the integer overlap Q = sum_j S^a_j S^b_j = N q_ab(0) takes the N + 1 values -N, -N+2, ..., N;
         * idx = (Q + N)/2 = number of agreeing sites in 0..N; bin = floor(idx * pq_bins / (N + 1)) */
        if (o->pq_bins > 0) {
            int pp = 0;
            for (int a = 0; a < R; ++a)
                for (int b = a + 1; b < R; ++b) {
                    if (pp >= 6) break;
                    const int *Sa = Sys(o, a, t), *Sb = Sys(o, b, t);
                    int64_t agree = 0;
                    for (int j = 0; j < N; ++j) if (Sa[j] == Sb[j]) ++agree;
                    o->pq[(size_t)t * o->pq_bins + (size_t)((agree * (int64_t)o->pq_bins) / ((int64_t)N + 1))] += 1;
                    ++pp;
                }
        }
        /* logarithmic binning: a measurement taken when the sweep counter is s >= 1 also goes to the
         * window k = min(floor(log2 s), n_windows - 1), i.e. s in [2^k, 2^(k+1)) */
        double *AW = NULL;
        if (o->n_windows > 0 && o->sweeps >= 1) {
            int k = 0;
            while ((o->sweeps >> (k + 1)) != 0) ++k;
            if (k > o->n_windows - 1) k = o->n_windows - 1;
            AW = o->accw + ((size_t)k * o->NT + t) * EA_NMOM;
            if (t == 0) o->n_meas_w[k] += 1;
        }
        add_moments(o->acc + (size_t)t * EA_NMOM, rec, pa, pb, P);
        if (AW) add_moments(AW, rec, pa, pb, P);
    }
    o->n_meas += 1;
}

/* driver loop: sweep -> PT (if due) -> measure (if due)               DESIGN.md R16 */
void ea_run(ea_oracle *o, int n_sweeps, int pt_every, int meas_every)
{
    for (int s = 1; s <= n_sweeps; ++s) {
        sweep_once(o);
        if (pt_every > 0 && (o->sweeps % (uint64_t)pt_every) == 0) ea_pt_exchange(o);
        if (meas_every > 0 && (o->sweeps % (uint64_t)meas_every) == 0) ea_measure(o, NULL);
    }
}

/* ------------------------------------------------------------------------ getters */
void ea_get_spins(const ea_oracle *o, int8_t *out)          /* [R][NT][N] */
{
    size_t n = (size_t)o->R * o->NT * o->N;
    for (size_t i = 0; i < n; ++i) out[i] = (int8_t)o->S[i];
}
void ea_set_spins(ea_oracle *o, const int8_t *in)
{
    size_t n = (size_t)o->R * o->NT * o->N;
    for (size_t i = 0; i < n; ++i) o->S[i] = in[i] > 0 ? 1 : -1;
    for (int a = 0; a < o->R; ++a)
        for (int t = 0; t < o->NT; ++t)
            recompute(o, Sys(o, a, t), &o->U[a * o->NT + t], &o->M[a * o->NT + t]);
}
void ea_get_couplings(const ea_oracle *o, float *out)       /* [3][N] */
{
    for (int i = 0; i < 3 * o->N; ++i)
        out[i] = o->kind == EA_PMJ ? (float)o->Jpm[i] : o->Jg[i];
}
/* test hook for the gauge-covariance pin: overwrite the +-1 couplings */
void ea_set_couplings_pm(ea_oracle *o, const int8_t *in)
{
    for (int i = 0; i < 3 * o->N; ++i) o->Jpm[i] = in[i] > 0 ? 1 : -1;
    for (int a = 0; a < o->R; ++a)
        for (int t = 0; t < o->NT; ++t)
            recompute(o, Sys(o, a, t), &o->U[a * o->NT + t], &o->M[a * o->NT + t]);
}
void ea_get_energies(const ea_oracle *o, int64_t *U, int32_t *M)   /* tracked, [R][NT] */
{
    for (int i = 0; i < o->R * o->NT; ++i) { if (U) U[i] = o->U[i]; if (M) M[i] = o->M[i]; }
}
void ea_recompute_energies(const ea_oracle *o, int64_t *U, int32_t *M)
{
    for (int a = 0; a < o->R; ++a)
        for (int t = 0; t < o->NT; ++t)
            recompute(o, o->S + ((size_t)a * o->NT + t) * o->N, &U[a * o->NT + t], &M[a * o->NT + t]);
}
/* literal Eq. 1 in double for one system */
double ea_hamiltonian(const ea_oracle *o, int a, int t)
{
    const int *S = o->S + ((size_t)a * o->NT + t) * o->N;
    double E = 0.0;
    for (int i = 0; i < o->N; ++i) {
        for (int d = 0; d < 3; ++d)
            E -= Jval(o, d, i) * (double)(S[i] * S[o->nbr[i * 6 + 2 * d]]);
        E -= o->h * (double)S[i];
    }
    return E;
}
double ea_energy_pt(const ea_oracle *o, int a, int t) { return energy_pt(o, a, t); }
void ea_get_thresholds(const ea_oracle *o, uint64_t *out)   /* [NT][7][2] */
{
    memcpy(out, o->thr, sizeof(uint64_t) * o->NT * 14);
}
void ea_get_moments(const ea_oracle *o, double *out, int64_t *n_meas)   /* [NT][66] */
{
    memcpy(out, o->acc, sizeof(double) * o->NT * EA_NMOM);
    if (n_meas) *n_meas = o->n_meas;
}
void ea_get_counters(const ea_oracle *o, uint64_t *sweeps, uint64_t *exchanges)
{
    if (sweeps) *sweeps = o->sweeps;
    if (exchanges) *exchanges = o->exchanges;
}
/* diagnostics: switch on the P(q) histogram with n_bins bins (1 <= n_bins <= N + 1; N + 1 = one bin per value of q) */
int ea_enable_pq(ea_oracle *o, int n_bins)
{
    if (n_bins < 1 || n_bins > o->N + 1) return -1;
    free(o->pq);
    o->pq = (uint64_t *)calloc((size_t)o->NT * n_bins, sizeof(uint64_t));
    o->pq_bins = o->pq ? n_bins : 0;
    return o->pq ? 0 : -1;
}
void ea_get_pq(const ea_oracle *o, uint64_t *out)          /* [NT][pq_bins] */
{
    memcpy(out, o->pq, sizeof(uint64_t) * (size_t)o->NT * o->pq_bins);
}
/* diagnostics: switch on the per-window accumulators of the logarithmic-binning test */
int ea_enable_log_binning(ea_oracle *o, int n_windows)
{
    if (n_windows < 1 || n_windows > 40) return -1;
    free(o->accw); free(o->n_meas_w);
    o->accw = (double *)calloc((size_t)n_windows * o->NT * EA_NMOM, sizeof(double));
    o->n_meas_w = (int64_t *)calloc((size_t)n_windows, sizeof(int64_t));
    o->n_windows = (o->accw && o->n_meas_w) ? n_windows : 0;
    return o->n_windows ? 0 : -1;
}
void ea_get_window_moments(const ea_oracle *o, int k, double *out, int64_t *n_meas)   /* [NT][66] of window k */
{
    memcpy(out, o->accw + (size_t)k * o->NT * EA_NMOM, sizeof(double) * o->NT * EA_NMOM);
    if (n_meas) *n_meas = o->n_meas_w[k];
}
void ea_get_pt_stats(const ea_oracle *o, uint64_t *proposed, uint64_t *accepted)
{
    *proposed = o->n_pt_prop; *accepted = o->n_pt_acc;
}

/* time series for the equilibrium pins (tests/test_oracle_equilibrium.py): after every sweep
 * (and PT step, if due) record the literal Eq.-1 energy inputs (U, M) of every system and the
 * integer overlap Q_t = sum_j S^0_j S^1_j of replicas 0 and 1 at every slot. */
void ea_run_series(ea_oracle *o, int n_sweeps, int pt_every, int64_t *U_out, int32_t *M_out, int32_t *Q_out)
{
    const int RT = o->R * o->NT;
    for (int s = 0; s < n_sweeps; ++s) {
        sweep_once(o);
        if (pt_every > 0 && (o->sweeps % (uint64_t)pt_every) == 0) ea_pt_exchange(o);
        for (int i = 0; i < RT; ++i) {
            if (U_out) U_out[(size_t)s * RT + i] = o->U[i];
            if (M_out) M_out[(size_t)s * RT + i] = o->M[i];
        }
        if (Q_out && o->R >= 2)
            for (int t = 0; t < o->NT; ++t) {
                const int *A = Sys(o, 0, t), *B = Sys(o, 1, t);
                int32_t q = 0;
                for (int j = 0; j < o->N; ++j) q += A[j] * B[j];
                Q_out[(size_t)s * o->NT + t] = q;
            }
    }
}
