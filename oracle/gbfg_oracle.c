/* gbfg_oracle.c — the ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, single-threaded CPU statement of what libgbfg's hot path computes
 * (catalog of galactic binaries -> confusion-noise PSD by iterative subtraction).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this file's library.  It shares NO code with paper_2602_18560_b200/csrc:
 * no headers, helpers, tables or constant generators; every constant is typed here.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md at build time; DESIGN.md §3 lists
 * every reading taken where the paper is silent):
 *   - algorithm steps 1-10 of Appendix D, loop reading DESIGN.md R6
 *   - running median, eq. (D2), normalisation C eq. (D3)
 *   - total PSD S_n = S_instr + S_gal, eq. (10)
 *   - SNR inner product eqs. (11)-(12) PAPER.md:159-166 in BASELINE.json:configs[0]'s
 *     power-domain form  rho^2 = sum_bins 4 P_i / S_n ;  threshold rho_th = 7
 *   - GW-driven chirp eq. (4) PAPER.md:63 inside BASELINE.json:configs[0]'s generator
 *   - subtraction = scatter-add of -template, eq. (D4)
 *
 * Arithmetic: IEEE-754 binary64, round-to-nearest-even, every operation singly rounded
 * (compile with -O2 -ffp-contract=off, no -ffast-math).  fma() is used only where the
 * DESIGN.md §4 specification of the elementary functions says "fma".
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   philox4x32_10      Random123 known-answer vectors
 *   u01                range/exactness; KS of f, z against closed-form CDFs
 *   orc_log/exp10/sincos   mpmath at 40 digits, <= 4 ulp; glibc libm
 *   fdot               eq. (4) values SURVEY.md App. A via mpmath
 *   instrument noise   Robson-curve values SURVEY.md App. A, mpmath re-evaluation
 *   source_bins        worked examples SURVEY.md App. A (tests/golden/worked_sources.txt)
 *   deposit            brute force; difference-array identity; sum conservation; +1/-1 = 0
 *   running median     sort-per-output definition; scipy.ndimage.median_filter(mode='reflect')
 *   snr                closed form for an isolated source; long-double summation; scalings
 *   loop               power conservation; monotone foreground; idempotence; rho_th -> inf, 0+
 *   channel-sum noise  exact rationals; eq. (11) for an isolated source at 40 digits (R14)
 * parity unpinned: iteration counts / N_res against the paper's Table III
 * and the catalog distribution against the paper's population (different data model,
 * DESIGN.md §3 R0).
 */
#define _POSIX_C_SOURCE 199309L
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>

/* ------------------------------------------------------------------------------------ */
/* Stage (i) — Philox4x32-10 (Salmon et al. 2011), R1                          */
/* ------------------------------------------------------------------------------------ */

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* 52 random bits -> u in (0,1): u = (x + 1/2) * 2^-52, exact in binary64, never 0 or 1. */
double orc_u01(uint32_t w_lo, uint32_t w_hi)
{
    uint64_t x = (((uint64_t)w_hi << 32) | (uint64_t)w_lo) >> 12;
    return ((double)x + 0.5) * 0x1p-52;
}

/* ------------------------------------------------------------------------------------ */
/* Elementary functions, specified operation by operation in DESIGN.md §4 so that the    */
/* CUDA side (which implements the same text independently) agrees to the bit.           */
/* ------------------------------------------------------------------------------------ */

static const double ORC_SQRT_HALF = 0.7071067811865476;
static const double ORC_LN2_HI = 0.6931471803691238;       /* 0x3FE62E42FEE00000 */
static const double ORC_LN2_LO = 1.9082149292705877e-10;   /* 0x3DEA39EF35793C76 */
static const double ORC_LOG10_E = 0.4342944819032518;
static const double ORC_LN10 = 2.302585092994046;
static const double ORC_LOG2_10 = 3.321928094887362;
static const double ORC_LOG10_2_HI = 0.3010299955494702;   /* 0x3FD3441350800000 */
static const double ORC_LOG10_2_LO = 1.1451100898021838e-10;
static const double ORC_PIO2_HI = 1.5707963267341256;      /* 0x3FF921FB54400000 */
static const double ORC_PIO2_LO = 6.077100506506192e-11;
static const double ORC_PIO2 = 1.5707963267948966;
static const double ORC_TWO_OVER_PI = 0.6366197723675814;
static const double ORC_TWO_PI = 6.283185307179586;

/* natural log of a positive normal double: atanh series on m in [sqrt(1/2), sqrt(2)) */
double orc_log(double x)
{
    int e;
    double m = frexp(x, &e);               /* x = m * 2^e, m in [1/2, 1) */
    if (m < ORC_SQRT_HALF) { m = 2.0 * m; e = e - 1; }
    double s = (m - 1.0) / (m + 1.0);
    double z = s * s;
    double q = 1.0 / 23.0;
    q = fma(q, z, 1.0 / 21.0);
    q = fma(q, z, 1.0 / 19.0);
    q = fma(q, z, 1.0 / 17.0);
    q = fma(q, z, 1.0 / 15.0);
    q = fma(q, z, 1.0 / 13.0);
    q = fma(q, z, 1.0 / 11.0);
    q = fma(q, z, 1.0 / 9.0);
    q = fma(q, z, 1.0 / 7.0);
    q = fma(q, z, 1.0 / 5.0);
    q = fma(q, z, 1.0 / 3.0);
    double t = 2.0 * s;
    double lm = fma(t * z, q, t);          /* log m = 2s + 2s z (1/3 + z/5 + ...) */
    double de = (double)e;
    return de * ORC_LN2_HI + fma(de, ORC_LN2_LO, lm);
}

/* e^t for |t| <= 0.36 : Taylor through t^14 */
static double orc_exp_small(double t)
{
    double p = 1.0 / 87178291200.0;        /* 1/14! */
    p = fma(p, t, 1.0 / 6227020800.0);     /* 1/13! */
    p = fma(p, t, 1.0 / 479001600.0);
    p = fma(p, t, 1.0 / 39916800.0);
    p = fma(p, t, 1.0 / 3628800.0);
    p = fma(p, t, 1.0 / 362880.0);
    p = fma(p, t, 1.0 / 40320.0);
    p = fma(p, t, 1.0 / 5040.0);
    p = fma(p, t, 1.0 / 720.0);
    p = fma(p, t, 1.0 / 120.0);
    p = fma(p, t, 1.0 / 24.0);
    p = fma(p, t, 1.0 / 6.0);
    p = fma(p, t, 0.5);
    return 1.0 + fma(t * t, p, t);
}

/* 10^y for |y| < 300 (result normal) */
double orc_exp10(double y)
{
    double k = rint(y * ORC_LOG2_10);
    double r = fma(-k, ORC_LOG10_2_HI, y);
    r = fma(-k, ORC_LOG10_2_LO, r);
    double t = r * ORC_LN10;
    return ldexp(orc_exp_small(t), (int)k);
}

/* sin and cos of phi, |phi| <= pi/4 (+ rounding): Taylor through phi^19 / phi^18 */
static void orc_sincos_small(double phi, double *sn, double *cs)
{
    double z = phi * phi;
    double p = -1.0 / 121645100408832000.0;     /* -1/19! */
    p = fma(p, z, 1.0 / 355687428096000.0);     /* +1/17! */
    p = fma(p, z, -1.0 / 1307674368000.0);      /* -1/15! */
    p = fma(p, z, 1.0 / 6227020800.0);          /* +1/13! */
    p = fma(p, z, -1.0 / 39916800.0);           /* -1/11! */
    p = fma(p, z, 1.0 / 362880.0);              /* +1/9!  */
    p = fma(p, z, -1.0 / 5040.0);               /* -1/7!  */
    p = fma(p, z, 1.0 / 120.0);                 /* +1/5!  */
    p = fma(p, z, -1.0 / 6.0);                  /* -1/3!  */
    *sn = fma(phi * z, p, phi);
    double q = -1.0 / 6402373705728000.0;       /* -1/18! */
    q = fma(q, z, 1.0 / 20922789888000.0);      /* +1/16! */
    q = fma(q, z, -1.0 / 87178291200.0);        /* -1/14! */
    q = fma(q, z, 1.0 / 479001600.0);           /* +1/12! */
    q = fma(q, z, -1.0 / 3628800.0);            /* -1/10! */
    q = fma(q, z, 1.0 / 40320.0);               /* +1/8!  */
    q = fma(q, z, -1.0 / 720.0);                /* -1/6!  */
    q = fma(q, z, 1.0 / 24.0);                  /* +1/4!  */
    q = fma(q, z, -0.5);                        /* -1/2!  */
    *cs = fma(z, q, 1.0);
}

static void orc_quadrant(int quad, double sn, double cs, double *s_out, double *c_out)
{
    switch (quad & 3) {
    case 0: *s_out = sn;  *c_out = cs;  break;
    case 1: *s_out = cs;  *c_out = -sn; break;
    case 2: *s_out = -sn; *c_out = -cs; break;
    default: *s_out = -cs; *c_out = sn; break;
    }
}

/* sin(2 pi u), cos(2 pi u) for u in [0,1): the reduction is exact (argument in turns) */
void orc_sincos2pi(double u, double *s_out, double *c_out)
{
    double t = 4.0 * u;
    double q = rint(t);
    double d = t - q;                      /* exact, |d| <= 1/2 */
    double sn, cs;
    orc_sincos_small(d * ORC_PIO2, &sn, &cs);
    orc_quadrant((int)q, sn, cs, s_out, c_out);
}

/* sin(x), cos(x) for |x| < 1e5: two-constant Cody-Waite reduction by pi/2 */
void orc_sincos(double x, double *s_out, double *c_out)
{
    double q = rint(x * ORC_TWO_OVER_PI);
    double r = fma(-q, ORC_PIO2_HI, x);
    r = fma(-q, ORC_PIO2_LO, r);
    double sn, cs;
    orc_sincos_small(r, &sn, &cs);
    orc_quadrant((int)((long long)q & 3), sn, cs, s_out, c_out);
}

/* ------------------------------------------------------------------------------------ */
/* Grid (R2)                                                                   */
/* ------------------------------------------------------------------------------------ */

typedef struct {
    double f_min, f_max, t_obs;
    int64_t n_bins;
    int32_t scale_log2;
} orc_grid;

/* n_bins = ceil((f_max - f_min) * T): every f in [f_min, f_max) has a bin of width 1/T */
int64_t orc_n_bins(double f_min, double f_max, double t_obs)
{
    return (int64_t)ceil((f_max - f_min) * t_obs);
}

/* ------------------------------------------------------------------------------------ */
/* Stage (i) — catalog sampling, BASELINE.json:configs[0] generator, R1        */
/* ------------------------------------------------------------------------------------ */

typedef struct {
    double slope, logA_offset, logA_sigma, logMc_mean, logMc_sigma;
    int64_t n_src;
} orc_pop;

static const double ORC_LOG10_K = 2.6090342225545732;      /* log10((96/5) pi^(8/3)), eq. (4) */
static const double ORC_LOG10_TSUN = -5.3075504747653498;  /* log10(G Msun / c^3 / s), 4.925490947641267e-6 s */

void orc_sample_catalog(const orc_grid *g, const orc_pop *pop, uint32_t cat_id, uint64_t seed,
                        int64_t i_begin, int64_t i_end, double *A, double *f, double *fdot)
{
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    const double lfmin = orc_log(g->f_min) * ORC_LOG10_E;
    const double lfmax = orc_log(g->f_max) * ORC_LOG10_E;
    const double f_top = nextafter(g->f_max, 0.0);
    const double oms = 1.0 - pop->slope;
    const int flat_in_log = fabs(oms) < 1e-12;
    double c0, c1, c2;
    if (flat_in_log) {                      /* p(f) ∝ 1/f : log f uniform */
        c0 = lfmin; c1 = lfmax - lfmin; c2 = 1.0;
    } else {                                /* inverse CDF of p(f) ∝ f^-s on [f_min, f_max) */
        double a = orc_exp10(oms * lfmin);
        double b = orc_exp10(oms * lfmax);
        c0 = a; c1 = b - a; c2 = 1.0 / oms;
    }
    for (int64_t i = i_begin; i < i_end; ++i) {
        uint32_t ctr[4] = {(uint32_t)i, (uint32_t)((uint64_t)i >> 32), 0u, cat_id};
        uint32_t w0[4], w1[4];
        orc_philox4x32_10(ctr, key, w0);
        ctr[2] = 1u;
        orc_philox4x32_10(ctr, key, w1);
        double u_f = orc_u01(w0[0], w0[1]);
        double u_1 = orc_u01(w0[2], w0[3]);
        double u_2 = orc_u01(w1[0], w1[1]);
        /* frequency */
        double lf;
        if (flat_in_log) {
            lf = c0 + u_f * c1;
        } else {
            double x = c0 + u_f * c1;
            lf = (orc_log(x) * ORC_LOG10_E) * c2;
        }
        double fi = orc_exp10(lf);
        if (fi < g->f_min) fi = g->f_min;
        if (fi >= g->f_max) fi = f_top;
        /* Box-Muller normals */
        double r = sqrt(-2.0 * orc_log(u_1));
        double sn, cs;
        orc_sincos2pi(u_2, &sn, &cs);
        double z_A = r * cs;
        double z_M = r * sn;
        /* amplitude: log10 A ~ N(off + (2/3) log10(f / 1 mHz), sigma) */
        double t1 = lf + 3.0;
        double t2 = (2.0 / 3.0) * t1;
        double t3 = pop->logA_offset + t2;
        double t4 = pop->logA_sigma * z_A;
        double Ai = orc_exp10(t3 + t4);
        /* chirp: eq. (4) with log10(Mc/Msun) ~ N(mean, sigma) */
        double lmc = pop->logMc_mean + pop->logMc_sigma * z_M;
        double m1 = (5.0 / 3.0) * (ORC_LOG10_TSUN + lmc);
        double m2 = (11.0 / 3.0) * lf;
        double fd = orc_exp10((ORC_LOG10_K + m1) + m2);
        A[i - i_begin] = Ai;
        f[i - i_begin] = fi;
        fdot[i - i_begin] = fd;
    }
}

/* ------------------------------------------------------------------------------------ */
/* The paper's own population sampler (R12): Table I            */
/* (PAPER.md:81-87), eqs. (7)-(9), Gaussian copula of Appendix A steps     */
/* (iii)-(iv).  Elementary functions as DESIGN.md R12 lists them.          */
/* ------------------------------------------------------------------------------------ */
static double orc_expn(double y) { return orc_exp10(y * ORC_LOG10_E); }   /* e^y */

/* Lengths of the fixed recurrences below (R12 derives them and states the domain they cover:
 * 0.25 <= alpha_Gamma <= 16, |z| <= 8.6).  Macros only so that tests/test_oracle_paper_sampler.py can build this
 * file "one notch shorter" and show that the pins catch it; the product of this file uses the defaults. */
#ifndef ORC_ERFC_SERIES_TERMS
#define ORC_ERFC_SERIES_TERMS 80
#endif
#ifndef ORC_ERFC_CF_DEPTH
#define ORC_ERFC_CF_DEPTH 40
#endif
#ifndef ORC_GAMMA_SERIES_TERMS
#define ORC_GAMMA_SERIES_TERMS 48
#endif
#ifndef ORC_GAMMA_CF_DEPTH
#define ORC_GAMMA_CF_DEPTH 40
#endif
#ifndef ORC_QUANTILE_NEWTON_STEPS
#define ORC_QUANTILE_NEWTON_STEPS 10
#endif

/* erfc(t), t >= 0: for t < 2 the all-positive series erf t = (2/sqrt pi) e^{-t^2} sum 2^n t^{2n+1} / (2n+1)!!
 * (80 terms), else the continued fraction e^{-t^2} / (sqrt pi (t + (1/2)/(t + 1/(t + (3/2)/(t + ...))))), depth 40,
 * evaluated from the bottom */
double orc_erfc_pos(double t)
{
    const double SQRT_PI = 1.7724538509055159;
    double t2 = t * t;
    if (t < 2.0) {
        double term = t, sum = t;
        for (int n = 1; n < ORC_ERFC_SERIES_TERMS; ++n) {
            term = term * (2.0 * t2) / (double)(2 * n + 1);
            sum = sum + term;
        }
        return 1.0 - (2.0 / SQRT_PI) * orc_expn(-t2) * sum;
    }
    double r = t;
    for (int k = ORC_ERFC_CF_DEPTH; k >= 1; --k) r = t + (0.5 * (double)k) / r;
    return orc_expn(-t2) / (SQRT_PI * r);
}

/* tail probability of a standard normal beyond z on z's own side: Phi(z) for z <= 0, 1 - Phi(z) for z > 0 */
double orc_norm_tail(double z)
{
    return 0.5 * orc_erfc_pos(fabs(z) * 0.7071067811865476);
}

/* regularized incomplete gamma functions P(a,x), Q(a,x) and the prefactor x^a e^-x / Gamma(a); lg = ln Gamma(a).
 * x < a + 3: series P = pref * sum_{n>=0} x^n / (a (a+1) ... (a+n)), 48 terms, Q = 1 - P;
 * else Legendre's continued fraction Q = pref / (x+1-a - 1(1-a)/(x+3-a - 2(2-a)/(x+5-a - ...))), depth 40, P = 1 - Q */
void orc_gamma_pq(double a, double x, double lg, double *P, double *Q, double *pref_out)
{
    double pref = orc_expn((a * orc_log(x) - x) - lg);
    if (x < a + 3.0) {
        double term = 1.0 / a, sum = term;
        for (int n = 1; n <= ORC_GAMMA_SERIES_TERMS; ++n) {
            term = term * x / (a + (double)n);
            sum = sum + term;
        }
        *P = sum * pref;
        *Q = 1.0 - *P;
    } else {
        double r = (x + (double)(2 * ORC_GAMMA_CF_DEPTH + 1)) - a;        /* depth 40: x + 81 - a */
        for (int k = ORC_GAMMA_CF_DEPTH; k >= 1; --k) r = ((x + (double)(2 * k - 1)) - a) - ((double)k * ((double)k - a)) / r;
        *Q = pref / r;
        *P = 1.0 - *Q;
    }
    *pref_out = pref;
}

/* x with P(a,x) = Phi(z): Wilson-Hilferty start from z, then 10 Newton steps on the logarithm of the tail
 * probability on z's side (P for z <= 0, Q for z > 0), each step kept within [x/10, 2x + 4].
 * lg = ln Gamma(a), lg1 = ln Gamma(a + 1). */
double orc_gamma_quantile(double a, double lg, double lg1, double z)
{
    double tail = orc_norm_tail(z);
    double c = 1.0 / (9.0 * a);
    double w = (1.0 - c) + z * sqrt(c);
    double x = a * ((w * w) * w);
    if (!(w > 0.0) || x < 1e-6 * a) x = orc_expn((orc_log(tail) + lg1) / a);   /* far lower tail: P ~ x^a / Gamma(a+1) */
    for (int it = 0; it < ORC_QUANTILE_NEWTON_STEPS; ++it) {
        double P, Q, pref;
        orc_gamma_pq(a, x, lg, &P, &Q, &pref);
        double pdf = pref / x;
        double g = (z <= 0.0) ? P * orc_log(P / tail) : -(Q * orc_log(Q / tail));
        double xn = x - g / pdf;
        if (xn < 0.1 * x) xn = 0.1 * x;
        if (xn > 2.0 * x + 4.0) xn = 2.0 * x + 4.0;
        x = xn;
    }
    return x;
}

typedef struct {
    uint32_t struct_size, reserved;
    double alpha_pl;       /* p(f) ∝ f^alpha_pl on the grid's band (Table I) */
    double alpha_gamma, beta_gamma, mu_gamma;   /* log10(fdot) - mu_gamma ~ Gamma(alpha, rate beta), eq. (7) */
    double mu, sigma;      /* log10[(f/Hz)^(-2/3) A] - mu ~ LogNormal(0, sigma), eq. (8) */
    double rho;            /* Gaussian-copula correlation of f and fdot, eqs. (A4)-(A5) */
    int64_t n_src;
} orc_pop_paper;

void orc_sample_catalog_paper(const orc_grid *g, const orc_pop_paper *pop, uint32_t cat_id, uint64_t seed,
                              int64_t i_begin, int64_t i_end, double *A, double *f, double *fdot)
{
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    const double lfmin = orc_log(g->f_min) * ORC_LOG10_E;
    const double lfmax = orc_log(g->f_max) * ORC_LOG10_E;
    const double f_top = nextafter(g->f_max, 0.0);
    const double oms = 1.0 + pop->alpha_pl;              /* exponent of the CDF: f^(1 + alpha) */
    const int flat_in_log = fabs(oms) < 1e-12;
    double c0, c1, c2;
    if (flat_in_log) {
        c0 = lfmin; c1 = lfmax - lfmin; c2 = 1.0;
    } else {
        double a = orc_exp10(oms * lfmin);
        double b = orc_exp10(oms * lfmax);
        c0 = a; c1 = b - a; c2 = 1.0 / oms;
    }
    const double lg = lgamma(pop->alpha_gamma), lg1 = lgamma(pop->alpha_gamma + 1.0);
    const double rho_c = sqrt(1.0 - pop->rho * pop->rho);
    for (int64_t i = i_begin; i < i_end; ++i) {
        uint32_t ctr[4] = {(uint32_t)i, (uint32_t)((uint64_t)i >> 32), 2u, cat_id};   /* blocks 2 and 3 */
        uint32_t w0[4], w1[4];
        orc_philox4x32_10(ctr, key, w0);
        ctr[2] = 3u;
        orc_philox4x32_10(ctr, key, w1);
        double u_1 = orc_u01(w0[0], w0[1]), u_2 = orc_u01(w0[2], w0[3]);
        double u_3 = orc_u01(w1[0], w1[1]), u_4 = orc_u01(w1[2], w1[3]);
        double r = sqrt(-2.0 * orc_log(u_1));
        double sn, cs;
        orc_sincos2pi(u_2, &sn, &cs);
        double n1 = r * cs, n2 = r * sn;
        double r3 = sqrt(-2.0 * orc_log(u_3));
        double s3, c3;
        orc_sincos2pi(u_4, &s3, &c3);
        double z3 = r3 * c3;
        /* step (iii): (z1, z2) ~ N(0, Sigma) */
        double z1 = n1;
        double z2 = pop->rho * n1 + rho_c * n2;
        /* step (iv), frequency: u' = Phi(z1) through the inverse CDF of the truncated power law */
        double t1 = orc_norm_tail(z1);
        double uf = (z1 <= 0.0) ? t1 : 1.0 - t1;
        double lf;
        if (flat_in_log) {
            lf = c0 + uf * c1;
        } else {
            double x = c0 + uf * c1;
            lf = (orc_log(x) * ORC_LOG10_E) * c2;
        }
        double fi = orc_exp10(lf);
        if (fi < g->f_min) fi = g->f_min;
        if (fi >= g->f_max) fi = f_top;
        /* step (iv), chirp: v' = Phi(z2) through the inverse Gamma CDF, eq. (7) */
        double xg = orc_gamma_quantile(pop->alpha_gamma, lg, lg1, z2);
        double fd = orc_exp10(pop->mu_gamma + xg / pop->beta_gamma);
        /* amplitude, eq. (8): A~ = exp(sigma z3) (log-normal), log10 A = mu + A~ + (2/3) log10(f / Hz) */
        double at = orc_expn(pop->sigma * z3);
        double Ai = orc_exp10((pop->mu + at) + (2.0 / 3.0) * lf);
        A[i - i_begin] = Ai;
        f[i - i_begin] = fi;
        fdot[i - i_begin] = fd;
    }
}

/* ------------------------------------------------------------------------------------ */
/* Instrument noise: Robson, Cornish & Liu 2019 sky-averaged curve (PAPER.md:670 ref [70]) */
/* with BASELINE.json:configs[0]'s constants, at bin centres.  DESIGN.md R3.              */
/* ------------------------------------------------------------------------------------ */

double orc_robson_sn(double fq)
{
    const double L = 2.5e9, fstar = 19.09e-3;
    double r2 = 2.0e-3 / fq;  r2 = r2 * r2;                   /* (2 mHz / f)^2 */
    double p_oms = (1.5e-11 * 1.5e-11) * (1.0 + r2 * r2);
    double r4 = 0.4e-3 / fq;
    double r8 = fq / 8.0e-3;  r8 = r8 * r8;
    double p_acc = (3.0e-15 * 3.0e-15) * (1.0 + r4 * r4) * (1.0 + r8 * r8);
    double x = fq / fstar;
    double sn, cs;
    orc_sincos(x, &sn, &cs);
    double y = ORC_TWO_PI * fq;  y = y * y;  y = y * y;       /* (2 pi f)^4 */
    double acc = 2.0 * (1.0 + cs * cs) * p_acc / y;
    return (10.0 / (3.0 * L * L)) * (p_oms + acc) * (1.0 + 0.6 * (x * x));
}

/* SciRDv1 noise in the TDI A/E/T channels, eqs. (C1)-(C5) PAPER.md:494-509, and its rescaling by the
 * TDI response, eqs. (B2)-(B5) PAPER.md:475-487 (R11).  P in pm, A in fm s^-2, L in m.
 * out[0] = S^AA = S^EE (C3), out[1] = S^TT (C4) (both times 4 sin^2(2 f/f*) when tdi2, C5),
 * out[2] = S^AA / R_AA, out[3] = S^TT / R_TT (B2; the TDI generation cancels in the ratio).
 * (C2) is garbled in PAPER.md:496: "(f / 8 mHz^4)" is read as (f / 8 mHz)^4.
 * 1 - cos x is taken as 2 sin^2(x/2): no cancellation at the low end of the band. */
void orc_aet_noise(double fq, double P, double A, double L, int tdi2, double out[4])
{
    const double c = 299792458.0;
    double fstar = c / (ORC_TWO_PI * L);
    double x = fq / fstar;
    double sn, cs, sh, ch;
    orc_sincos(x, &sn, &cs);
    orc_sincos(0.5 * x, &sh, &ch);
    double omc = 2.0 * (sh * sh);                               /* 1 - cos x */
    double k2 = ORC_TWO_PI * fq / c;  k2 = k2 * k2;             /* (2 pi f / c)^2 */
    double r2 = 2.0e-3 / fq;  r2 = r2 * r2;
    double a_oms = P * 1.0e-12;
    double p_oms = (a_oms * a_oms) * (1.0 + r2 * r2) * k2;     /* (C1) */
    double r4 = 0.4e-3 / fq;
    double r8 = fq / 8.0e-3;  r8 = r8 * r8;
    double a_tm = A * 1.0e-15;
    double y = ORC_TWO_PI * fq;  y = y * y;  y = y * y;         /* (2 pi f)^4 */
    double p_tm = (a_tm * a_tm) * (1.0 + r4 * r4) * (1.0 + r8 * r8) / y * k2;   /* (C2) */
    double s2 = sn * sn;
    double s_aa = 8.0 * s2 * (4.0 * (1.0 + cs + cs * cs) * p_tm + (2.0 + cs) * p_oms);   /* (C3) */
    double s_tt = 16.0 * s2 * (2.0 * (omc * omc) * p_tm + omc * p_oms);                  /* (C4) */
    double x2 = x * x;
    double pre = 16.0 * s2 * x2;                                /* (B3) */
    double r_aa = pre * (0.45 / (1.0 + 0.7 * x2));              /* (B4), 9/20 */
    double x4 = x2 * x2;
    double r_tt = pre * (0.45 * (x4 * x2) / (1.8e3 + 0.7 * (x4 * x4)));   /* (B5) */
    out[2] = s_aa / r_aa;
    out[3] = s_tt / r_tt;
    if (tdi2) {
        double s2x, c2x;
        orc_sincos(2.0 * x, &s2x, &c2x);
        double fac = 4.0 * (s2x * s2x);                         /* (C5) */
        s_aa = fac * s_aa;
        s_tt = fac * s_tt;
    }
    out[0] = s_aa;
    out[1] = s_tt;
}

/* the four curves at the bin centres f_min + (k + 1/2)/T; any output may be NULL */
void orc_instrument_noise_aet(const orc_grid *g, double P, double A, double L, int tdi2,
                              double *s_aa, double *s_tt, double *sh_aa, double *sh_tt)
{
    for (int64_t k = 0; k < g->n_bins; ++k) {
        double fk = g->f_min + ((double)k + 0.5) / g->t_obs;
        double o[4];
        orc_aet_noise(fk, P, A, L, tdi2, o);
        if (s_aa) s_aa[k] = o[0];
        if (s_tt) s_tt[k] = o[1];
        if (sh_aa) sh_aa[k] = o[2];
        if (sh_tt) sh_tt[k] = o[3];
    }
}

/* Noise curve of the SNR summed over the TDI channels, eq. (11) PAPER.md:159-166 (R14).  In the power domain a
 * source's strain power p enters channel X with the sky-averaged response R_XX, so that channel's term of eq. (11) is
 * 4 p R_XX / S^XX = 4 p / S_h^XX; A and E are equal (C3), hence  rho^2 = sum_bins 4 p (2 / S_h^AA + 1 / S_h^TT)
 * = sum_bins 4 p / S_sum  with  S_sum = 1 / ((2 / S_h^AA) + (1 / S_h^TT)):  the loop run on S_sum as its s_instr is the
 * channel-summed SNR.  Four IEEE operations per bin, in this order. */
void orc_channel_sum_noise(const double *sh_aa, const double *sh_tt, int64_t n, double *out)
{
    for (int64_t k = 0; k < n; ++k) {
        double ta = 2.0 / sh_aa[k];
        double tt = 1.0 / sh_tt[k];
        double s = ta + tt;
        out[k] = 1.0 / s;
    }
}

void orc_instrument_noise(const orc_grid *g, double *s_instr)
{
    for (int64_t k = 0; k < g->n_bins; ++k) {
        double fk = g->f_min + ((double)k + 0.5) / g->t_obs;
        s_instr[k] = orc_robson_sn(fk);
    }
}

/* ------------------------------------------------------------------------------------ */
/* Stage (ii) — deposit (R2).                                                  */
/* ------------------------------------------------------------------------------------ */

/* Returns 0 if the source deposits, 1 = DOMAIN (NaN, A<0, fdot<0, f outside the band),
 * 2 = RANGE (width or quantised power out of the int64 headroom). */
int orc_source_bins(const orc_grid *g, double A, double f, double fdot,
                    int64_t *k0, int64_t *w, int64_t *w_eff, double *p, int64_t *q)
{
    if (!(A >= 0.0) || !(fdot >= 0.0) || !(f >= g->f_min) || !(f < g->f_max)) return 1;
    double T = g->t_obs;
    double T2 = T * T;
    double kk = floor((f - g->f_min) * T);
    if (!(kk < (double)g->n_bins)) return 1;
    double ww = ceil(fdot * T2);
    if (!(ww < 0x1p62)) return 2;
    if (ww < 1.0) ww = 1.0;
    double P = (A * A) * (0.5 * T);
    double pp = P / ww;
    double qd = ldexp(pp, -g->scale_log2);
    if (!(qd < 0x1p62)) return 2;
    *k0 = (int64_t)kk;
    *w = (int64_t)ww;
    *w_eff = (*w < g->n_bins - *k0) ? *w : (g->n_bins - *k0);
    *p = pp;
    *q = llrint(qd);
    return 0;
}

/* spectrum[k] += sign * q_i for k in [k0_i, k0_i + w_eff_i).  sel == NULL: sources 0..n-1,
 * else the n_sel listed indices.  Returns the number of rejected sources. */
int64_t orc_deposit(const orc_grid *g, const double *A, const double *f, const double *fdot,
                    int64_t n, const int64_t *sel, int64_t n_sel, int32_t sign, int64_t *spectrum)
{
    int64_t rejected = 0;
    int64_t count = sel ? n_sel : n;
    for (int64_t j = 0; j < count; ++j) {
        int64_t i = sel ? sel[j] : j;
        int64_t k0, w, w_eff, q; double p;
        if (orc_source_bins(g, A[i], f[i], fdot[i], &k0, &w, &w_eff, &p, &q)) { ++rejected; continue; }
        for (int64_t k = k0; k < k0 + w_eff; ++k) spectrum[k] += (int64_t)sign * q;
    }
    return rejected;
}

/* ------------------------------------------------------------------------------------ */
/* Stage (iii) — running median, eq. (D2), R3: odd window W = 2h+1 centred on  */
/* k, half-sample-symmetric reflection at both ends, statistic = the h-th (0-based)      */
/* smallest of the 2h+1 values.                                                          */
/* ------------------------------------------------------------------------------------ */

static int64_t orc_reflect(int64_t j, int64_t n)
{
    if (j < 0) j = -j - 1;
    if (j >= n) j = 2 * n - 1 - j;
    return j;
}

static int orc_cmp_i64(const void *a, const void *b)
{
    int64_t x = *(const int64_t *)a, y = *(const int64_t *)b;
    return (x > y) - (x < y);
}

/* The definition written out: sort every window.  Outputs k in [k_begin, k_end). */
int orc_running_median_sort(const int64_t *x, int64_t n, int32_t window,
                            int64_t k_begin, int64_t k_end, int64_t *out)
{
    if (window < 1 || (window & 1) == 0) return -1;
    int64_t h = window / 2;
    if (n < h + 1) return -1;
    int64_t *buf = (int64_t *)malloc(sizeof(int64_t) * (size_t)window);
    for (int64_t k = k_begin; k < k_end; ++k) {
        for (int64_t j = -h; j <= h; ++j) buf[j + h] = x[orc_reflect(k + j, n)];
        qsort(buf, (size_t)window, sizeof(int64_t), orc_cmp_i64);
        out[k - k_begin] = buf[h];
    }
    free(buf);
    return 0;
}

/* Same result, sliding: keep the window as a sorted array, erase the value that leaves and
 * insert the value that enters (O(W) per step).  Checked against the definition above. */
int orc_running_median(const int64_t *x, int64_t n, int32_t window, int64_t *out)
{
    if (window < 1 || (window & 1) == 0) return -1;
    int64_t h = window / 2, W = window;
    if (n < h + 1) return -1;
    int64_t *win = (int64_t *)malloc(sizeof(int64_t) * (size_t)W);
    for (int64_t j = -h; j <= h; ++j) win[j + h] = x[orc_reflect(j, n)];
    qsort(win, (size_t)W, sizeof(int64_t), orc_cmp_i64);
    out[0] = win[h];
    for (int64_t k = 1; k < n; ++k) {
        int64_t gone = x[orc_reflect(k - 1 - h, n)];
        int64_t come = x[orc_reflect(k + h, n)];
        if (gone != come) {
            int64_t lo = 0, hi = W;                       /* first position with win[pos] >= gone */
            while (lo < hi) { int64_t mid = (lo + hi) / 2; if (win[mid] < gone) lo = mid + 1; else hi = mid; }
            int64_t at = lo;
            lo = 0; hi = W;                               /* first position with win[pos] > come */
            while (lo < hi) { int64_t mid = (lo + hi) / 2; if (win[mid] <= come) lo = mid + 1; else hi = mid; }
            int64_t to = lo;
            if (to > at) {                                /* erase at, insert before to */
                memmove(win + at, win + at + 1, sizeof(int64_t) * (size_t)(to - 1 - at));
                win[to - 1] = come;
            } else {
                memmove(win + to + 1, win + to, sizeof(int64_t) * (size_t)(at - to));
                win[to] = come;
            }
        }
        out[k] = win[h];
    }
    free(win);
    return 0;
}

/* psd[k] = s_instr[k] + C * (med[k] * 2^scale_log2), eqs. (10), (D2), (D3) */
void orc_psd(const int64_t *med, const double *s_instr, int64_t n, double median_norm,
             int32_t scale_log2, double *psd)
{
    for (int64_t k = 0; k < n; ++k) {
        double e = ldexp((double)med[k], scale_log2);
        psd[k] = s_instr[k] + median_norm * e;
    }
}

/* ------------------------------------------------------------------------------------ */
/* Running-mean estimator, eq. (D1) PAPER.md:538 (the paper's production choice, :176, :552);  */
/* DESIGN.md R8.  Same window as the median: W = 2h+1 bins centred on k, ends reflected.        */
/* The exact object is the int64 window SUM; the mean enters the PSD as one division by W.      */
/* ------------------------------------------------------------------------------------ */

/* The definition written out: add up every window.  Outputs k in [k_begin, k_end). */
int orc_running_sum_def(const int64_t *x, int64_t n, int32_t window,
                        int64_t k_begin, int64_t k_end, int64_t *out)
{
    if (window < 1 || (window & 1) == 0) return -1;
    int64_t h = window / 2;
    if (n < h + 1) return -1;
    for (int64_t k = k_begin; k < k_end; ++k) {
        int64_t acc = 0;
        for (int64_t j = -h; j <= h; ++j) acc += x[orc_reflect(k + j, n)];
        out[k - k_begin] = acc;
    }
    return 0;
}

/* Same result, sliding: subtract the value that leaves, add the value that enters (integers:
 * no rounding, so this is the definition regrouped).  Checked against the definition above. */
int orc_running_sum(const int64_t *x, int64_t n, int32_t window, int64_t *out)
{
    if (window < 1 || (window & 1) == 0) return -1;
    int64_t h = window / 2;
    if (n < h + 1) return -1;
    int64_t acc = 0;
    for (int64_t j = -h; j <= h; ++j) acc += x[orc_reflect(j, n)];
    out[0] = acc;
    for (int64_t k = 1; k < n; ++k) {
        acc -= x[orc_reflect(k - 1 - h, n)];
        acc += x[orc_reflect(k + h, n)];
        out[k] = acc;
    }
    return 0;
}

/* psd[k] = s_instr[k] + (sum[k] * 2^scale_log2) / W, eqs. (10), (D1) */
void orc_psd_mean(const int64_t *sum, const double *s_instr, int64_t n, int32_t window,
                  int32_t scale_log2, double *psd)
{
    for (int64_t k = 0; k < n; ++k) {
        double e = ldexp((double)sum[k], scale_log2);
        double m = e / (double)window;
        psd[k] = s_instr[k] + m;
    }
}

/* ------------------------------------------------------------------------------------ */
/* Stage (iv) — SNR and selection, eqs. (11)-(12) in the power domain, R4.     */
/* ------------------------------------------------------------------------------------ */

/* rho^2 of one source: ascending-bin sum of (4 p) / psd[k] with a binary64 accumulator.
 * Returns NaN for a rejected source. */
double orc_rho2(const orc_grid *g, double A, double f, double fdot, const double *psd)
{
    int64_t k0, w, w_eff, q; double p;
    if (orc_source_bins(g, A, f, fdot, &k0, &w, &w_eff, &p, &q)) return NAN;
    double four_p = 4.0 * p;
    double acc = 0.0;
    for (int64_t k = k0; k < k0 + w_eff; ++k) acc = acc + four_p / psd[k];
    return acc;
}

/* Same sum with a long double accumulator and long double divisions (pin only). */
long double orc_rho2_ld(const orc_grid *g, double A, double f, double fdot, const double *psd)
{
    int64_t k0, w, w_eff, q; double p;
    if (orc_source_bins(g, A, f, fdot, &k0, &w, &w_eff, &p, &q)) return (long double)NAN;
    long double acc = 0.0L;
    for (int64_t k = k0; k < k0 + w_eff; ++k) acc += (long double)(4.0 * p) / (long double)psd[k];
    return acc;
}

double orc_rho2_ld_as_double(const orc_grid *g, double A, double f, double fdot, const double *psd)
{
    return (double)orc_rho2_ld(g, A, f, fdot, psd);
}

/* Tests every source with resolved[i] == 0; a source is newly resolved iff rho2 > rho_th^2
 * (strict, algorithm line 7 PAPER.md:527).  Sets resolved[i] = 1, appends i to sel (ascending
 * i), writes rho2_out[i] for every tested source (if non-NULL; untested entries untouched),
 * counts sources with |rho2 / rho_th^2 - 1| <= 2e-9 into *near.  Returns the number selected. */
int64_t orc_snr_select(const orc_grid *g, const double *A, const double *f, const double *fdot,
                       int64_t n, const double *psd, double rho_th, uint8_t *resolved,
                       double *rho2_out, int64_t *sel, int64_t *near)
{
    double thr = rho_th * rho_th;
    int64_t n_sel = 0, n_near = 0;
    for (int64_t i = 0; i < n; ++i) {
        if (resolved[i]) continue;
        double r2 = orc_rho2(g, A[i], f[i], fdot[i], psd);
        if (rho2_out) rho2_out[i] = r2;
        if (r2 != r2) continue;                    /* rejected source: never resolved */
        if (fabs(r2 / thr - 1.0) <= 2e-9) ++n_near;
        if (r2 > thr) { resolved[i] = 1; sel[n_sel++] = i; }
    }
    if (near) *near = n_near;
    return n_sel;
}

/* ------------------------------------------------------------------------------------ */
/* Stage (v) — the loop, algorithm steps 4-10, R6.          */
/* ------------------------------------------------------------------------------------ */

typedef struct {
    int32_t n_iter;
    int32_t converged;
    int64_t n_resolved;
    int64_t n_near_threshold;
} orc_iter_result;

/* Stopwatch around the three stage calls of the loop below (bench.py's cpu_baseline reports where the oracle's
 * time goes).  Measurement only: nothing here feeds back into a result.
 * [0] estimator passes (median or mean, + PSD), [1] SNR passes, [2] subtractions; seconds, accumulated per thread. */
static __thread double orc_stage_s[3];
static double orc_now(void)
{
    struct timespec ts;
    clock_gettime(CLOCK_MONOTONIC, &ts);
    return (double)ts.tv_sec + 1e-9 * (double)ts.tv_nsec;
}
void orc_stage_seconds(double out[3], int reset)
{
    for (int i = 0; i < 3; ++i) { out[i] = orc_stage_s[i]; if (reset) orc_stage_s[i] = 0.0; }
}

/* spectrum: in = total deposited spectrum, out = residual.  resolved: in/out flags.
 * n_new_per_iter (nullable, length max_iter) receives the newly-resolved count of each
 * iteration.  median / psd always correspond to the returned residual. */
static int orc_estimate(int estimator, const int64_t *spectrum, const double *s_instr, int64_t n_bins,
                        int32_t window, double median_norm, int32_t scale_log2, int64_t *stat, double *psd)
{
    int rc;
    if (estimator == 1) {                      /* running mean, eq. (D1): stat = window sums */
        rc = orc_running_sum(spectrum, n_bins, window, stat);
        if (rc == 0) orc_psd_mean(stat, s_instr, n_bins, window, scale_log2, psd);
    } else {                                   /* running median, eq. (D2)-(D3) */
        rc = orc_running_median(spectrum, n_bins, window, stat);
        if (rc == 0) orc_psd(stat, s_instr, n_bins, median_norm, scale_log2, psd);
    }
    return rc;
}

/* estimator: 0 = running median (eqs. D2-D3), 1 = running mean (eq. D1; `median` receives the
 * window sums, median_norm is not used). */
/* psd_rtol > 0: the second stop rule of PAPER.md:530, 552, "convergence in S_n is reached" (R13): from the
 * second iteration on, delta = max_k |S_n^(i)[k] - S_n^(i-1)[k]| / S_n^(i-1)[k]; delta <= psd_rtol ends the loop
 * before that iteration's SNR test (converged = 2).  psd_rtol <= 0: the rule is off. */
int orc_subtract_until_converged_tol(const orc_grid *g, const double *A, const double *f,
                                 const double *fdot, int64_t n, const double *s_instr,
                                 int32_t window, double median_norm, double rho_th, int32_t max_iter,
                                 int32_t estimator, double psd_rtol,
                                 int64_t *spectrum, int64_t *median, double *psd, uint8_t *resolved,
                                 orc_iter_result *res, int64_t *n_new_per_iter)
{
    int64_t *sel = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n > 0 ? n : 1));
    double *prev = (double *)malloc(sizeof(double) * (size_t)g->n_bins);
    res->n_iter = 0; res->converged = 0; res->n_resolved = 0; res->n_near_threshold = 0;
    int rc = 0;
    int32_t it;
    for (it = 0; it < max_iter; ++it) {
        double t0 = orc_now();
        rc = orc_estimate(estimator, spectrum, s_instr, g->n_bins, window, median_norm, g->scale_log2, median, psd);
        orc_stage_s[0] += orc_now() - t0;
        if (rc) break;
        if (psd_rtol > 0.0 && it > 0) {
            double delta = 0.0;
            for (int64_t k = 0; k < g->n_bins; ++k) {
                double d = fabs(psd[k] - prev[k]) / prev[k];
                if (d > delta) delta = d;
            }
            if (delta <= psd_rtol) {
                if (n_new_per_iter) n_new_per_iter[it] = 0;
                res->n_iter = it + 1; res->converged = 2;
                break;
            }
        }
        if (psd_rtol > 0.0) memcpy(prev, psd, sizeof(double) * (size_t)g->n_bins);
        int64_t near = 0;
        t0 = orc_now();
        int64_t n_new = orc_snr_select(g, A, f, fdot, n, psd, rho_th, resolved, NULL, sel, &near);
        orc_stage_s[1] += orc_now() - t0;
        res->n_near_threshold += near;
        if (n_new_per_iter) n_new_per_iter[it] = n_new;
        if (n_new == 0) { res->n_iter = it + 1; res->converged = 1; break; }
        t0 = orc_now();
        orc_deposit(g, A, f, fdot, n, sel, n_new, -1, spectrum);
        orc_stage_s[2] += orc_now() - t0;
        res->n_resolved += n_new;
    }
    if (rc == 0 && !res->converged) {          /* cap hit: PSD must match the returned residual */
        res->n_iter = max_iter;
        double t0 = orc_now();
        rc = orc_estimate(estimator, spectrum, s_instr, g->n_bins, window, median_norm, g->scale_log2, median, psd);
        orc_stage_s[0] += orc_now() - t0;
    }
    free(sel);
    free(prev);
    return rc;
}

int orc_subtract_until_converged_est(const orc_grid *g, const double *A, const double *f,
                                 const double *fdot, int64_t n, const double *s_instr,
                                 int32_t window, double median_norm, double rho_th, int32_t max_iter,
                                 int32_t estimator,
                                 int64_t *spectrum, int64_t *median, double *psd, uint8_t *resolved,
                                 orc_iter_result *res, int64_t *n_new_per_iter)
{
    return orc_subtract_until_converged_tol(g, A, f, fdot, n, s_instr, window, median_norm, rho_th, max_iter, estimator, 0.0,
                                            spectrum, median, psd, resolved, res, n_new_per_iter);
}

int orc_subtract_until_converged(const orc_grid *g, const double *A, const double *f,
                                 const double *fdot, int64_t n, const double *s_instr,
                                 int32_t window, double median_norm, double rho_th, int32_t max_iter,
                                 int64_t *spectrum, int64_t *median, double *psd, uint8_t *resolved,
                                 orc_iter_result *res, int64_t *n_new_per_iter)
{
    return orc_subtract_until_converged_est(g, A, f, fdot, n, s_instr, window, median_norm, rho_th, max_iter, 0,
                                            spectrum, median, psd, resolved, res, n_new_per_iter);
}
