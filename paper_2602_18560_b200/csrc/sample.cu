// sample.cu — stage (i): Philox4x32-10 catalog sampling, and the instrument-noise helper.
//
// Follows DESIGN.md R1 (counter layout, draws) and §4 (elementary functions, operation by
// operation).  The kernel is ALU-bound (two Philox blocks + 2 log + 3 exp10 + sincos + sqrt per
// source against 24 bytes written); two sources per thread so that every store is 128 bits wide.
#include <string.h>

#include "gbfg_common.cuh"

namespace gbfg {

// ------------------------------------------------------------------------------ DESIGN.md §4
#define GB_SQRT_HALF 0.7071067811865476
#define GB_LN2_HI 0.6931471803691238
#define GB_LN2_LO 1.9082149292705877e-10
#define GB_LOG10_E 0.4342944819032518
#define GB_LN10 2.302585092994046
#define GB_LOG2_10 3.321928094887362
#define GB_LOG10_2_HI 0.3010299955494702
#define GB_LOG10_2_LO 1.1451100898021838e-10
#define GB_PIO2 1.5707963267948966
#define GB_PIO2_HI 1.5707963267341256
#define GB_PIO2_LO 6.077100506506192e-11
#define GB_TWO_OVER_PI 0.6366197723675814
#define GB_TWO_PI 6.283185307179586
#define GB_LOG10_K 2.6090342225545732      /* log10((96/5) pi^(8/3)), eq. (4) */
#define GB_LOG10_TSUN -5.3075504747653498  /* log10(G Msun / c^3 / 1 s) */

__host__ __device__ inline double det_log(double x)
{
    int e;
    double m = frexp(x, &e);
    if (m < GB_SQRT_HALF) { m = 2.0 * m; e -= 1; }
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
    double lm = fma(t * z, q, t);
    double de = (double)e;
    return de * GB_LN2_HI + fma(de, GB_LN2_LO, lm);
}

__host__ __device__ inline double det_exp_small(double t)
{
    double p = 1.0 / 87178291200.0;
    p = fma(p, t, 1.0 / 6227020800.0);
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

__host__ __device__ inline double det_exp10(double y)
{
    double k = rint(y * GB_LOG2_10);
    double r = fma(-k, GB_LOG10_2_HI, y);
    r = fma(-k, GB_LOG10_2_LO, r);
    double t = r * GB_LN10;
    return ldexp(det_exp_small(t), (int)k);
}

__host__ __device__ inline void det_sincos_small(double phi, double &sn, double &cs)
{
    double z = phi * phi;
    double p = -1.0 / 121645100408832000.0;
    p = fma(p, z, 1.0 / 355687428096000.0);
    p = fma(p, z, -1.0 / 1307674368000.0);
    p = fma(p, z, 1.0 / 6227020800.0);
    p = fma(p, z, -1.0 / 39916800.0);
    p = fma(p, z, 1.0 / 362880.0);
    p = fma(p, z, -1.0 / 5040.0);
    p = fma(p, z, 1.0 / 120.0);
    p = fma(p, z, -1.0 / 6.0);
    sn = fma(phi * z, p, phi);
    double q = -1.0 / 6402373705728000.0;
    q = fma(q, z, 1.0 / 20922789888000.0);
    q = fma(q, z, -1.0 / 87178291200.0);
    q = fma(q, z, 1.0 / 479001600.0);
    q = fma(q, z, -1.0 / 3628800.0);
    q = fma(q, z, 1.0 / 40320.0);
    q = fma(q, z, -1.0 / 720.0);
    q = fma(q, z, 1.0 / 24.0);
    q = fma(q, z, -0.5);
    cs = fma(z, q, 1.0);
}

__host__ __device__ inline void det_quadrant(int quad, double sn, double cs, double &s_out, double &c_out)
{
    switch (quad & 3) {
    case 0: s_out = sn;  c_out = cs;  break;
    case 1: s_out = cs;  c_out = -sn; break;
    case 2: s_out = -sn; c_out = -cs; break;
    default: s_out = -cs; c_out = sn; break;
    }
}

__host__ __device__ inline void det_sincos2pi(double u, double &s_out, double &c_out)
{
    double t = 4.0 * u;
    double n = rint(t);
    double d = t - n;
    double sn, cs;
    det_sincos_small(d * GB_PIO2, sn, cs);
    det_quadrant((int)n, sn, cs, s_out, c_out);
}

__host__ __device__ inline void det_sincos(double x, double &s_out, double &c_out)
{
    double n = rint(x * GB_TWO_OVER_PI);
    double r = fma(-n, GB_PIO2_HI, x);
    r = fma(-n, GB_PIO2_LO, r);
    double sn, cs;
    det_sincos_small(r, sn, cs);
    det_quadrant((int)((long long)n & 3), sn, cs, s_out, c_out);
}

// ------------------------------------------------------------------------------ Philox4x32-10
struct U4 { uint32_t x, y, z, w; };

__device__ __forceinline__ U4 philox4x32_10(U4 c, uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        U4 n;
        n.x = hi1 ^ c.y ^ k0;
        n.y = lo1;
        n.z = hi0 ^ c.w ^ k1;
        n.w = lo0;
        c = n;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return c;
}

__device__ __forceinline__ double u01(uint32_t lo, uint32_t hi)
{
    uint64_t x = (((uint64_t)hi << 32) | (uint64_t)lo) >> 12;
    return ((double)x + 0.5) * 0x1p-52;
}

// Per-catalog constants (host-computed with the same det_* functions, R1).
struct PopDev {
    double c0, c1, c2;          // frequency draw
    int flat_in_log;
    double logA_offset, logA_sigma, logMc_mean, logMc_sigma;
    double f_min, f_max, f_top; // clamp
    int64_t n_src;              // sources this launch draws ...
    int64_t i_base;             // ... the first of which is source i_base of its catalog
    uint32_t cat_id, key0, key1;
};

__device__ __forceinline__ void draw_source(const PopDev &P, int64_t i_rel, double &A, double &f, double &fdot)
{
    const int64_t i = P.i_base + i_rel;
    U4 ctr;
    ctr.x = (uint32_t)i; ctr.y = (uint32_t)((uint64_t)i >> 32); ctr.z = 0u; ctr.w = P.cat_id;
    U4 b0 = philox4x32_10(ctr, P.key0, P.key1);
    ctr.z = 1u;
    U4 b1 = philox4x32_10(ctr, P.key0, P.key1);
    double u_f = u01(b0.x, b0.y);
    double u_1 = u01(b0.z, b0.w);
    double u_2 = u01(b1.x, b1.y);
    double lf;
    if (P.flat_in_log) {
        lf = P.c0 + u_f * P.c1;
    } else {
        double x = P.c0 + u_f * P.c1;
        lf = (det_log(x) * GB_LOG10_E) * P.c2;
    }
    double fi = det_exp10(lf);
    if (fi < P.f_min) fi = P.f_min;
    if (fi >= P.f_max) fi = P.f_top;
    double r = sqrt(-2.0 * det_log(u_1));
    double sn, cs;
    det_sincos2pi(u_2, sn, cs);
    double z_A = r * cs;
    double z_M = r * sn;
    double t1 = lf + 3.0;
    double t2 = (2.0 / 3.0) * t1;
    double t3 = P.logA_offset + t2;
    double t4 = P.logA_sigma * z_A;
    A = det_exp10(t3 + t4);
    double lmc = P.logMc_mean + P.logMc_sigma * z_M;
    double m1 = (5.0 / 3.0) * (GB_LOG10_TSUN + lmc);
    double m2 = (11.0 / 3.0) * lf;
    fdot = det_exp10((GB_LOG10_K + m1) + m2);
    f = fi;
}

// Two sources per thread, 128-bit stores.  Arrays are offset to the catalog's first source; the
// pair (2t, 2t+1) is aligned when that offset is even, else a scalar path handles the ends.
// DEPOSIT: stage (ii) in the same kernel (gbfg_simulate).  The sampling is bound by its arithmetic (two Philox
// blocks, 2 log, 3 exp10, sincos, sqrt per source) and leaves the memory pipes idle; the deposit is a handful of
// 64-bit reductions per source that a kernel of its own spends its time waiting for.  Drawn and deposited from the
// same registers, the reductions retire under the next source's arithmetic and the catalog is not read back.
struct DepositDev {
    GridDev g;
    int64_t *spectrum, *diff;       // the catalog's row
    int64_t *err_count;
    int *wide_flag;
    DepositMarks mk;
    int cat;
};

template <bool DEPOSIT>
__device__ __forceinline__ void deposit_drawn(const DepositDev &D, double a, double fr, double fd, int &rejected)
{
    if (!DEPOSIT) return;
    const SrcBins s = source_bins(D.g, a, fr, fd);
    if (s.status) { ++rejected; return; }
    if (s.q != 0) deposit_one(s, s.q, D.g.n_bins, D.cat, D.spectrum, D.diff, D.wide_flag, D.mk);
}

template <bool DEPOSIT>
__global__ void __launch_bounds__(256)
sample_kernel(PopDev P, double *__restrict__ A, double *__restrict__ f, double *__restrict__ fdot, int head, DepositDev D)
{
    int rejected = 0;
    // sources [0, head) (0 or 1 of them) are done by thread 0 scalar so that the pairs are 16-byte aligned
    int64_t n_pairs = (P.n_src - head) / 2;
    int64_t tail = head + 2 * n_pairs;
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t pr = t; pr < n_pairs; pr += stride) {
        int64_t i = head + 2 * pr;
        double a0, f0, d0, a1, f1, d1;
        draw_source(P, i, a0, f0, d0);
        draw_source(P, i + 1, a1, f1, d1);
        *reinterpret_cast<double2 *>(A + i) = make_double2(a0, a1);
        *reinterpret_cast<double2 *>(f + i) = make_double2(f0, f1);
        *reinterpret_cast<double2 *>(fdot + i) = make_double2(d0, d1);
        deposit_drawn<DEPOSIT>(D, a0, f0, d0, rejected);
        deposit_drawn<DEPOSIT>(D, a1, f1, d1, rejected);
    }
    if (t == 0) {
        for (int64_t i = 0; i < head; ++i) { draw_source(P, i, A[i], f[i], fdot[i]); deposit_drawn<DEPOSIT>(D, A[i], f[i], fdot[i], rejected); }
        for (int64_t i = tail; i < P.n_src; ++i) { draw_source(P, i, A[i], f[i], fdot[i]); deposit_drawn<DEPOSIT>(D, A[i], f[i], fdot[i], rejected); }
    }
    if (DEPOSIT && D.err_count) {
        for (int o = 16; o; o >>= 1) rejected += __shfl_down_sync(0xffffffffu, rejected, o);
        if ((threadIdx.x & 31) == 0 && rejected) atomic_add_i64(D.err_count, rejected);
    }
}

// Robson et al. 2019 curve at bin centres (R3)
__device__ __forceinline__ double robson_sn(double fq)
{
    const double L = 2.5e9, fstar = 19.09e-3;
    double r2 = 2.0e-3 / fq;  r2 = r2 * r2;
    double p_oms = (1.5e-11 * 1.5e-11) * (1.0 + r2 * r2);
    double r4 = 0.4e-3 / fq;
    double r8 = fq / 8.0e-3;  r8 = r8 * r8;
    double p_acc = (3.0e-15 * 3.0e-15) * (1.0 + r4 * r4) * (1.0 + r8 * r8);
    double x = fq / fstar;
    double sn, cs;
    det_sincos(x, sn, cs);
    double y = GB_TWO_PI * fq;  y = y * y;  y = y * y;
    double acc = 2.0 * (1.0 + cs * cs) * p_acc / y;
    return (10.0 / (3.0 * L * L)) * (p_oms + acc) * (1.0 + 0.6 * (x * x));
}

__global__ void __launch_bounds__(256)
instrument_noise_kernel(double f_min, double T, int64_t n_bins, double *__restrict__ s_instr)
{
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (; k < n_bins; k += stride) {
        double fk = f_min + ((double)k + 0.5) / T;
        s_instr[k] = robson_sn(fk);
    }
}

// ------------------------------------------------------------------------------ DESIGN.md R12
// The paper's own population sampler: Table I, eqs. (7)-(9), Gaussian copula (App. A).
#define GB_SQRT_PI 1.7724538509055159
#define GB_INV_SQRT2 0.7071067811865476

__host__ __device__ inline double det_expn(double y) { return det_exp10(y * GB_LOG10_E); }

// erfc(t), t >= 0: all-positive series below 2, continued fraction of depth 40 from the bottom above
__host__ __device__ inline double det_erfc_pos(double t)
{
    const double t2 = t * t;
    if (t < 2.0) {
        double term = t, sum = t;
        for (int n = 1; n < 80; ++n) {
            term = term * (2.0 * t2) / (double)(2 * n + 1);
            sum = sum + term;
        }
        return 1.0 - (2.0 / GB_SQRT_PI) * det_expn(-t2) * sum;
    }
    double r = t;
    for (int k = 40; k >= 1; --k) r = t + (0.5 * (double)k) / r;
    return det_expn(-t2) / (GB_SQRT_PI * r);
}

// Phi(z) for z <= 0, 1 - Phi(z) for z > 0
__host__ __device__ inline double det_norm_tail(double z)
{
    return 0.5 * det_erfc_pos(fabs(z) * GB_INV_SQRT2);
}

// P(a,x), Q(a,x), x^a e^-x / Gamma(a): series (48 terms) below a + 3, Legendre's continued fraction (depth 40) above
__host__ __device__ inline void det_gamma_pq(double a, double x, double lg, double &P, double &Q, double &pref)
{
    pref = det_expn((a * det_log(x) - x) - lg);
    if (x < a + 3.0) {
        double term = 1.0 / a, sum = term;
        for (int n = 1; n <= 48; ++n) {
            term = term * x / (a + (double)n);
            sum = sum + term;
        }
        P = sum * pref;
        Q = 1.0 - P;
    } else {
        double r = (x + 81.0) - a;
        for (int k = 40; k >= 1; --k) r = ((x + (double)(2 * k - 1)) - a) - ((double)k * ((double)k - a)) / r;
        Q = pref / r;
        P = 1.0 - Q;
    }
}

// x with P(a,x) = Phi(z): Wilson-Hilferty start, 10 Newton steps on the log of the tail probability on z's side
__host__ __device__ inline double det_gamma_quantile(double a, double lg, double lg1, double z)
{
    const double tail = det_norm_tail(z);
    const double c = 1.0 / (9.0 * a);
    const double w = (1.0 - c) + z * sqrt(c);
    double x = a * ((w * w) * w);
    if (!(w > 0.0) || x < 1e-6 * a) x = det_expn((det_log(tail) + lg1) / a);
    for (int it = 0; it < 10; ++it) {
        double P, Q, pref;
        det_gamma_pq(a, x, lg, P, Q, pref);
        const double pdf = pref / x;
        const double g = (z <= 0.0) ? P * det_log(P / tail) : -(Q * det_log(Q / tail));
        double xn = x - g / pdf;
        if (xn < 0.1 * x) xn = 0.1 * x;
        if (xn > 2.0 * x + 4.0) xn = 2.0 * x + 4.0;
        x = xn;
    }
    return x;
}

struct PopPaperDev {
    double c0, c1, c2;          // frequency draw
    int flat_in_log;
    double alpha_gamma, beta_gamma, mu_gamma, lg, lg1;
    double mu, sigma, rho, rho_c;
    double f_min, f_max, f_top;
    int64_t n_src;
    uint32_t cat_id, key0, key1;
};

__device__ __forceinline__ void draw_source_paper(const PopPaperDev &P, int64_t i, double &A, double &f, double &fdot)
{
    U4 ctr;
    ctr.x = (uint32_t)i; ctr.y = (uint32_t)((uint64_t)i >> 32); ctr.z = 2u; ctr.w = P.cat_id;
    const U4 b0 = philox4x32_10(ctr, P.key0, P.key1);
    ctr.z = 3u;
    const U4 b1 = philox4x32_10(ctr, P.key0, P.key1);
    const double u_1 = u01(b0.x, b0.y), u_2 = u01(b0.z, b0.w);
    const double u_3 = u01(b1.x, b1.y), u_4 = u01(b1.z, b1.w);
    const double r = sqrt(-2.0 * det_log(u_1));
    double sn, cs;
    det_sincos2pi(u_2, sn, cs);
    const double n1 = r * cs, n2 = r * sn;
    const double r3 = sqrt(-2.0 * det_log(u_3));
    double s3, c3;
    det_sincos2pi(u_4, s3, c3);
    const double z3 = r3 * c3;
    const double z1 = n1;
    const double z2 = P.rho * n1 + P.rho_c * n2;
    const double t1 = det_norm_tail(z1);
    const double uf = (z1 <= 0.0) ? t1 : 1.0 - t1;
    double lf;
    if (P.flat_in_log) {
        lf = P.c0 + uf * P.c1;
    } else {
        const double x = P.c0 + uf * P.c1;
        lf = (det_log(x) * GB_LOG10_E) * P.c2;
    }
    double fi = det_exp10(lf);
    if (fi < P.f_min) fi = P.f_min;
    if (fi >= P.f_max) fi = P.f_top;
    const double xg = det_gamma_quantile(P.alpha_gamma, P.lg, P.lg1, z2);
    fdot = det_exp10(P.mu_gamma + xg / P.beta_gamma);
    const double at = det_expn(P.sigma * z3);
    A = det_exp10((P.mu + at) + (2.0 / 3.0) * lf);
    f = fi;
}

__global__ void __launch_bounds__(128)
sample_paper_kernel(PopPaperDev P, double *__restrict__ A, double *__restrict__ f, double *__restrict__ fdot)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (; i < P.n_src; i += stride) {
        double a, fr, fd;
        draw_source_paper(P, i, a, fr, fd);
        A[i] = a; f[i] = fr; fdot[i] = fd;
    }
}

// SciRDv1 noise of the TDI channels and its rescaling by the response (R11; eqs. C1-C5
// PAPER.md:494-509, B2-B5 PAPER.md:475-487), operation by operation as R11 lists them.
struct AetOut { double s_aa, s_tt, sh_aa, sh_tt; };

__device__ __forceinline__ AetOut aet_noise(double fq, double P, double A, double L, int tdi2)
{
    const double c = 299792458.0;
    const double fstar = c / (GB_TWO_PI * L);
    const double x = fq / fstar;
    double sn, cs, sh, ch;
    det_sincos(x, sn, cs);
    det_sincos(0.5 * x, sh, ch);
    const double omc = 2.0 * (sh * sh);                       // 1 - cos x
    double k2 = GB_TWO_PI * fq / c;  k2 = k2 * k2;
    double r2 = 2.0e-3 / fq;  r2 = r2 * r2;
    const double a_oms = P * 1.0e-12;
    const double p_oms = (a_oms * a_oms) * (1.0 + r2 * r2) * k2;
    const double r4 = 0.4e-3 / fq;
    double r8 = fq / 8.0e-3;  r8 = r8 * r8;
    const double a_tm = A * 1.0e-15;
    double y = GB_TWO_PI * fq;  y = y * y;  y = y * y;
    const double p_tm = (a_tm * a_tm) * (1.0 + r4 * r4) * (1.0 + r8 * r8) / y * k2;
    const double s2 = sn * sn;
    double s_aa = 8.0 * s2 * (4.0 * (1.0 + cs + cs * cs) * p_tm + (2.0 + cs) * p_oms);
    double s_tt = 16.0 * s2 * (2.0 * (omc * omc) * p_tm + omc * p_oms);
    const double x2 = x * x;
    const double pre = 16.0 * s2 * x2;
    const double r_aa = pre * (0.45 / (1.0 + 0.7 * x2));
    const double x4 = x2 * x2;
    const double r_tt = pre * (0.45 * (x4 * x2) / (1.8e3 + 0.7 * (x4 * x4)));
    AetOut o;
    o.sh_aa = s_aa / r_aa;
    o.sh_tt = s_tt / r_tt;
    if (tdi2) {
        double s2x, c2x;
        det_sincos(2.0 * x, s2x, c2x);
        const double fac = 4.0 * (s2x * s2x);
        s_aa = fac * s_aa;
        s_tt = fac * s_tt;
    }
    o.s_aa = s_aa;
    o.s_tt = s_tt;
    return o;
}

__global__ void __launch_bounds__(256)
instrument_noise_aet_kernel(double f_min, double T, int64_t n_bins, double P, double A, double L, int tdi2,
                            double *__restrict__ s_aa, double *__restrict__ s_tt,
                            double *__restrict__ sh_aa, double *__restrict__ sh_tt)
{
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (; k < n_bins; k += stride) {
        const double fk = f_min + ((double)k + 0.5) / T;
        const AetOut o = aet_noise(fk, P, A, L, tdi2);
        if (s_aa) s_aa[k] = o.s_aa;
        if (s_tt) s_tt[k] = o.s_tt;
        if (sh_aa) sh_aa[k] = o.sh_aa;
        if (sh_tt) sh_tt[k] = o.sh_tt;
    }
}

// S_sum = 1 / ((2 / S_h^AA) + (1 / S_h^TT)): eq. (11) summed over A, E, T in the power domain (R14)
__global__ void __launch_bounds__(256)
channel_sum_noise_kernel(const double *__restrict__ sh_aa, const double *__restrict__ sh_tt, int64_t n, double *__restrict__ out)
{
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (; k < n; k += stride) {
        const double ta = 2.0 / sh_aa[k];
        const double tt = 1.0 / sh_tt[k];
        const double s = ta + tt;
        out[k] = 1.0 / s;
    }
}

}  // namespace gbfg

using namespace gbfg;

extern "C" int gbfg_channel_sum_noise(const double *dev_Sh_AA, const double *dev_Sh_TT, int64_t n_bins, double *dev_Sh_sum,
                                      void *stream)
{
    if (!dev_Sh_AA || !dev_Sh_TT || !dev_Sh_sum || n_bins < 1) return GBFG_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    int blocks = (int)((n_bins + 255) / 256);
    const int cap = sm_count() * 8;
    if (blocks > cap) blocks = cap;
    {
        LaunchTimer lt(K_NOISE, (cudaStream_t)stream);
        channel_sum_noise_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(dev_Sh_AA, dev_Sh_TT, n_bins, dev_Sh_sum);
    }
    GBFG_LAUNCH_CHECK("channel_sum_noise_kernel");
    return GBFG_OK;
}

extern "C" int gbfg_instrument_noise(const gbfg_grid *grid, double *dev_s_instr, void *stream)
{
    if (!grid || grid->struct_size != sizeof(gbfg_grid) || !dev_s_instr) return GBFG_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    int blocks = (int)((grid->n_bins + 255) / 256);
    int cap = sm_count() * 8;
    if (blocks > cap) blocks = cap;
    {
        LaunchTimer lt(K_NOISE, (cudaStream_t)stream);
        instrument_noise_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(grid->f_min, grid->t_obs, grid->n_bins, dev_s_instr);
    }
    GBFG_LAUNCH_CHECK("instrument_noise_kernel");
    return GBFG_OK;
}

extern "C" int gbfg_instrument_noise_aet(const gbfg_grid *grid, double P_pm, double A_fm, double L_m, int32_t tdi2,
                                         double *dev_S_AA, double *dev_S_TT, double *dev_Sh_AA, double *dev_Sh_TT,
                                         void *stream)
{
    if (!grid || grid->struct_size != sizeof(gbfg_grid)) return GBFG_ERR_INVALID_ARG;
    if (!(P_pm > 0.0) || !(A_fm > 0.0) || !(L_m > 0.0)) return GBFG_ERR_INVALID_ARG;
    if (!dev_S_AA && !dev_S_TT && !dev_Sh_AA && !dev_Sh_TT) return GBFG_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    int blocks = (int)((grid->n_bins + 255) / 256);
    int cap = sm_count() * 8;
    if (blocks > cap) blocks = cap;
    {
        LaunchTimer lt(K_NOISE, (cudaStream_t)stream);
        instrument_noise_aet_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(grid->f_min, grid->t_obs, grid->n_bins, P_pm, A_fm,
                                                                              L_m, tdi2 ? 1 : 0, dev_S_AA, dev_S_TT, dev_Sh_AA, dev_Sh_TT);
    }
    GBFG_LAUNCH_CHECK("instrument_noise_aet_kernel");
    return GBFG_OK;
}

// cat_ids (HOST [n_cat], nullable): Philox counter word 3 of catalog c; NULL: first_cat_id + c
int gbfg::sample_catalog_paper_ids(const gbfg_grid *grid, const gbfg_pop_paper *pops, const int64_t *offsets,
                                   int32_t n_cat, uint32_t first_cat_id, const uint32_t *cat_ids, uint64_t seed,
                                   double *dev_A, double *dev_f, double *dev_fdot, void *stream)
{
    if (!grid || grid->struct_size != sizeof(gbfg_grid) || !pops || !offsets) return GBFG_ERR_INVALID_ARG;
    if (n_cat < 1) return GBFG_ERR_INVALID_ARG;
    if (n_cat > GBFG_MAX_CAT) return GBFG_ERR_UNSUPPORTED;
    if (offsets[0] != 0) return GBFG_ERR_INVALID_ARG;
    for (int c = 0; c < n_cat; ++c) {
        const gbfg_pop_paper &p = pops[c];
        if (p.struct_size != sizeof(gbfg_pop_paper) || p.n_src < 0) return GBFG_ERR_INVALID_ARG;
        if (offsets[c + 1] - offsets[c] != p.n_src) return GBFG_ERR_INVALID_ARG;
        if (!(p.alpha_gamma > 0.0) || !(p.beta_gamma > 0.0) || !(p.sigma >= 0.0) || !(p.rho >= 0.0) || !(p.rho < 1.0))
            return GBFG_ERR_INVALID_ARG;
        // the fixed-length recurrences of DESIGN.md R12 are stated (and pinned) for this range; Table I draws alpha from [1, 3]
        if (p.alpha_gamma < GBFG_PAPER_ALPHA_MIN || p.alpha_gamma > GBFG_PAPER_ALPHA_MAX) return GBFG_ERR_UNSUPPORTED;
    }
    if (offsets[n_cat] > 0 && (!dev_A || !dev_f || !dev_fdot)) return GBFG_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    const double lfmin = det_log(grid->f_min) * GB_LOG10_E;
    const double lfmax = det_log(grid->f_max) * GB_LOG10_E;
    for (int c = 0; c < n_cat; ++c) {
        const gbfg_pop_paper &p = pops[c];
        if (p.n_src == 0) continue;
        PopPaperDev P;
        const double oms = 1.0 + p.alpha_pl;
        P.flat_in_log = fabs(oms) < 1e-12;
        if (P.flat_in_log) {
            P.c0 = lfmin; P.c1 = lfmax - lfmin; P.c2 = 1.0;
        } else {
            const double a = det_exp10(oms * lfmin);
            const double b = det_exp10(oms * lfmax);
            P.c0 = a; P.c1 = b - a; P.c2 = 1.0 / oms;
        }
        P.alpha_gamma = p.alpha_gamma; P.beta_gamma = p.beta_gamma; P.mu_gamma = p.mu_gamma;
        P.lg = lgamma(p.alpha_gamma); P.lg1 = lgamma(p.alpha_gamma + 1.0);
        P.mu = p.mu; P.sigma = p.sigma; P.rho = p.rho; P.rho_c = sqrt(1.0 - p.rho * p.rho);
        P.f_min = grid->f_min; P.f_max = grid->f_max; P.f_top = nextafter(grid->f_max, 0.0);
        P.n_src = p.n_src;
        P.cat_id = cat_ids ? cat_ids[c] : first_cat_id + (uint32_t)c;
        P.key0 = (uint32_t)seed; P.key1 = (uint32_t)(seed >> 32);
        int64_t blocks = (p.n_src + 127) / 128;
        const int64_t cap = (int64_t)sm_count() * 16;
        if (blocks > cap) blocks = cap;
        {
            LaunchTimer lt(K_SAMPLE, (cudaStream_t)stream);
            sample_paper_kernel<<<(int)blocks, 128, 0, (cudaStream_t)stream>>>(P, dev_A + offsets[c], dev_f + offsets[c],
                                                                              dev_fdot + offsets[c]);
        }
        GBFG_LAUNCH_CHECK("sample_paper_kernel");
    }
    return GBFG_OK;
}

extern "C" int gbfg_sample_catalog_paper(const gbfg_grid *grid, const gbfg_pop_paper *pops, const int64_t *offsets,
                                         int32_t n_cat, uint32_t first_cat_id, uint64_t seed,
                                         double *dev_A, double *dev_f, double *dev_fdot, void *stream)
{
    return sample_catalog_paper_ids(grid, pops, offsets, n_cat, first_cat_id, nullptr, seed, dev_A, dev_f, dev_fdot, stream);
}

// cat_ids (HOST [n_cat], nullable): Philox counter word 3 of catalog c; NULL: first_cat_id + c
int gbfg::sample_catalog_ids(const gbfg_grid *grid, const gbfg_pop *pops, const int64_t *offsets,
                             int32_t n_cat, uint32_t first_cat_id, const uint32_t *cat_ids, uint64_t seed,
                             double *dev_A, double *dev_f, double *dev_fdot, void *stream, const SampleDeposit *dep)
{
    if (!grid || grid->struct_size != sizeof(gbfg_grid) || !pops || !offsets) return GBFG_ERR_INVALID_ARG;
    if (n_cat < 1) return GBFG_ERR_INVALID_ARG;
    if (n_cat > GBFG_MAX_CAT) return GBFG_ERR_UNSUPPORTED;
    if (offsets[0] != 0) return GBFG_ERR_INVALID_ARG;
    for (int c = 0; c < n_cat; ++c) {
        if (pops[c].struct_size != sizeof(gbfg_pop) || pops[c].n_src < 0) return GBFG_ERR_INVALID_ARG;
        if (offsets[c + 1] - offsets[c] != pops[c].n_src) return GBFG_ERR_INVALID_ARG;
    }
    if (offsets[n_cat] > 0 && (!dev_A || !dev_f || !dev_fdot)) return GBFG_ERR_INVALID_ARG;
    if (((uintptr_t)dev_A | (uintptr_t)dev_f | (uintptr_t)dev_fdot) & 15) return GBFG_ERR_INVALID_ARG;
    int rc = check_device();
    if (rc) return rc;
    const double lfmin = det_log(grid->f_min) * GB_LOG10_E;
    const double lfmax = det_log(grid->f_max) * GB_LOG10_E;
    for (int c = 0; c < n_cat; ++c) {
        const gbfg_pop &p = pops[c];
        if (p.n_src == 0) continue;
        PopDev P;
        double oms = 1.0 - p.slope;
        P.flat_in_log = fabs(oms) < 1e-12;
        if (P.flat_in_log) {
            P.c0 = lfmin; P.c1 = lfmax - lfmin; P.c2 = 1.0;
        } else {
            double a = det_exp10(oms * lfmin);
            double b = det_exp10(oms * lfmax);
            P.c0 = a; P.c1 = b - a; P.c2 = 1.0 / oms;
        }
        P.logA_offset = p.logA_offset; P.logA_sigma = p.logA_sigma;
        P.logMc_mean = p.logMc_mean; P.logMc_sigma = p.logMc_sigma;
        P.f_min = grid->f_min; P.f_max = grid->f_max; P.f_top = nextafter(grid->f_max, 0.0);
        P.n_src = p.n_src;
        P.cat_id = cat_ids ? cat_ids[c] : first_cat_id + (uint32_t)c;
        P.key0 = (uint32_t)seed; P.key1 = (uint32_t)(seed >> 32);
        DepositDev D;
        memset(&D, 0, sizeof(D));
        if (dep) {
            D.g = make_grid_dev(grid);
            D.spectrum = dep->spectrum + (int64_t)c * grid->n_bins;
            D.diff = dep->diff + (int64_t)c * grid->n_bins;
            D.err_count = dep->err_count; D.wide_flag = dep->wide_flag; D.mk = dep->mk; D.cat = c;
        }
        // pieces of at most `piece` sources (even, so that the pairs of every piece stay 16-byte aligned); after each
        // piece the caller is told which sources of the batch are now on their way (gbfg_simulate builds their
        // candidate records next to the drawing of the following piece)
        int64_t piece = p.n_src;
        if (dep && dep->piece > 0 && dep->piece < piece) piece = dep->piece & ~(int64_t)1;
        for (int64_t i0 = 0; i0 < p.n_src; i0 += piece) {
            const int64_t cnt = p.n_src - i0 < piece ? p.n_src - i0 : piece;
            P.n_src = cnt;
            P.i_base = i0;
            int head = (int)((offsets[c] + i0) & 1);          // keep the pairs 16-byte aligned
            if (head > cnt) head = (int)cnt;
            int64_t n_pairs = (cnt - head) / 2;
            int64_t blocks = (n_pairs + 255) / 256;
            if (blocks < 1) blocks = 1;
            int64_t cap = (int64_t)sm_count() * 16;
            if (blocks > cap) blocks = cap;
            double *pA = dev_A + offsets[c] + i0, *pf = dev_f + offsets[c] + i0, *pd = dev_fdot + offsets[c] + i0;
            {
                LaunchTimer lt(K_SAMPLE, (cudaStream_t)stream);
                if (dep) sample_kernel<true><<<(int)blocks, 256, 0, (cudaStream_t)stream>>>(P, pA, pf, pd, head, D);
                else sample_kernel<false><<<(int)blocks, 256, 0, (cudaStream_t)stream>>>(P, pA, pf, pd, head, D);
            }
            GBFG_LAUNCH_CHECK("sample_kernel");
            if (dep && dep->after_piece) {
                const int rc2 = dep->after_piece(dep->ctx, offsets[c] + i0, offsets[c] + i0 + cnt);
                if (rc2) return rc2;
            }
        }
    }
    return GBFG_OK;
}

extern "C" int gbfg_sample_catalog(const gbfg_grid *grid, const gbfg_pop *pops, const int64_t *offsets,
                                   int32_t n_cat, uint32_t first_cat_id, uint64_t seed,
                                   double *dev_A, double *dev_f, double *dev_fdot, void *stream)
{
    return sample_catalog_ids(grid, pops, offsets, n_cat, first_cat_id, nullptr, seed, dev_A, dev_f, dev_fdot, stream);
}
