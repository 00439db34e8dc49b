// chirp.cuh -- SURVEY.md 8(f)-3: waveform generation on the device, fused with the projection (step i of P:408).
//
// The chirp + ringdown MODEL (the input recipe of BASELINE.json configs 1-4; leading-order chirp of
// the order of Eq. (4.2), damped-sinusoid ringdown) with parameters (ltdi_chirp), tau = t_c - t:
//   inspiral (tau > tau_cut):  Phi = phi_c - 2 (tau / 5 Mc)^(5/8),   amp = 4 (Mc c / d_L)(5 Mc / (256 tau))^(1/4)
//   ringdown (x = tau_cut - tau >= 0):  Phi = Phi(tau_cut) + 2 pi [f_rd x - (f_rd - f_cut) tau_rd (1 - e^(-x / tau_rd))],
//                                       amp = amp(tau_cut) e^(-x / tau_rd)
//   h+ = amp (1 + cos^2 iota) / 2 cos Phi,   hx = amp cos iota sin Phi.
//
// Precision.  A year of inspiral is Phi ~ 1e5 .. 1e6 rad: in plain fp64 the phase alone would carry 1e-11 rad of white
// noise, which the differences of the response amplify beyond the 1e-11 parity bar.  The phase is therefore evaluated
// in double-double: tau = (t_c - t0) - (n dt - delta) in dd, u^(5/8) = (u^(1/8))^5 with three dd square roots (no log /
// exp needed), reduction by multiples of pi / 2 in dd, then the fp64 sincos of the reduced angle with its low part as a
// first-order correction.  The amplitude and the ringdown terms are smooth factors: plain fp64.
#pragma once
#include "common.cuh"
#include "dd.cuh"

#define LTDI_CHIRP_STRIDE 20   /* doubles per source in the workspace */

struct ChirpDev {
    dd tc0;          /* t_c - t0 [s] */
    dd inv5mc;       /* 1 / (5 Mc) [1/s] */
    dd phi_cut;      /* phi_c - 2 (tau_cut / 5 Mc)^(5/8) */
    double phi_c;
    double amp0;     /* 4 (Mc c / d_L)(5 Mc / 256)^(1/4): amp = amp0 tau^(-1/4) */
    double amp_cut;  /* amp0 tau_cut^(-1/4) */
    double ap, ac;   /* (1 + cos^2 iota) / 2, cos iota */
    double tau_cut, inv_tau_rd, f_rd, c_rd;   /* c_rd = (f_rd - f_cut) tau_rd */
    double pad[5];
};
static_assert(sizeof(ChirpDev) == LTDI_CHIRP_STRIDE * sizeof(double), "ChirpDev layout");

// host: derived constants in long double
inline int chirp_fill(const ltdi_chirp &w, double t0, ChirpDev *out)
{
    if (!(w.mc_s > 0.0) || !(w.dist_m > 0.0) || !(w.tau_cut > 0.0) || !(w.tau_rd > 0.0) || !(w.f_rd > 0.0)) return LTDI_EINVAL;
    auto split = [](long double v) { dd r; r.hi = (double)v; r.lo = (double)(v - (long double)r.hi); return r; };
    const long double pi_l = 3.14159265358979323846264338327950288L;
    const long double mc = w.mc_s;
    ChirpDev c = {};
    c.tc0 = split((long double)w.t_c - (long double)t0);
    c.inv5mc = split(1.0L / (5.0L * mc));
    c.phi_cut = split((long double)w.phi_c - 2.0L * powl((long double)w.tau_cut / (5.0L * mc), 0.625L));
    c.phi_c = w.phi_c;
    c.amp0 = (double)(4.0L * (mc * (long double)LTDI_C_LIGHT / (long double)w.dist_m) * powl(5.0L * mc / 256.0L, 0.25L));
    c.amp_cut = (double)((long double)c.amp0 * powl((long double)w.tau_cut, -0.25L));
    c.ap = 0.5 * (1.0 + w.cos_iota * w.cos_iota);
    c.ac = w.cos_iota;
    c.tau_cut = w.tau_cut;
    c.inv_tau_rd = 1.0 / w.tau_rd;
    c.f_rd = w.f_rd;
    const long double f_cut = (1.0L / pi_l) * powl(5.0L / (256.0L * (long double)w.tau_cut), 0.375L) * powl(mc, -0.625L);
    c.c_rd = (double)(((long double)w.f_rd - f_cut) * (long double)w.tau_rd);
    *out = c;
    return LTDI_OK;
}

// sin and cos of a dd angle of any size met here (|a| < 1e9): reduction by multiples of pi / 2 with a three-part
// constant in dd, fp64 sincos of the reduced high part, first-order correction by the low part
__device__ __forceinline__ void sincos_ddarg(dd a, double &s, double &c)
{
    const double P1 = 1.570796326794896558e+00, P2 = 6.123233995736766036e-17, P3 = -1.497384904859169833e-33;
    const double k = rint(a.hi * 0.63661977236758134308);
    dd r = dd_sub(a, two_prod(k, P1));
    r = dd_sub(r, two_prod(k, P2));
    r = dd_add_d(r, -k * P3);
    double sh, ch;
    sincos(r.hi, &sh, &ch);
    const double ss = fma(r.lo, ch, sh), cc = fma(-r.lo, sh, ch);
    switch (((long long)k) & 3) {
    case 0: s = ss; c = cc; break;
    case 1: s = cc; c = -ss; break;
    case 2: s = -ss; c = -cc; break;
    default: s = -cc; c = ss; break;
    }
}

// h+, hx of source w at time t0 + s (s in dd)
__device__ __forceinline__ void chirp_eval(const ChirpDev &w, dd s, double &hp, double &hc)
{
    const dd tau = dd_sub(w.tc0, s);
    dd phase;
    double amp;
    const double x = (w.tau_cut - tau.hi) - tau.lo;   /* time after the join */
    if (x <= 0.0) {
        const dd u = dd_mul(tau, w.inv5mc);
        const dd r = dd_sqrt(dd_sqrt(dd_sqrt(u)));     /* u^(1/8) */
        const dd r2 = dd_mul(r, r);
        dd r5 = dd_mul(dd_mul(r2, r2), r);             /* u^(5/8) */
        r5.hi *= -2.0; r5.lo *= -2.0;
        phase = dd_add_d(r5, w.phi_c);
        amp = w.amp0 * rsqrt(sqrt(tau.hi));
    } else {
        const double e1 = expm1(-x * w.inv_tau_rd);   /* decay - 1 */
        phase = dd_add_d(w.phi_cut, 6.283185307179586477 * fma(w.f_rd, x, w.c_rd * e1));
        amp = w.amp_cut * (1.0 + e1);
    }
    double sn, cs;
    sincos_ddarg(phase, sn, cs);
    hp = amp * w.ap * cs;
    hc = amp * w.ac * sn;
}

// the model sampled on the grid: one thread per sample, blockIdx.y = source
__global__ void __launch_bounds__(256) chirp_grid_kernel(const ChirpDev *__restrict__ wav, double dt, int64_t n, int64_t ld,
                                                         double *__restrict__ hp, double *__restrict__ hc)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int64_t b = blockIdx.y;
    double a, c;
    chirp_eval(wav[b], two_prod((double)i, dt), a, c);
    hp[b * ld + i] = a;
    hc[b * ld + i] = c;
}

// ---------------------------------------------------------------------------------------------------------------------
// The harmonic-sum waveform of an eccentric inspiral (config 5's recipe as a model; oracle O13b): orbital evolution table
// [7][nk] (t, F, e, l, dF/dt, de/dt, dl/dt at the knots) carried to the sample time by cubic Hermite interpolation, then
// Peters-Mathews harmonics n = 1 .. nharm (Barack & Cutler 2004, Eqs. 7-9).  The mean anomaly l reaches 1e3 .. 1e5 rad:
// the sample time is formed in double-double, l = l_k + (Hermite increment) is kept as a double-double sum and reduced
// like the chirp phase; cos / sin (n l) by rotation.  Bessel functions: J_{n+2}, J_{n+1} by their power series (the
// highest orders converge fastest), the three below by the downward recurrence (stable in that direction).
// ---------------------------------------------------------------------------------------------------------------------
#define LTDI_ECC_STRIDE 8
#define LTDI_ECC_MAXHARM 16

struct EccDev { double M, amp, ci, c2g, s2g, l0, pad0, pad1; };   /* amp = (2 pi M)^(2/3) eta M c / d_L */

inline int ecc_fill(const double *par /* M, eta, d_L, cos iota, gamma, l0 */, EccDev *out)
{
    if (!(par[0] > 0.0) || !(par[1] > 0.0) || !(par[2] > 0.0)) return LTDI_EINVAL;
    const long double pi_l = 3.14159265358979323846264338327950288L;
    EccDev c = {};
    c.M = par[0];
    c.amp = (double)(powl(2.0L * pi_l * (long double)par[0], 2.0L / 3.0L) * (long double)par[1] * (long double)par[0] *
                     (long double)LTDI_C_LIGHT / (long double)par[2]);
    c.ci = par[3];
    c.c2g = (double)cosl(2.0L * (long double)par[4]);
    c.s2g = (double)sinl(2.0L * (long double)par[4]);
    c.l0 = par[5];
    *out = c;
    return LTDI_OK;
}

/* 1 / j, j < 96: the term ratios of the series below without a division */
__constant__ double c_recip[96] = {0.0, 1.0 / 1.0, 1.0 / 2.0, 1.0 / 3.0, 1.0 / 4.0, 1.0 / 5.0, 1.0 / 6.0, 1.0 / 7.0, 1.0 / 8.0, 1.0 / 9.0, 1.0 / 10.0, 1.0 / 11.0, 1.0 / 12.0, 1.0 / 13.0, 1.0 / 14.0, 1.0 / 15.0, 1.0 / 16.0, 1.0 / 17.0, 1.0 / 18.0, 1.0 / 19.0, 1.0 / 20.0, 1.0 / 21.0, 1.0 / 22.0, 1.0 / 23.0, 1.0 / 24.0, 1.0 / 25.0, 1.0 / 26.0, 1.0 / 27.0, 1.0 / 28.0, 1.0 / 29.0, 1.0 / 30.0, 1.0 / 31.0, 1.0 / 32.0, 1.0 / 33.0, 1.0 / 34.0, 1.0 / 35.0, 1.0 / 36.0, 1.0 / 37.0, 1.0 / 38.0, 1.0 / 39.0, 1.0 / 40.0, 1.0 / 41.0, 1.0 / 42.0, 1.0 / 43.0, 1.0 / 44.0, 1.0 / 45.0, 1.0 / 46.0, 1.0 / 47.0, 1.0 / 48.0, 1.0 / 49.0, 1.0 / 50.0, 1.0 / 51.0, 1.0 / 52.0, 1.0 / 53.0, 1.0 / 54.0, 1.0 / 55.0, 1.0 / 56.0, 1.0 / 57.0, 1.0 / 58.0, 1.0 / 59.0, 1.0 / 60.0, 1.0 / 61.0, 1.0 / 62.0, 1.0 / 63.0, 1.0 / 64.0, 1.0 / 65.0, 1.0 / 66.0, 1.0 / 67.0, 1.0 / 68.0, 1.0 / 69.0, 1.0 / 70.0, 1.0 / 71.0, 1.0 / 72.0, 1.0 / 73.0, 1.0 / 74.0, 1.0 / 75.0, 1.0 / 76.0, 1.0 / 77.0, 1.0 / 78.0, 1.0 / 79.0, 1.0 / 80.0, 1.0 / 81.0, 1.0 / 82.0, 1.0 / 83.0, 1.0 / 84.0, 1.0 / 85.0, 1.0 / 86.0, 1.0 / 87.0, 1.0 / 88.0, 1.0 / 89.0, 1.0 / 90.0, 1.0 / 91.0, 1.0 / 92.0, 1.0 / 93.0, 1.0 / 94.0, 1.0 / 95.0};

/* J_k(x) and J_{k+1}(x) by their power series, 1 <= k <= 66, 0 <= x <= 8:
 * J_k = (x/2)^k / k! sum_m (-x^2/4)^m / (m! (k+1)_m); the sum stops where the terms fall below 1e-20 of its first */
__device__ __forceinline__ void bessel_pair(int k, double x, double &jk, double &jk1)
{
    const double q = -0.25 * x * x;
    double ta = 1.0, sa = 1.0, tb = 1.0, sb = 1.0;
#pragma unroll 1
    for (int m = 1; m <= 28; ++m) {
        const double qm = q * c_recip[m];
        ta *= qm * c_recip[k + m];
        tb *= qm * c_recip[k + 1 + m];
        sa += ta;
        sb += tb;
        if (fabs(ta) < 1e-20) break;      /* |tb| < |ta| */
    }
    double pre = 1.0;
    const double hx = 0.5 * x;
#pragma unroll 1
    for (int i = 1; i <= k; ++i) pre *= hx * c_recip[i];
    jk = pre * sa;
    jk1 = pre * hx * c_recip[k + 1] * sb;
}

__global__ void __launch_bounds__(128) ecc_grid_kernel(const double *__restrict__ tab, int64_t nk, const EccDev *__restrict__ wav,
                                                       int nharm, double t0, double dt, int64_t n, int64_t ld,
                                                       double *__restrict__ hp, double *__restrict__ hc)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int64_t b = blockIdx.y;
    const EccDev w = wav[b];
    const double *tk = tab + b * 7 * nk;
    const dd t = dd_add_d(two_prod((double)i, dt), t0);
    int64_t lo = 0, hi = nk;                              /* first knot > t */
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (tk[mid] <= t.hi) lo = mid + 1; else hi = mid;
    }
    const int64_t idx = min(max(lo - 1, (int64_t)0), nk - 2);
    const double h = tk[idx + 1] - tk[idx];
    const double u = ((t.hi - tk[idx]) + t.lo) / h;
    const double um = 1.0 - u;
    const double h10 = u * um * um, h01 = u * u * (3.0 - 2.0 * u), h11 = u * u * (u - 1.0);
    auto herm_inc = [&](int row) {   /* value - y_k */
        const double *y = tk + row * nk, *dy = tk + (row + 3) * nk;
        return h01 * (y[idx + 1] - y[idx]) + h * (h10 * dy[idx] + h11 * dy[idx + 1]);
    };
    const double F = tk[nk + idx] + herm_inc(1);
    const double e = tk[2 * nk + idx] + herm_inc(2);
    const dd ell = dd_add_d(two_sum(tk[3 * nk + idx], herm_inc(3)), w.l0);
    double sl, cl;
    sincos_ddarg(ell, sl, cl);
    const double A = w.amp * cbrt(F * F);
    const double sq = sqrt(1.0 - e * e), ci2 = w.ci * w.ci;
    double cn = 1.0, sn = 0.0, sp = 0.0, sc = 0.0;
#pragma unroll 1
    for (int k = 1; k <= nharm; ++k) {
        const double c2 = cn * cl - sn * sl, s2 = sn * cl + cn * sl;   /* cos, sin (k l) */
        cn = c2; sn = s2;
        const double x = (double)k * e;
        double jp2, jp1, j0, jm1, jm2;
        if (x < 1e-8) {   /* J_m(x) -> (x/2)^m / m!: only orders 0 and 1 matter at this level */
            jp2 = 0.0; jp1 = 0.0;
            j0 = 0.0; jm1 = k == 1 ? 1.0 : (k == 2 ? 0.5 * x : 0.0); jm2 = k == 2 ? 1.0 : (k == 1 ? -0.5 * x : (k == 3 ? 0.5 * x : 0.0));
            if (k == 1) j0 = 0.5 * x;
        } else {
            bessel_pair(k + 1, x, jp1, jp2);
            const double ix = 2.0 / x;
            j0 = (double)(k + 1) * ix * jp1 - jp2;            /* J_{m-1} = (2 m / x) J_m - J_{m+1} */
            jm1 = (double)k * ix * j0 - jp1;
            jm2 = (double)(k - 1) * ix * jm1 - j0;             /* k = 1: J_{-1} = -J_1 comes out of the recurrence */
        }
        const double an = -(double)k * A * (jm2 - 2.0 * e * jm1 + (2.0 / (double)k) * j0 + 2.0 * e * jp1 - jp2) * cn;
        const double bn = -(double)k * A * sq * (jm2 - 2.0 * j0 + jp2) * sn;
        const double cc = 2.0 * A * j0 * cn;
        sp += -(1.0 + ci2) * (an * w.c2g - bn * w.s2g) + (1.0 - ci2) * cc;
        sc += 2.0 * w.ci * (bn * w.c2g + an * w.s2g);
    }
    hp[b * ld + i] = sp;
    hc[b * ld + i] = sc;
}
