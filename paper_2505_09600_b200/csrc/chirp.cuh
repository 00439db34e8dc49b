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
