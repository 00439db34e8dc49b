// orbit.cuh -- S0: orbit / delay kernel (first-order Keplerian orbits, G5-G7).
//
// One thread per time sample writes the table rows of its sample: spacecraft positions R_i(t_n) [m], link unit
// vectors n_l(t_n) for l = +1,+2,+3 (sender -> receiver; n_-l = -n_l) and the six light travel times
// L_l(t_n) [s] as doubles (24 rows), plus the LOW PARTS of n_l and L_l as floats (15 rows): n_l and L_l are
// computed in double-double arithmetic (dd.cuh) and stored as hi + lo.
//
// Why double-double.  n_l = (R_r - R_s) / |R_r - R_s| from positions rounded to fp64 (1.5e11 m +- 2e-5 m, arms of
// 2.5e9 m) carries white noise of 1e-14; the gen-2.0 LFA, Eq. (B33), differences the link series twice and
// amplifies it to 4e-10 in X at config 3 (measured: the oracle's own double build sits there).  Here the arm
// vectors are formed analytically -- the R cos(alpha) terms of the two spacecraft cancel in exact arithmetic, what
// remains is O(e R) = O(L) -- from sin / cos of the orbital phase evaluated in dd (phase alpha = Omega t_n + alpha0
// in dd: t_n = t0 + n dt rounded to fp64 alone would move n_l by 7e-16 at t = 1 yr).  The positions themselves enter
// the response only through k.R / c (needed to 1e-13 s): they are stored as correctly rounded doubles.
//
// Cost: the kernel is bound by the FP64 pipe, not by HBM (252 B written per sample), and runs once per time grid; the
// analytic modes form the unit vectors of the rigid triangle directly (no norm, no division).
#pragma once
#include "common.cuh"
#include "dd.cuh"

struct OrbitKernelParams {
    double t0, dt;
    int64_t n, stride;
    double arm_m, R_m, omega, alpha0;
    dd omega_dd;           /* 2 pi / period */
    dd sb[3], cb[3];       /* sin, cos of beta_i = 2 pi i / 3 + rot0 */
    dd half_eR, s3_eR;     /* e R / 2 and sqrt(3) e R [m], e = L / (2 sqrt(3) R) */
    dd inv_c;              /* 1 / c */
    dd L_static;           /* arm / c */
    /* analytic orbits: coefficients of the unit vector of link l in (cos 2 alpha, sin 2 alpha, cos alpha, sin alpha):
     * PA = (e R / 2)(cos beta_r - cos beta_s) / L, PB = the same with sin, PA3 = 3 PA, PB3 = 3 PB, PC = sqrt(3) e R (cos beta_r -
     * cos beta_s) / L, PD with sin */
    dd PA[3], PB[3], PA3[3], PB3[3], PC[3], PD[3];
    dd sin_c[11], cos_c[12]; /* (-1)^m / (2m+1)!, (-1)^m / (2m)! */
    int mode;
    const double *R_in; /* tables mode: [3][3][n]; knots mode: [3][3][nk] */
    const double *L_in; /* tables mode: [6][n] */
    /* knots mode (numerical orbit files): knot j at time tk0 + j dtk, Lagrange order korder */
    int64_t nk;
    double tk0, dtk;
    dd inv_dtk;
    int korder;
    double *tab;
};

// Lagrange weights w_k(u) and their first derivative, k = -(M/2-1) .. M/2, M <= 16 (prefix x suffix products with the
// product rule carried along; denominators from c_lag_inv_den)
__device__ __forceinline__ void knot_weights(double u, int M, double *w, double *dw)
{
    const double *c = c_lag_inv_den + (M / 2 - 1) * LTDI_MAX_TAPS;
    const int kmin = -(M / 2 - 1);
    double pf[16], pf1[16];
    double f = 1.0, f1 = 0.0;
    for (int i = 0; i < M; ++i) {
        pf[i] = f; pf1[i] = f1;
        const double e = u - (double)(kmin + i);
        f1 = f1 * e + f;
        f = f * e;
    }
    double g = 1.0, g1 = 0.0;
    for (int i = M - 1; i >= 0; --i) {
        w[i] = c[i] * (pf[i] * g);
        dw[i] = c[i] * (pf1[i] * g + pf[i] * g1);
        const double e = u - (double)(kmin + i);
        g1 = g1 * e + g;
        g = g * e;
    }
}

// sin and cos of a dd angle, absolute error < 1e-30 for |a| < 1e5: reduction by multiples of pi / 2 (three-part
// constant), Taylor series on |r| <= pi / 4 -- the high-order tail (terms below 1e-11) in plain fp64
__device__ __forceinline__ void sincos_dd(dd a, const OrbitKernelParams &p, dd &s, dd &c)
{
    const double P1 = 1.570796326794896558e+00, P2 = 6.123233995736766036e-17, P3 = -1.497384904859169833e-33;
    const double k = rint(a.hi * 0.63661977236758134308);
    dd r = dd_sub(a, two_prod(k, P1));
    r = dd_sub(r, two_prod(k, P2));
    r = dd_add_d(r, -k * P3);
    const dd r2 = dd_mul(r, r);
    /* sin r / r and cos r as polynomials in r^2 */
    double ts = p.sin_c[10].hi, tc = p.cos_c[11].hi;
#pragma unroll
    for (int m = 9; m >= 6; --m) ts = fma(ts, r2.hi, p.sin_c[m].hi);
#pragma unroll
    for (int m = 10; m >= 6; --m) tc = fma(tc, r2.hi, p.cos_c[m].hi);
    dd ps = dd_make(ts, 0.0), pc = dd_make(tc, 0.0);
#pragma unroll
    for (int m = 5; m >= 0; --m) {
        ps = dd_add_fast(dd_mul(ps, r2), p.sin_c[m]);   /* Horner steps: no cancellation */
        pc = dd_add_fast(dd_mul(pc, r2), p.cos_c[m]);
    }
    ps = dd_mul(ps, r);
    const int q = ((int)k) & 3;
    switch (q) {
    case 0: s = ps; c = pc; break;
    case 1: s = pc; c = dd_neg(ps); break;
    case 2: s = dd_neg(ps); c = dd_neg(pc); break;
    default: s = dd_neg(pc); c = ps; break;
    }
}

// KNOTS: the numerical-orbit instance (kept apart: its stencil arrays would cost the analytic modes registers)
template <bool KNOTS>
__global__ void __launch_bounds__(128) orbit_delay_kernel(const __grid_constant__ OrbitKernelParams p)
{
    const int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= p.n) return;
    double R[3][3], V[3][3];
    dd dv[3][3];   /* arm vectors R_r - R_s of links +1, +2, +3 [m] (tables, orbit files), or the unit vectors themselves (analytic orbits) */
    if (!KNOTS && p.mode == LTDI_ORBIT_TABLES) {
#pragma unroll
        for (int i = 0; i < 9; ++i) {
            R[i / 3][i % 3] = p.R_in[(int64_t)i * p.n + n];
            V[i / 3][i % 3] = 0.0;
        }
#pragma unroll
        for (int l = 0; l < 3; ++l) {
            const int s = link_sender(l), r = link_receiver(l);
#pragma unroll
            for (int a = 0; a < 3; ++a) dv[l][a] = two_sum(R[r][a], -R[s][a]);
        }
    } else if (KNOTS) {
        // Numerical orbit file (O11, G28): positions tabulated at knots, centred Lagrange interpolation of
        // order korder on the knot grid; velocities = derivative of the interpolant.  Position in the grid in dd
        // (t_n rounded to fp64 alone would move the arm vectors by 1e-6 m through the 500 m/s relative velocities).
        dd t = two_prod((double)n, p.dt);
        t = dd_add_d(t, p.t0);
        const dd sg = dd_mul(dd_add_d(t, -p.tk0), p.inv_dtk);
        double jf = floor(sg.hi);
        double u = (sg.hi - jf) + sg.lo;
        if (u < 0.0) { jf -= 1.0; u += 1.0; }
        if (u >= 1.0) { jf += 1.0; u -= 1.0; }
        const int M = p.korder + 1;
        const int64_t j0 = (int64_t)jf - (M / 2 - 1);     /* first knot of the stencil (host: 0 <= j0, j0 + M <= nk) */
        double w[16], dw[16];
        knot_weights(u, M, w, dw);
#pragma unroll
        for (int i = 0; i < 9; ++i) {
            const double *K = p.R_in + (int64_t)i * p.nk + j0;
            double acc = 0.0, dacc = 0.0;
            for (int m = 0; m < M; ++m) {
                acc = fma(w[m], K[m], acc);
                dacc = fma(dw[m], K[m], dacc);
            }
            R[i / 3][i % 3] = acc;
            V[i / 3][i % 3] = dacc / p.dtk;
        }
        // arm vectors: the knot differences D_m = K_r[m] - K_s[m] are formed without rounding (two_sum) and
        // interpolated about the central knot, d = D_c + sum_m w_m (D_m - D_c): the rounding of the weights then acts
        // on |D_m - D_c| ~ 1e8 m instead of on 2.5e9 m (weights sum to 1), which leaves 1e-8 m, 4e-18 of the arm
        const int mc = M / 2 - 1;
#pragma unroll
        for (int l = 0; l < 3; ++l) {
            const int s = link_sender(l), r = link_receiver(l);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const double *Kr = p.R_in + (int64_t)(3 * r + a) * p.nk + j0, *Ks = p.R_in + (int64_t)(3 * s + a) * p.nk + j0;
                const dd Dc = two_sum(Kr[mc], -Ks[mc]);
                double acc = 0.0;
                for (int m = 0; m < M; ++m) {
                    const dd Dm = two_sum(Kr[m], -Ks[m]);
                    acc = fma(w[m], (Dm.hi - Dc.hi) + (Dm.lo - Dc.lo), acc);
                }
                dv[l][a] = dd_add_d(Dc, acc);
            }
        }
    } else {
        // alpha(t) = Omega t + alpha0; spacecraft i: beta_i = 2 pi (i-1)/3 + rot0.  Positions to first order in the
        // eccentricity e = L / (2 sqrt(3) R): a rigid triangle of side L, cartwheeling at 1 AU.
        dd t = two_prod((double)n, p.dt);
        t = dd_add_d(t, p.t0);
        const dd alpha = dd_add_d(dd_mul(p.omega_dd, t), p.alpha0);
        dd sa, ca;
        sincos_dd(alpha, p, sa, ca);
        dd s2a = dd_mul(sa, ca);
        s2a.hi *= 2.0; s2a.lo *= 2.0;
        const dd c2a = dd_mul(dd_sub(ca, sa), dd_add(ca, sa));
        const dd Rc = dd_mul_d(ca, p.R_m), Rs = dd_mul_d(sa, p.R_m);
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            /* 2 alpha - beta_i and alpha - beta_i by the addition theorems.  The positions enter the response through k.R / c
             * only and are stored as doubles: the O(e R) terms in plain fp64 (1e-7 m), the R cos(alpha) term in dd */
            const double c2 = fma(c2a.hi, p.cb[i].hi, s2a.hi * p.sb[i].hi), s2 = fma(s2a.hi, p.cb[i].hi, -c2a.hi * p.sb[i].hi);
            const double c1 = fma(ca.hi, p.cb[i].hi, sa.hi * p.sb[i].hi), s1 = fma(sa.hi, p.cb[i].hi, -ca.hi * p.sb[i].hi);
            const double eR = 2.0 * p.half_eR.hi;
            R[i][0] = dd_to_double(dd_add_d(Rc, p.half_eR.hi * (c2 - 3.0 * p.cb[i].hi)));
            R[i][1] = dd_to_double(dd_add_d(Rs, p.half_eR.hi * (s2 - 3.0 * p.sb[i].hi)));
            R[i][2] = -p.s3_eR.hi * c1;
            V[i][0] = -p.R_m * p.omega * sa.hi - eR * p.omega * s2;
            V[i][1] = p.R_m * p.omega * ca.hi + eR * p.omega * c2;
            V[i][2] = p.s3_eR.hi * p.omega * s1;
        }
        /* The unit vectors directly.  In R_r - R_s the R cos(alpha), R sin(alpha) terms cancel identically and what is left
         * is linear in the DIFFERENCES cos beta_r - cos beta_s, sin beta_r - sin beta_s (host constants: no cancellation
         * between the two spacecraft on the device):
         *   d_x = (e R / 2) [cos 2a dcb + sin 2a dsb - 3 dcb],  d_y = (e R / 2) [sin 2a dcb - cos 2a dsb - 3 dsb],
         *   d_z = -sqrt(3) e R [cos a dcb + sin a dsb].
         * The first-order Keplerian constellation is a rigid triangle: with w = e^{-i beta_r} - e^{-i beta_s}, |w|^2 = 3,
         *   |d|^2 = (e R)^2 / 4 [30 - 6 Re(e^{2 i a} w^2)] + 3 (e R)^2 / 2 [3 + Re(e^{2 i a} w^2)] = 12 (e R)^2 = L^2
         * at every time, so n_l = d / L with 1 / L folded into the coefficients: neither the norm nor its reciprocal (a dd
         * square root and a dd division per link and sample) is needed; tables and orbit files need both. */
#pragma unroll
        for (int l = 0; l < 3; ++l) {
            /* sums of O(1) terms with an O(1) result, stored to 2^-77 (double + float): the 11-addition sum serves */
            dv[l][0] = dd_sub_fast(dd_add_fast(dd_mul(c2a, p.PA[l]), dd_mul(s2a, p.PB[l])), p.PA3[l]);
            dv[l][1] = dd_sub_fast(dd_sub_fast(dd_mul(s2a, p.PA[l]), dd_mul(c2a, p.PB[l])), p.PB3[l]);
            dv[l][2] = dd_neg(dd_add_fast(dd_mul(ca, p.PC[l]), dd_mul(sa, p.PD[l])));
        }
    }
    double *out = p.tab + n;
    float *lo = reinterpret_cast<float *>(p.tab + (int64_t)LTDI_TABLE_ROWS * p.stride) + n;
#pragma unroll
    for (int i = 0; i < 9; ++i) out[(int64_t)(ROW_R + i) * p.stride] = R[i / 3][i % 3];
#pragma unroll
    for (int l = 0; l < 3; ++l) {
        const int s = link_sender(l), r = link_receiver(l);
        const bool analytic = !KNOTS && p.mode != LTDI_ORBIT_TABLES;   /* dv holds the unit vector already */
        dd len = p.L_static, inv = dd_make(1.0, 0.0);                   /* analytic: len is not used */
        if (!analytic) {
            const dd len2 = dd_add(dd_add(dd_mul(dv[l][0], dv[l][0]), dd_mul(dv[l][1], dv[l][1])), dd_mul(dv[l][2], dv[l][2]));
            len = dd_sqrt(len2);
            inv = dd_div(dd_make(1.0, 0.0), len);
        }
        dd nh[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            nh[a] = analytic ? dv[l][a] : dd_mul(dv[l][a], inv);
            out[(int64_t)(ROW_N + 3 * l + a) * p.stride] = nh[a].hi;
            lo[(int64_t)(LO_N + 3 * l + a) * p.stride] = (float)nh[a].lo;
        }
        dd Lp, Lm; /* link +l (s -> r) and -l (r -> s) */
        if (p.mode == LTDI_ORBIT_STATIC_EQUALARM) {
            Lp = Lm = p.L_static;
        } else if (KNOTS || p.mode == LTDI_ORBIT_KEPLERIAN) {
            // first-order light time |d|/c (1 + n.V_sender / c): L_l != L_-l (Eq. B22)
            const double nvs = nh[0].hi * V[s][0] + nh[1].hi * V[s][1] + nh[2].hi * V[s][2];
            const double nvr = -(nh[0].hi * V[r][0] + nh[1].hi * V[r][1] + nh[2].hi * V[r][2]);
            const dd lc = (!KNOTS && p.mode == LTDI_ORBIT_KEPLERIAN) ? p.L_static : dd_mul(len, p.inv_c);
            Lp = dd_mul(lc, two_sum(1.0, nvs * p.inv_c.hi));
            Lm = dd_mul(lc, two_sum(1.0, nvr * p.inv_c.hi));
        } else {
            Lp = dd_make(p.L_in[(int64_t)l * p.n + n], 0.0);
            Lm = dd_make(p.L_in[(int64_t)(l + 3) * p.n + n], 0.0);
        }
        out[(int64_t)(ROW_L + l) * p.stride] = Lp.hi;
        out[(int64_t)(ROW_L + 3 + l) * p.stride] = Lm.hi;
        lo[(int64_t)(LO_L + l) * p.stride] = (float)Lp.lo;
        lo[(int64_t)(LO_L + 3 + l) * p.stride] = (float)Lm.lo;
    }
}
