// response.cuh -- S1-S8: source frame, projection, TDI, LFA and hybrid kernels.
//
// One CTA computes one tile of TN consecutive output samples of one source, fused:
//   phase H   stage the window of h+, hx the tile can reach into shared memory
//   phase A   full links y_slr (Eq. 2.5, six links) on the tile plus its TDI halo      [full, hybrid]
//   phase A'  LFA links (Eq. B10, three links) on the tile plus halo plus stencil rim  [LFA, hybrid]
//   phase B'  first / second central difference of the LFA links                       [LFA, hybrid]
//   phase C   Michelson X, Y, Z (Eq. 2.7 / 2.8 resp. B25 / B33), blend (4.5)/(4.6), A, E, T (2.9)
// The link series never leave shared memory unless the caller asks for them (d_y).
#pragma once
#include "common.cuh"

struct HybDev { double t_hyb, window_s, sigma_s, taper; };

struct RespParams {
    const double *tab;   /* orbit table */
    int64_t stride, n;
    double t0, dt;
    const double *hp, *hc;
    int64_t ld, batch;
    const double *frames; /* [batch][LTDI_FRAME_STRIDE]: k, u, v, cos 2psi, sin 2psi */
    const HybDev *hyb;    /* [n_hyb] */
    int64_t n_hyb;
    int which, gen, M, fd;
    int64_t m1, m2, w;    /* reaches (samples) */
    int64_t lo, hi;       /* output margins */
    double *A, *E, *T, *XYZ, *Y;
    int tile;             /* TN */
    int yr;               /* samples of link series per tile = TN + m2 + M/2 + 1 */
    int hw;               /* samples of staged strain per tile */
    int off_yL, off_dL, off_hs; /* shared-memory offsets (doubles) of the LFA links, their derivative, the strain */
    int qmax;             /* bound on |integer shift| of a projection delay (m1 - M/2) */
    int nested;           /* nested TDI delays (tuned path only) */
    int sagnac;           /* alpha, beta, gamma in place of X, Y, Z (generic kernel only) */
    const struct ChirpDev *chirp; /* waveform model constants [batch], or nullptr (sampled strain) */
    int lfa6;             /* all six LFA links and the Michelson variables of Eq. (B20) / (B30) (generic kernel) */
    int lfa_terms, lfa_point, xw; /* terms of Eq. (B4), expansion point LTDI_LFA_*, xw = terms - 1 */
    int64_t ntiles;
};

// ---------------------------------------------------------------------------------------------
// S1: source frame, Eq. (2.1) with G1: k = -e_r, u = -e_phi, v = -e_theta; cos 2psi, sin 2psi (2.3)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void source_frame_one(double beta, double lam, double psi, double *f)
{
    double sb, cb, sl, cl, s2, c2;
    sincos(beta, &sb, &cb);
    sincos(lam, &sl, &cl);
    sincos(2.0 * psi, &s2, &c2);
    f[0] = -cb * cl; f[1] = -cb * sl; f[2] = -sb;   /* k */
    f[3] = sl;       f[4] = -cl;      f[5] = 0.0;   /* u */
    f[6] = -sb * cl; f[7] = -sb * sl; f[8] = cb;    /* v */
    f[9] = c2;       f[10] = s2;
}

// ---------------------------------------------------------------------------------------------
// Lagrange fractional delay (G10): taps k = -(M/2-1) .. M/2 around sample j = n - ceil(d/dt)
// ---------------------------------------------------------------------------------------------
template <int MT>
struct Lagrange {
    double w[MT ? MT : LTDI_MAX_TAPS];

    // w_k(eps) = c_k * prod_{m<k}(eps - m) * prod_{m>k}(eps - m): forward prefix products, then
    // a backward sweep with the running suffix product.
    __device__ __forceinline__ void weights(double eps, int M)
    {
        const int Mx = MT ? MT : M;
        const double *c = c_lag_inv_den + (Mx / 2 - 1) * LTDI_MAX_TAPS;
        const int kmin = -(Mx / 2 - 1);
        double run = 1.0;
#pragma unroll
        for (int i = 0; i < Mx; ++i) {
            w[i] = run;
            run *= eps - (double)(kmin + i);
        }
        run = 1.0;
#pragma unroll
        for (int i = Mx - 1; i >= 0; --i) {
            w[i] = (w[i] * run) * c[i];
            run *= eps - (double)(kmin + i);
        }
    }
    __device__ __forceinline__ double dot(const double *x, int M) const
    {
        const int Mx = MT ? MT : M;
        double acc = 0.0;
#pragma unroll
        for (int i = 0; i < Mx; ++i) acc = fma(w[i], x[i], acc);
        return acc;
    }
};

// delay d [s] -> integer shift q = ceil(d / dt), eps = q - d / dt in [0, 1); only the small
// quantity d / dt enters, never the absolute time.
__device__ __forceinline__ void split_delay(double d, double dt, int &q, double &eps)
{
    const double s = d / dt;
    const double qc = ceil(s);
    q = (int)qc;
    eps = qc - s;
}
// projection delays are bounded by the margin formula (|k.R|/c + L <= 1.02 (R + arm)/c); a table that
// violates the bound reads inside the staged window instead of out of bounds
__device__ __forceinline__ int clamp_shift(int q, int qmax) { return max(-qmax, min(qmax, q)); }

// geometry of one sample for one source (S2)
struct Geom {
    double kR[3];          /* k . R_i / c [s] */
    double Fp[3], Fc[3];   /* F^+_l, F^x_l for |l| = 1, 2, 3 (even in n_l) */
    double kn[3];          /* k . n_l for l = +1, +2, +3 */
    double L[6];           /* light travel times [s] */
};

__device__ __forceinline__ void load_geometry(const RespParams &p, const double *fr, int64_t m, Geom &g)
{
    const double *t = p.tab + m;
    const double inv_c = 1.0 / LTDI_C_LIGHT;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const double x = t[(int64_t)(ROW_R + 3 * i + 0) * p.stride];
        const double y = t[(int64_t)(ROW_R + 3 * i + 1) * p.stride];
        const double z = t[(int64_t)(ROW_R + 3 * i + 2) * p.stride];
        g.kR[i] = (fr[0] * x + fr[1] * y + fr[2] * z) * inv_c;
    }
#pragma unroll
    for (int l = 0; l < 3; ++l) {
        const double x = t[(int64_t)(ROW_N + 3 * l + 0) * p.stride];
        const double y = t[(int64_t)(ROW_N + 3 * l + 1) * p.stride];
        const double z = t[(int64_t)(ROW_N + 3 * l + 2) * p.stride];
        const double un = fr[3] * x + fr[4] * y + fr[5] * z;
        const double vn = fr[6] * x + fr[7] * y + fr[8] * z;
        g.kn[l] = fr[0] * x + fr[1] * y + fr[2] * z;
        const double xip = un * un - vn * vn; /* (2.4a) */
        const double xic = 2.0 * un * vn;     /* (2.4b) */
        g.Fp[l] = xip * fr[9] + xic * fr[10]; /* (2.2) + (2.3) folded, G17 */
        g.Fc[l] = xic * fr[9] - xip * fr[10];
    }
#pragma unroll
    for (int l = 0; l < 6; ++l) g.L[l] = t[(int64_t)(ROW_L + l) * p.stride];
}

__device__ __forceinline__ void load_light_times(const RespParams &p, int64_t n, double L[6])
{
#pragma unroll
    for (int l = 0; l < 6; ++l) L[l] = p.tab[(int64_t)(ROW_L + l) * p.stride + n];
}

// strain access: staged window in shared memory (index relative to h0) or global memory
template <bool STAGE>
struct Strain {
    const double *hp, *hc; /* STAGE: shared arrays whose element 0 is absolute sample h0 */
    int64_t h0;
    __device__ __forceinline__ const double *plus(int64_t i) const { return hp + (i - h0); }
    __device__ __forceinline__ const double *cross(int64_t i) const { return hc + (i - h0); }
};

// Eq. (2.5): the six links at sample m
template <int MT, bool STAGE>
__device__ __forceinline__ void links_full(const RespParams &p, const Strain<STAGE> &h, const double *fr, int64_t m,
                                           double y[6])
{
    Geom g;
    load_geometry(p, fr, m, g);
    Lagrange<MT> lag;
    const int half = (MT ? MT : p.M) / 2 - 1;
    double rp[3], rc[3]; /* h+, hx at the receiver times t - k.R_r / c (2.6b) */
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        int q;
        double eps;
        split_delay(g.kR[i], p.dt, q, eps);
        q = clamp_shift(q, p.qmax);
        lag.weights(eps, p.M);
        const int64_t j = m - q - half;
        rp[i] = lag.dot(h.plus(j), p.M);
        rc[i] = lag.dot(h.cross(j), p.M);
    }
#pragma unroll
    for (int l = 0; l < 6; ++l) {
        const int s = link_sender(l), r = link_receiver(l), a = l % 3;
        int q;
        double eps;
        split_delay(g.L[l] + g.kR[s], p.dt, q, eps); /* (2.6a) */
        q = clamp_shift(q, p.qmax);
        lag.weights(eps, p.M);
        const int64_t j = m - q - half;
        const double sp = lag.dot(h.plus(j), p.M);
        const double sc = lag.dot(h.cross(j), p.M);
        const double kn = l < 3 ? g.kn[a] : -g.kn[a];
        y[l] = (g.Fp[a] * (sp - rp[r]) + g.Fc[a] * (sc - rc[r])) / (2.0 * (1.0 - kn));
    }
}

// first central difference of the strain times (2 dt) resp. (12 dt): numerators only
template <int FD>
__device__ __forceinline__ double fd1_num(const double *x)
{
    if (FD == 2) return x[1] - x[-1];
    return 8.0 * (x[1] - x[-1]) - (x[2] - x[-2]);
}

// third central difference of the strain times (2 dt^3) resp. (8 dt^3): numerators only, written as
// differences of symmetric pairs
template <int FD>
__device__ __forceinline__ double fd3_num(const double *x)
{
    const double p1 = x[1] - x[-1], p2 = x[2] - x[-2];
    if (FD == 2) return p2 - 2.0 * p1;
    return 8.0 * p2 - 13.0 * p1 - (x[3] - x[-3]);
}

// Eq. (B10) at the retarded time (B1): the three links l = +1, +2, +3 at sample m.  SURVEY 8(f)-2: with
// p.lfa_terms = 2 the m = 1 term of Eq. (B4) is added; p.lfa_point moves the expansion point to (B13) / (B14).
template <int MT, bool STAGE>
__device__ __forceinline__ void links_lfa(const RespParams &p, const Strain<STAGE> &h, const double *fr, int64_t m,
                                          double y[3])
{
    Geom g;
    load_geometry(p, fr, m, g);
    Lagrange<MT> lag;
    const int Mx = MT ? MT : p.M;
    const int half = Mx / 2 - 1;
    const double den = (p.fd == 2 ? 2.0 : 12.0) * p.dt;
    const double den3 = (p.fd == 2 ? 2.0 : 8.0) * p.dt * p.dt * p.dt;
#pragma unroll
    for (int l = 0; l < 3; ++l) {
        const int s = link_sender(l), r = link_receiver(l);
        int q;
        double eps;
        const double tau = p.lfa_point == LTDI_LFA_CENTRAL ? 0.5 * g.L[l] + 0.5 * (g.kR[s] + g.kR[r])      /* (B1) */
                           : p.lfa_point == LTDI_LFA_BACKWARD ? g.L[l] + g.kR[s] : g.kR[r];                 /* (B13), (B14) */
        split_delay(tau, p.dt, q, eps);
        q = clamp_shift(q, p.qmax);
        lag.weights(eps, p.M);
        const double *xp = h.plus(m - q - half), *xc = h.cross(m - q - half);
        double ap = 0.0, ac = 0.0;
        if (p.fd == 2) {
#pragma unroll
            for (int i = 0; i < Mx; ++i) {
                ap = fma(lag.w[i], fd1_num<2>(xp + i), ap);
                ac = fma(lag.w[i], fd1_num<2>(xc + i), ac);
            }
        } else {
#pragma unroll
            for (int i = 0; i < Mx; ++i) {
                ap = fma(lag.w[i], fd1_num<4>(xp + i), ap);
                ac = fma(lag.w[i], fd1_num<4>(xc + i), ac);
            }
        }
        double dH = g.Fp[l] * (ap / den) + g.Fc[l] * (ac / den);
        if (p.lfa_terms >= 2) {   /* m = 1 term of (B4): (1/6) [(L_l / 2)(1 - k.n_l)]^2 d^3H/dt^3 */
            double bp = 0.0, bc = 0.0;
            for (int i = 0; i < Mx; ++i) {
                bp = fma(lag.w[i], p.fd == 2 ? fd3_num<2>(xp + i) : fd3_num<4>(xp + i), bp);
                bc = fma(lag.w[i], p.fd == 2 ? fd3_num<2>(xc + i) : fd3_num<4>(xc + i), bc);
            }
            const double hf = (0.5 * g.L[l]) * (1.0 - g.kn[l]);
            dH += hf * hf / 6.0 * (g.Fp[l] * (bp / den3) + g.Fc[l] * (bc / den3));
        }
        y[l] = -(0.5 * g.L[l]) * dH;
    }
}

// SURVEY 8(f)-2, Eq. (B20) / (B30): all six LFA links, each at the retarded time (B1) with ITS OWN light time
template <int MT, bool STAGE>
__device__ __forceinline__ void links_lfa6(const RespParams &p, const Strain<STAGE> &h, const double *fr, int64_t m,
                                           double y[6])
{
    Geom g;
    load_geometry(p, fr, m, g);
    Lagrange<MT> lag;
    const int Mx = MT ? MT : p.M;
    const int half = Mx / 2 - 1;
    const double den = (p.fd == 2 ? 2.0 : 12.0) * p.dt;
#pragma unroll 1
    for (int l = 0; l < 6; ++l) {
        const int s = link_sender(l), r = link_receiver(l), a = l % 3;
        int q;
        double eps;
        split_delay(0.5 * g.L[l] + 0.5 * (g.kR[s] + g.kR[r]), p.dt, q, eps);      /* (B1) */
        q = clamp_shift(q, p.qmax);
        lag.weights(eps, p.M);
        const double *xp = h.plus(m - q - half), *xc = h.cross(m - q - half);
        double ap = 0.0, ac = 0.0;
        for (int i = 0; i < Mx; ++i) {
            ap = fma(lag.w[i], p.fd == 2 ? fd1_num<2>(xp + i) : fd1_num<4>(xp + i), ap);
            ac = fma(lag.w[i], p.fd == 2 ? fd1_num<2>(xc + i) : fd1_num<4>(xc + i), ac);
        }
        y[l] = -(0.5 * g.L[l]) * (g.Fp[a] * (ap / den) + g.Fc[a] * (ac / den));   /* (B10) */
    }
}

// D_delay y: series ys (shared memory, element 0 = absolute sample y0, length len) at t_n - delay
template <int MT>
__device__ __forceinline__ double delayed(const RespParams &p, const double *ys, int64_t y0, int len, int64_t n,
                                          double delay)
{
    int q;
    double eps;
    split_delay(delay, p.dt, q, eps);
    Lagrange<MT> lag;
    lag.weights(eps, p.M);
    const int Mx = MT ? MT : p.M;
    int j = (int)(n - q - (Mx / 2 - 1) - y0);
    if (j < 0 || j + Mx > len) { /* outside the tile's halo: only for light times beyond the margin bound */
        double acc = 0.0;
        for (int i = 0; i < Mx; ++i) {
            const int jj = j + i;
            if (jj >= 0 && jj < len) acc = fma(lag.w[i], ys[jj], acc);
        }
        return acc;
    }
    return lag.dot(ys + j, p.M);
}

// Eq. (2.7) / (2.8), channel ch = 0, 1, 2 -> X, Y, Z (cyclic 1->2->3->1), all delays at t_n.
// Written in the factorised form X_1.5 = (1 - D_b)(D_dP P + Q) - (1 - D_a)(D_dU U + W),
// X_2.0 = (1 - D_{a+b}) X_1.5 with every operator product expanded into single delays.
template <int MT>
__device__ __forceinline__ double michelson_full(const RespParams &p, const double *yF, int64_t y0, int64_t n,
                                                 const double L[6], int ch)
{
    const int i2 = (1 + ch) % 3, i3 = (2 + ch) % 3;  /* |l| - 1 of the two arms: X: 2,3  Y: 3,1  Z: 1,2 */
    const double *P = yF + (size_t)i2 * p.yr;        /* y_{+p2}  (y_123 for X)  */
    const double *Q = yF + (size_t)(i2 + 3) * p.yr;  /* y_{-p2}  (y_3-21)       */
    const double *U = yF + (size_t)(i3 + 3) * p.yr;  /* y_{-p3}  (y_1-32)       */
    const double *W = yF + (size_t)i3 * p.yr;        /* y_{+p3}  (y_231)        */
    const double dP = L[i2 + 3], dU = L[i3];
    const double a = L[i2 + 3] + L[i2], b = L[i3] + L[i3 + 3];
    const int i0 = (int)(n - y0);
#define DEL(S, d) delayed<MT>(p, S, y0, p.yr, n, (d))
    double x = (DEL(P, dP) - DEL(P, dP + b)) + (Q[i0] - DEL(Q, b));
    x -= (DEL(U, dU) - DEL(U, dU + a)) + (W[i0] - DEL(W, a));
    if (p.gen == LTDI_GEN_20) {
        double z = (DEL(P, dP + a + b) - DEL(P, dP + a + 2.0 * b)) + (DEL(Q, a + b) - DEL(Q, a + 2.0 * b));
        z -= (DEL(U, dU + a + b) - DEL(U, dU + 2.0 * a + b)) + (DEL(W, a + b) - DEL(W, 2.0 * a + b));
        x -= z;
    }
#undef DEL
    return x;
}

// SURVEY 8(f)-4 (reading G33): the Sagnac combinations, channel ch = 0, 1, 2 -> alpha, beta, gamma.
// With S+ = y_{+3} + D_{+3} y_{+1} + D_{+3} D_{+1} y_{+2} (the beam 1 -> 3 -> 2 -> 1), S- = y_{-2} + D_{-2} y_{-1} +
// D_{-2} D_{-1} y_{-3} (1 -> 2 -> 3 -> 1) and the round-trip times T+ = L_3 + L_1 + L_2, T- = L_-2 + L_-1 + L_-3:
// gen 1.5: alpha = S+ - S- (6 terms); gen 2.0: alpha = (S+ + D_{T+} S-) - (S- + D_{T-} S+) (12 terms); all delays at t_n
// (P:151); beta, gamma by the cyclic permutation of the labels.
template <int MT>
__device__ __forceinline__ double sagnac_full(const RespParams &p, const double *yF, int64_t y0, int64_t n,
                                              const double L[6], int ch)
{
    const int k3 = (2 + ch) % 3, k1 = ch % 3, k2 = (1 + ch) % 3;   /* |l| - 1 of the labels 3, 1, 2 permuted */
    const double *P3 = yF + (size_t)k3 * p.yr, *P1 = yF + (size_t)k1 * p.yr, *P2 = yF + (size_t)k2 * p.yr;
    const double *M2 = yF + (size_t)(k2 + 3) * p.yr, *M1 = yF + (size_t)(k1 + 3) * p.yr, *M3 = yF + (size_t)(k3 + 3) * p.yr;
    const double Lp3 = L[k3], Lp1 = L[k1], Lp2 = L[k2], Lm2 = L[k2 + 3], Lm1 = L[k1 + 3], Lm3 = L[k3 + 3];
    const double Tp = Lp3 + Lp1 + Lp2, Tm = Lm2 + Lm1 + Lm3;
    const int i0 = (int)(n - y0);
#define DEL(S, d) delayed<MT>(p, S, y0, p.yr, n, (d))
    double a = P3[i0] + DEL(P1, Lp3) + DEL(P2, Lp3 + Lp1) - M2[i0] - DEL(M1, Lm2) - DEL(M3, Lm2 + Lm1);
    if (p.gen == LTDI_GEN_20)
        a += DEL(M2, Tp) + DEL(M1, Tp + Lm2) + DEL(M3, Tp + Lm2 + Lm1) - DEL(P3, Tm) - DEL(P1, Tm + Lp3) - DEL(P2, Tm + Lp3 + Lp1);
#undef DEL
    return a;
}

// Eq. (B25) (gen 1.5) / (B33) (gen 2.0): dL = first resp. second derivative of the LFA links
template <int MT>
__device__ __forceinline__ double michelson_lfa(const RespParams &p, const double *dL, int64_t y0, int64_t n,
                                                const double L[6], int ch)
{
    const int i2 = (1 + ch) % 3, i3 = (2 + ch) % 3;
    const double L2 = L[i2], L3 = L[i3]; /* positive-link values, G14 */
    const double *d123 = dL + (size_t)i2 * p.yr, *d231 = dL + (size_t)i3 * p.yr;
    if (p.gen == LTDI_GEN_15)
        return 4.0 * (L3 * delayed<MT>(p, d123, y0, p.yr, n, L3 + 0.5 * L2) -
                      L2 * delayed<MT>(p, d231, y0, p.yr, n, L2 + 0.5 * L3));
    return 8.0 * (L2 + L3) * (L3 * delayed<MT>(p, d123, y0, p.yr, n, 2.0 * L3 + 1.5 * L2) -
                              L2 * delayed<MT>(p, d231, y0, p.yr, n, 2.0 * L2 + 1.5 * L3));
}

// Eq. (B20) (gen 1.5) / (B30) (gen 2.0) at the mid-points (B18) / (B31) (G13): dlo / dhi = the lower / higher of the two
// time derivatives of the six LFA links, [6][yr] each
template <int MT>
__device__ __forceinline__ double michelson_b20(const RespParams &p, const double *dlo, const double *dhi, int64_t y0,
                                                int64_t n, const double L[6], int ch)
{
    const int i2 = (1 + ch) % 3, i3 = (2 + ch) % 3;
    const double Lp2 = L[i2], Lm2 = L[i2 + 3], Lp3 = L[i3], Lm3 = L[i3 + 3];
    const double a = Lm2 + Lp2, b = Lm3 + Lp3;
    double d2, d3, pre;
    if (p.gen == LTDI_GEN_15) { d2 = (Lm3 + Lm2 + Lp3) / 2; d3 = (Lm2 + Lp2 + Lp3) / 2; pre = 1.0; }
    else { d2 = Lm3 + Lm2 + Lp3 + Lp2 / 2; d3 = Lm2 + Lp2 + Lp3 + Lm3 / 2; pre = a + b; }
#define DLO(l, d) delayed<MT>(p, dlo + (size_t)(l) * p.yr, y0, p.yr, n, (d))
#define DHI(l, d) delayed<MT>(p, dhi + (size_t)(l) * p.yr, y0, p.yr, n, (d))
    /* P = y_{+p2}, Q = y_{-p2}, U = y_{-p3}, W = y_{+p3} */
    const double x = b * (DLO(i2, d2) - (Lm2 / 2) * DHI(i2, d2)) + b * (DLO(i2 + 3, d2) + (Lm2 / 2) * DHI(i2 + 3, d2)) -
                     a * (DLO(i3 + 3, d3) - (Lp3 / 2) * DHI(i3 + 3, d3)) - a * (DLO(i3, d3) + (Lp3 / 2) * DHI(i3, d3));
#undef DLO
#undef DHI
    return pre * x;
}

// Eqs. (4.1), (4.5) with G18; raised cosine, G20
__device__ __forceinline__ void hybrid_weights(const HybDev &h, double t, double &w_lfa, double &w_full)
{
    const double x0 = t - h.t_hyb, T = h.window_s;
    if (h.taper == (double)LTDI_TAPER_SIGMOID) {
        w_lfa = (x0 <= 0.5 * T) ? 1.0 / (1.0 + exp(x0 / h.sigma_s)) : 0.0;
        w_full = (x0 >= -0.5 * T) ? 1.0 / (1.0 + exp(-x0 / h.sigma_s)) : 0.0;
    } else {
        const double x = (x0 + 0.5 * T) / T;
        if (x <= 0.0) w_full = 0.0;
        else if (x >= 1.0) w_full = 1.0;
        else w_full = 0.5 * (1.0 - cospi(x));
        w_lfa = 1.0 - w_full;
    }
}

// ---------------------------------------------------------------------------------------------
// the fused tile kernel
// ---------------------------------------------------------------------------------------------
template <int MT, bool STAGE>
__global__ void __launch_bounds__(256) response_kernel(RespParams p)
{
    extern __shared__ double smem[];
    const int64_t b = (int64_t)blockIdx.x % p.batch;   /* sources fastest: concurrent CTAs share table rows in L2 */
    const int64_t tile = (int64_t)blockIdx.x / p.batch;
    const int64_t n0 = tile * p.tile;
    const int64_t n1 = min(n0 + (int64_t)p.tile, p.n);
    const int64_t y0 = n0 - p.m2;                     /* first sample of the link series of this tile */
    const int w = (int)p.w;
    const int tid = threadIdx.x, nthr = blockDim.x;

    __shared__ double fr[LTDI_FRAME_STRIDE];
    if (tid < LTDI_FRAME_STRIDE) fr[tid] = p.frames[b * LTDI_FRAME_STRIDE + tid];

    bool need_full = p.which == LTDI_RESPONSE_FULL, need_lfa = p.which == LTDI_RESPONSE_LFA;
    HybDev hyb = {0.0, 0.0, 1.0, 0.0};
    if (p.which == LTDI_RESPONSE_HYBRID) {
        hyb = p.hyb[p.n_hyb == 1 ? 0 : b];
        const double t_first = p.t0 + (double)n0 * p.dt, t_last = p.t0 + (double)(n1 - 1) * p.dt;
        need_lfa = (t_first - hyb.t_hyb) <= 0.5 * hyb.window_s;   /* some sample has w_LFA != 0, Eq. (4.5) */
        need_full = (t_last - hyb.t_hyb) >= -0.5 * hyb.window_s;  /* some sample has w_Full != 0 */
    }

    /* shared memory carve-up (offsets chosen by the host per response type) */
    double *yF = smem;             /* [6][yr]      full links, element 0 = sample y0      */
    double *yL = smem + p.off_yL;  /* [3][yr + 2w] LFA links, element 0 = sample y0 - w   */
    double *dL = smem + p.off_dL;  /* [3][yr]      their derivative, element 0 = y0       */
    double *hs = smem + p.off_hs;  /* [2][hw]      strain window, element 0 = sample h0   */

    Strain<STAGE> h;
    const int64_t src_off = b * p.ld;
    if (STAGE) {
        /* phase H: every sample any stencil of this tile can touch, clipped to the grid */
        const int64_t h0 = y0 - p.m1 - 3 * w - p.xw;
        for (int i = tid; i < p.hw; i += nthr) {
            const int64_t g = h0 + i;
            const bool in = g >= 0 && g < p.n;
            hs[i] = in ? p.hp[src_off + g] : 0.0;
            hs[p.hw + i] = in ? p.hc[src_off + g] : 0.0;
        }
        h.hp = hs;
        h.hc = hs + p.hw;
        h.h0 = h0;
    } else {
        h.hp = p.hp + src_off;
        h.hc = p.hc + src_off;
        h.h0 = 0;
    }
    __syncthreads();

    if (need_full) { /* phase A */
        for (int i = tid; i < p.yr; i += nthr) {
            const int64_t m = y0 + i;
            double y[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
            if (m >= p.m1 && m < p.n - p.m1) links_full<MT, STAGE>(p, h, fr, m, y);
#pragma unroll
            for (int l = 0; l < 6; ++l) yF[(size_t)l * p.yr + i] = y[l];
        }
    }
    if (need_lfa && p.lfa6) { /* six links, two derivatives of each */
        const int wy = w + p.xw;                     /* widest stencil applied to the links (third derivative for gen 2.0) */
        const int len = p.yr + 2 * wy;
        for (int i = tid; i < len; i += nthr) {
            const int64_t m = y0 - wy + i;
            double y[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
            if (m >= p.m1 + w && m < p.n - p.m1 - w) links_lfa6<MT, STAGE>(p, h, fr, m, y);
#pragma unroll
            for (int l = 0; l < 6; ++l) yL[(size_t)l * len + i] = y[l];
        }
        __syncthreads();
        const double dt = p.dt;
        double *dhi = dL + (size_t)6 * p.yr;
        for (int i = tid; i < p.yr; i += nthr) {
            const int64_t m = y0 + i;
            const bool in = m >= p.m1 + w + wy && m < p.n - p.m1 - w - wy;
            for (int l = 0; l < 6; ++l) {
                const double *x = yL + (size_t)l * len + i + wy; /* x[0] = y_l[m] */
                double d1 = 0.0, d2v = 0.0, d3v = 0.0;
                if (in) {
                    const double p1 = x[1] - x[-1];
                    const double s1 = (x[1] - x[0]) - (x[0] - x[-1]);
                    if (p.fd == 2) {
                        d1 = p1 / (2.0 * dt);
                        d2v = s1 / (dt * dt);
                        if (p.gen != LTDI_GEN_15) d3v = ((x[2] - x[-2]) - 2.0 * p1) / (2.0 * dt * dt * dt);
                    } else {
                        const double p2 = x[2] - x[-2];
                        const double s2 = (x[2] - x[0]) - (x[0] - x[-2]);
                        d1 = (8.0 * p1 - p2) / (12.0 * dt);
                        d2v = (16.0 * s1 - s2) / (12.0 * dt * dt);
                        if (p.gen != LTDI_GEN_15) d3v = (8.0 * p2 - 13.0 * p1 - (x[3] - x[-3])) / (8.0 * dt * dt * dt);
                    }
                }
                dL[(size_t)l * p.yr + i] = p.gen == LTDI_GEN_15 ? d1 : d2v;
                dhi[(size_t)l * p.yr + i] = p.gen == LTDI_GEN_15 ? d2v : d3v;
            }
        }
    } else if (need_lfa) { /* phase A' */
        const int len = p.yr + 2 * w;
        for (int i = tid; i < len; i += nthr) {
            const int64_t m = y0 - w + i;
            double y[3] = {0.0, 0.0, 0.0};
            if (m >= p.m1 + w + p.xw && m < p.n - p.m1 - w - p.xw) links_lfa<MT, STAGE>(p, h, fr, m, y);
#pragma unroll
            for (int l = 0; l < 3; ++l) yL[(size_t)l * len + i] = y[l];
        }
        __syncthreads();
        /* phase B': FD1 (gen 1.5) or FD2 (gen 2.0) of the LFA links, G15 */
        const double dt = p.dt;
        for (int i = tid; i < p.yr; i += nthr) {
            const int64_t m = y0 + i;
            const bool in = m >= p.m1 + 2 * w + p.xw && m < p.n - p.m1 - 2 * w - p.xw;
#pragma unroll
            for (int l = 0; l < 3; ++l) {
                const double *x = yL + (size_t)l * len + i + w; /* x[0] = y_l[m] */
                double d = 0.0;
                if (in) {
                    if (p.gen == LTDI_GEN_15) {
                        d = (p.fd == 2) ? (x[1] - x[-1]) / (2.0 * dt)
                                        : (8.0 * (x[1] - x[-1]) - (x[2] - x[-2])) / (12.0 * dt);
                    } else {
                        const double d1 = (x[1] - x[0]) - (x[0] - x[-1]);
                        if (p.fd == 2) d = d1 / (dt * dt);
                        else {
                            const double d2 = (x[2] - x[0]) - (x[0] - x[-2]);
                            d = (16.0 * d1 - d2) / (12.0 * dt * dt);
                        }
                    }
                }
                dL[(size_t)l * p.yr + i] = d;
            }
        }
    }
    __syncthreads();

    /* phase C */
    const double is2 = 0.70710678118654752440, is6 = 0.40824829046386301637, is3 = 0.57735026918962576451;
    for (int i = tid; i < p.tile; i += nthr) {
        const int64_t n = n0 + i;
        if (n >= n1) break;
        double X[3] = {0.0, 0.0, 0.0};
        double wa = 1.0, wb = 1.0;
        if (p.which == LTDI_RESPONSE_HYBRID) hybrid_weights(hyb, p.t0 + (double)n * p.dt, wa, wb);
        if (n >= p.lo && n < p.n - p.hi) {
            double L[6];
            load_light_times(p, n, L);
#pragma unroll 1
            for (int ch = 0; ch < 3; ++ch) {
                double x = 0.0;
                if (need_lfa && p.lfa6) x = michelson_b20<MT>(p, dL, dL + (size_t)6 * p.yr, y0, n, L, ch);
                else if (need_lfa && wa != 0.0) x = wa * michelson_lfa<MT>(p, dL, y0, n, L, ch);
                if (need_full && p.sagnac) x = sagnac_full<MT>(p, yF, y0, n, L, ch);
                else if (need_full && wb != 0.0) x = fma(wb, michelson_full<MT>(p, yF, y0, n, L, ch), x); /* (4.6) */
                X[ch] = x;
            }
        }
        const int64_t o = src_off + n;
        p.A[o] = (X[2] - X[0]) * is2;                 /* (2.9a) */
        p.E[o] = (X[0] - 2.0 * X[1] + X[2]) * is6;    /* (2.9b) */
        p.T[o] = (X[0] + X[1] + X[2]) * is3;          /* (2.9c) */
        if (p.XYZ) {
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) p.XYZ[((int64_t)ch * p.batch + b) * p.ld + n] = X[ch];
        }
        if (p.Y) {
            const int iy = (int)(n - y0);
#pragma unroll
            for (int l = 0; l < 6; ++l) {
                double v = 0.0;
                if (p.which == LTDI_RESPONSE_FULL) v = yF[(size_t)l * p.yr + iy];
                else if (p.which == LTDI_RESPONSE_LFA && p.lfa6) v = yL[(size_t)l * (p.yr + 2 * (w + p.xw)) + iy + w + p.xw];
                else if (p.which == LTDI_RESPONSE_LFA) v = l < 3 ? yL[(size_t)l * (p.yr + 2 * w) + iy + w] : 0.0;
                else if (n >= p.m1 + w && n < p.n - p.m1 - w) { /* (4.5) */
                    if (need_lfa && l < 3) v = wa * yL[(size_t)l * (p.yr + 2 * w) + iy + w];
                    if (need_full) v = fma(wb, yF[(size_t)l * p.yr + iy], v);
                }
                p.Y[((int64_t)l * p.batch + b) * p.ld + n] = v;
            }
        }
    }
}
