/*
 * lisa_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, step-by-step CPU implementation of the time-domain LISA response
 * of arXiv 2505.09600 (Valencia & Husa): full response, low-frequency
 * approximation (LFA) and hybrid.  Written from the paper ("P:n" = line n of
 * /root/reference/PAPER.md) with the readings listed in DESIGN.md ("G1".."G23",
 * SURVEY.md section 8c).  It shares no code, header, table or constant generator
 * with the CUDA path under paper_2505_09600_b200/csrc, and neither imports the
 * other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * The same source is compiled twice (oracle/build.py):
 *   -DORC_REAL_LD  : real = long double (x87 80 bit) -> the parity reference
 *   (default)      : real = double                  -> timed baseline, fp64 floor
 * Inputs and outputs are always IEEE double arrays; only the arithmetic in
 * between changes.  No blocking, fusion or reordering: every function follows
 * the cited equation in the paper's order.  OpenMP only splits the outermost
 * loop over output samples / sources, which are independent.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Lagrange exactness on
 * polynomials, weights sum to 1, integer delay = pure shift; stencil exactness
 * on polynomials; orthonormal triad; rigid-triangle orbit, |R_i| = R(1 +- e),
 * Sagnac amplitude of Eq. (B22); constant strain -> zero response;
 * monochromatic plane-wave closed form on a frozen constellation (Eq. C3);
 * X_2.0[n] = X_1.5[n] - X_1.5[n - 4L/(c dt)] for static equal arms; Eq. (3.7)
 * low-frequency relation; LFA -> full as f L / c -> 0 with the x / sin x law of
 * Eq. (B4); T^LFA = 0 for equal arms; psi invariances; Eq. (4.2)/(4.4) printed
 * values 0.95 / 0.97 / 0.99; taper partition of unity.
 * Rows added after the hot path, each pinned the same way (tests/test_oracle_*.py):
 * extended LFA (m = 1 term of (B4): (x - x^3/6)/sin x; (B13)/(B14): first-order
 * residual); O11 numerical orbits (polynomial trajectories exact, O1 reproduced);
 * O12 nested delays (laser-noise cancellation only with nested TDI 2.0, brute-force
 * chains); O13 waveform model (numpy generator, Eq. (4.2), join closed forms, the
 * interpolating response); O14 Eq. (B20)/(B30) (second-order agreement with the exact
 * combination of six unrelated links, (B25)/(B33) for equal constant arms);
 * O13b eccentric harmonic sums (numpy generator, circular limit, Peters-Mathews power
 * sum g(n, e)); O15 Sagnac alpha, beta, gamma (laser noise cancels in the 6-term form
 * iff the round trips agree and in the 12-term form for any constant L_l != L_-l, with
 * the residual in closed form; beams walked by spacecraft number; the operator identity
 * (1 - D^2)(1 - D) sum(alpha) = -(1 + D + D^2) sum(X) for equal arms).
 * Parity unpinned: absolute amplitudes of the paper's figures (no printed
 * input -> output example exists in the paper).
 */
#define _DEFAULT_SOURCE /* jn, jnl (Bessel functions of the first kind) with -std=c11 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORC_REAL_LD
typedef long double real;
#define R_SIN sinl
#define R_COS cosl
#define R_SQRT sqrtl
#define R_CEIL ceill
#define R_EXP expl
#define R_POW powl
#define R_PI 3.14159265358979323846264338327950288L
#define R_JN jnl
#else
typedef double real;
#define R_SIN sin
#define R_COS cos
#define R_SQRT sqrt
#define R_CEIL ceil
#define R_EXP exp
#define R_POW pow
#define R_PI 3.14159265358979323846
#define R_JN jn
#endif

#define ORC_OK 0
#define ORC_EINVAL (-1)

#define ORC_C_LIGHT 299792458.0 /* m/s, exact (SI) */

enum { ORC_GEN_15 = 15, ORC_GEN_20 = 20 };
enum { ORC_ORBIT_STATIC_EQUALARM = 0, ORC_ORBIT_KEPLERIAN = 1, ORC_ORBIT_TABLES = 2, ORC_ORBIT_KNOTS = 3 };
enum { ORC_TAPER_SIGMOID = 0, ORC_TAPER_COSINE = 1 };

typedef struct {
    double t0, dt;   /* t_n = t0 + n dt [s] */
    int64_t n;       /* samples */
    double arm_m;    /* nominal arm length L [m] */
    double R_m;      /* orbital radius R [m] */
    double period_s; /* orbital period [s], Omega = 2 pi / period */
    double alpha0;   /* orbital phase at t = 0 [rad] */
    double rot0;     /* constellation rotation phase [rad] */
    int32_t mode;    /* ORC_ORBIT_* */
} orc_orbit_desc;

typedef struct { double beta, lambda, psi; } orc_source;
typedef struct { double t_hyb, window_s, sigma_s; int32_t taper; } orc_hybrid;

/* Links: index 0..5 = l = +1,+2,+3,-1,-2,-3 ; y_{s l r}: sender s -> receiver r.
 * +1: 3->2 (y_312)  +2: 1->3 (y_123)  +3: 2->1 (y_231)
 * -1: 2->3 (y_2-13) -2: 3->1 (y_3-21) -3: 1->2 (y_1-32)      spacecraft 0-based below */
static const int LINK_S[6] = { 2, 0, 1, 1, 2, 0 };
static const int LINK_R[6] = { 1, 2, 0, 2, 0, 1 };

static int link_index(int label) /* label in {+-1,+-2,+-3} -> 0..5 */
{
    return label > 0 ? label - 1 : 2 - label;
}

/* ---------------------------------------------------------------------------------- */
/* O4  Lagrange fractional-delay interpolation (reading G10)                */
/* ---------------------------------------------------------------------------------- */

/* w_k(eps) = prod_{m != k} (eps - m) / (k - m),  k, m = -(M/2-1) .. M/2,  M = order+1 */
static void lagrange_weights(real eps, int order, real *w)
{
    const int M = order + 1, kmin = -(M / 2 - 1), kmax = M / 2;
    for (int k = kmin; k <= kmax; ++k) {
        real num = 1, den = 1;
        for (int m = kmin; m <= kmax; ++m) {
            if (m == k) continue;
            num *= (eps - (real)m);
            den *= (real)(k - m);
        }
        w[k - kmin] = num / den;
    }
}

/* split a delay d [s] into the integer shift q = ceil(d/dt) and eps = q - d/dt in [0,1).
 * Only the small quantity d/dt enters, never the absolute time. */
static void delay_split(real d, real dt, int64_t *q, real *eps)
{
    const real s = d / dt;
    const real qc = R_CEIL(s);
    *q = (int64_t)qc;
    *eps = qc - s;
}

/* value of the series x (length len, first element = absolute sample x0) at t_n - d.
 * Samples outside [x0, x0+len) read as 0 (they are only touched inside margins). */
static real interp_series(const real *x, int64_t x0, int64_t len, int64_t n, real d, real dt,
                          int order)
{
    real w[64];
    int64_t q;
    real eps;
    const int M = order + 1, kmin = -(M / 2 - 1);
    delay_split(d, dt, &q, &eps);
    lagrange_weights(eps, order, w);
    const int64_t j = n - q;
    real acc = 0;
    for (int i = 0; i < M; ++i) {
        const int64_t idx = j + kmin + i - x0;
        const real v = (idx >= 0 && idx < len) ? x[idx] : (real)0;
        acc += w[i] * v;
    }
    return acc;
}

/* same, reading a double array (the input strain) */
static real interp_input(const double *x, int64_t len, int64_t n, real d, real dt, int order)
{
    real w[64];
    int64_t q;
    real eps;
    const int M = order + 1, kmin = -(M / 2 - 1);
    delay_split(d, dt, &q, &eps);
    lagrange_weights(eps, order, w);
    const int64_t j = n - q;
    real acc = 0;
    for (int i = 0; i < M; ++i) {
        const int64_t idx = j + kmin + i;
        const real v = (idx >= 0 && idx < len) ? (real)x[idx] : (real)0;
        acc += w[i] * v;
    }
    return acc;
}

/* ---------------------------------------------------------------------------------- */
/* O8 stencils (reading G15): central differences of accuracy order 2 / 4             */
/* ---------------------------------------------------------------------------------- */
#define AT(x, i) ((real)(x)[(i)])

static real fd1_in(const double *x, int64_t i, real dt, int fd_order)
{
    if (fd_order == 2) return (AT(x, i + 1) - AT(x, i - 1)) / (2 * dt);
    return (8 * (AT(x, i + 1) - AT(x, i - 1)) - (AT(x, i + 2) - AT(x, i - 2))) / (12 * dt);
}
static real fd1_r(const real *x, int64_t i, real dt, int fd_order)
{
    if (fd_order == 2) return (x[i + 1] - x[i - 1]) / (2 * dt);
    return (8 * (x[i + 1] - x[i - 1]) - (x[i + 2] - x[i - 2])) / (12 * dt);
}
static real fd2_r(const real *x, int64_t i, real dt, int fd_order)
{
    const real d1 = (x[i + 1] - x[i]) - (x[i] - x[i - 1]);
    if (fd_order == 2) return d1 / (dt * dt);
    const real d2 = (x[i + 2] - x[i]) - (x[i] - x[i - 2]);
    return (16 * d1 - d2) / (12 * dt * dt);
}

static real fd3_r(const real *x, int64_t i, real dt, int fd_order)
{
    const real p1 = x[i + 1] - x[i - 1], p2 = x[i + 2] - x[i - 2];
    if (fd_order == 2) return (p2 - 2 * p1) / (2 * dt * dt * dt);
    const real p3 = x[i + 3] - x[i - 3];
    return (8 * p2 - 13 * p1 - p3) / (8 * dt * dt * dt);
}

/* third derivative (the m = 1 term of Eq. (B4) needs d^3 H / dt^3): central stencils of accuracy
 * order 2, (x[+2] - 2 x[+1] + 2 x[-1] - x[-2]) / (2 dt^3), and 4,
 * (-x[+3] + 8 x[+2] - 13 x[+1] + 13 x[-1] - 8 x[-2] + x[-3]) / (8 dt^3), written as differences of symmetric pairs
 * (reading G15 extended: same evaluation order idea as the first-derivative stencils) */
static real fd3_in(const double *x, int64_t i, real dt, int fd_order)
{
    const real p1 = AT(x, i + 1) - AT(x, i - 1), p2 = AT(x, i + 2) - AT(x, i - 2);
    if (fd_order == 2) return (p2 - 2 * p1) / (2 * dt * dt * dt);
    const real p3 = AT(x, i + 3) - AT(x, i - 3);
    return (8 * p2 - 13 * p1 - p3) / (8 * dt * dt * dt);
}

/* ---------------------------------------------------------------------------------- */
/* O1  orbits (readings G5, G6, G7): first-order Keplerian, rigid rotating triangle   */
/* ---------------------------------------------------------------------------------- */
typedef struct {
    orc_orbit_desc d;
    const double *Rtab; /* mode TABLES: [3][3][n] spacecraft, component, sample [m];
                         * mode KNOTS: [3][3][nk] spacecraft, component, knot [m] (a numerical orbit file) */
    const double *Ltab; /* mode TABLES: [6][n] light travel times [s], link order +1,+2,+3,-1,-2,-3;
                         * mode KNOTS: {tk0, dtk, nk, p_orb}: knot j at time tk0 + j dtk, Lagrange order p_orb */
} orbit_ctx;

/* O11 numerical orbits ("realistic ESA orbits"; reading G28): the spacecraft positions are
 * tabulated at nk equidistant knots and brought to the sample time t by centred Lagrange interpolation of odd order
 * p_orb on the knot grid -- the same weights as O4 with u = (t - tk0) / dtk - floor(.) in [0, 1) and taps
 * k = -(M/2 - 1) .. M/2 around the knot at or before t; the velocities are the time derivative of that interpolant
 * (derivative of the weights by the product rule, divided by dtk).  The light travel times then follow G6. */
static void knot_weights(real u, int order, real *w, real *dw)
{
    const int M = order + 1, kmin = -(M / 2 - 1), kmax = M / 2;
    for (int k = kmin; k <= kmax; ++k) {
        real den = 1, num = 1, dnum = 0;
        for (int m = kmin; m <= kmax; ++m)
            if (m != k) den *= (real)(k - m);
        for (int m = kmin; m <= kmax; ++m) {       /* product rule: sum over the factor that is differentiated */
            if (m == k) continue;
            real part = 1;
            for (int j = kmin; j <= kmax; ++j)
                if (j != k && j != m) part *= (u - (real)j);
            dnum += part;
            num *= (u - (real)m);
        }
        w[k - kmin] = num / den;
        dw[k - kmin] = dnum / den;
    }
}

static void knot_positions(const orbit_ctx *o, real t, real R[3][3], real V[3][3])
{
    const real tk0 = (real)o->Ltab[0], dtk = (real)o->Ltab[1];
    const int64_t nk = (int64_t)o->Ltab[2];
    const int order = (int)o->Ltab[3], M = order + 1, kmin = -(M / 2 - 1);
    real w[64], dw[64];
    const real s = (t - tk0) / dtk;
    int64_t j = (int64_t)s;
    if ((real)j > s) --j;                      /* floor */
    knot_weights(s - (real)j, order, w, dw);
    for (int i = 0; i < 3; ++i)
        for (int a = 0; a < 3; ++a) {
            real acc = 0, dacc = 0;
            for (int m = 0; m < M; ++m) {
                const int64_t idx = j + kmin + m;
                const real v = (idx >= 0 && idx < nk) ? (real)o->Rtab[(int64_t)(i * 3 + a) * nk + idx] : (real)0;
                acc += w[m] * v;
                dacc += dw[m] * v;
            }
            R[i][a] = acc;
            V[i][a] = dacc / dtk;
        }
}

typedef struct {
    real R[3][3];  /* spacecraft positions [m] */
    real nh[6][3]; /* link unit vectors, sender -> receiver (G7) */
    real L[6];     /* light travel times [s] */
} geom_t;

static void orbit_geometry(const orbit_ctx *o, int64_t n, geom_t *g)
{
    const real c = ORC_C_LIGHT;
    real V[3][3] = { { 0 } };
    if (o->d.mode == ORC_ORBIT_TABLES) {
        for (int i = 0; i < 3; ++i)
            for (int a = 0; a < 3; ++a) g->R[i][a] = (real)o->Rtab[(int64_t)(i * 3 + a) * o->d.n + n];
    } else if (o->d.mode == ORC_ORBIT_KNOTS) {
        knot_positions(o, (real)o->d.t0 + (real)n * (real)o->d.dt, g->R, V);
    } else {
        const real t = (real)o->d.t0 + (real)n * (real)o->d.dt;
        const real R = o->d.R_m, L = o->d.arm_m;
        const real adot = 2 * R_PI / (real)o->d.period_s;
        const real alpha = adot * t + (real)o->d.alpha0;
        const real e = L / (2 * R_SQRT((real)3) * R);
        for (int i = 0; i < 3; ++i) {
            const real b = 2 * R_PI * (real)i / 3 + (real)o->d.rot0;
            g->R[i][0] = R * R_COS(alpha) + (real)0.5 * e * R * (R_COS(2 * alpha - b) - 3 * R_COS(b));
            g->R[i][1] = R * R_SIN(alpha) + (real)0.5 * e * R * (R_SIN(2 * alpha - b) - 3 * R_SIN(b));
            g->R[i][2] = -R_SQRT((real)3) * e * R * R_COS(alpha - b);
            V[i][0] = -R * adot * R_SIN(alpha) - e * R * adot * R_SIN(2 * alpha - b);
            V[i][1] = R * adot * R_COS(alpha) + e * R * adot * R_COS(2 * alpha - b);
            V[i][2] = R_SQRT((real)3) * e * R * adot * R_SIN(alpha - b);
        }
    }
    for (int l = 0; l < 6; ++l) {
        const int s = LINK_S[l], r = LINK_R[l];
        real dvec[3], len2 = 0;
        for (int a = 0; a < 3; ++a) {
            dvec[a] = g->R[r][a] - g->R[s][a]; /* L_l n_l ~ R_r - R_s */
            len2 += dvec[a] * dvec[a];
        }
        const real len = R_SQRT(len2);
        for (int a = 0; a < 3; ++a) g->nh[l][a] = dvec[a] / len;
        if (o->d.mode == ORC_ORBIT_STATIC_EQUALARM) {
            g->L[l] = (real)o->d.arm_m / c; /* "equal and constant" delays */
        } else if (o->d.mode == ORC_ORBIT_KEPLERIAN || o->d.mode == ORC_ORBIT_KNOTS) {
            /* first-order light time: L_l != L_-l through the sender velocity (B22) */
            real nv = 0;
            for (int a = 0; a < 3; ++a) nv += g->nh[l][a] * V[s][a];
            g->L[l] = (len / c) * (1 + nv / c);
        } else {
            g->L[l] = (real)o->Ltab[(int64_t)l * o->d.n + n];
        }
    }
}

/* ---------------------------------------------------------------------------------- */
/* O2  source frame, Eq. (2.1) with reading G1; O3 antenna patterns (2.2)-(2.4)        */
/* ---------------------------------------------------------------------------------- */
typedef struct { real k[3], u[3], v[3], c2, s2; } frame_t;

static void source_frame(const orc_source *s, frame_t *f)
{
    const real b = s->beta, l = s->lambda, p = s->psi;
    f->k[0] = -R_COS(b) * R_COS(l); f->k[1] = -R_COS(b) * R_SIN(l); f->k[2] = -R_SIN(b); /* -e_r     */
    f->u[0] = R_SIN(l);             f->u[1] = -R_COS(l);            f->u[2] = 0;         /* -e_phi   */
    f->v[0] = -R_SIN(b) * R_COS(l); f->v[1] = -R_SIN(b) * R_SIN(l); f->v[2] = R_COS(b);  /* -e_theta */
    f->c2 = R_COS(2 * p);
    f->s2 = R_SIN(2 * p);
}

static real dot3(const real *a, const real *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

/* F^+_l, F^x_l such that H_l = F^+ h_+ + F^x h_x  ( = xi^+ h^SSB_+ + xi^x h^SSB_x, (2.2)+(2.3), G17 ) */
static void antenna(const frame_t *f, const real *nh, real *Fp, real *Fc)
{
    const real un = dot3(f->u, nh), vn = dot3(f->v, nh);
    const real xip = un * un - vn * vn; /* (2.4a) */
    const real xic = 2 * un * vn;       /* (2.4b) */
    *Fp = xip * f->c2 + xic * f->s2;
    *Fc = -xip * f->s2 + xic * f->c2;
}

/* ---------------------------------------------------------------------------------- */
/* O10 margins (reading G11)                                                          */
/* ---------------------------------------------------------------------------------- */
typedef struct { int64_t m1, m2, w, lo, hi; } margins_t;

static int64_t iceil(double x) { return (int64_t)ceil(x); }

static void margins(const orc_orbit_desc *d, int gen, int order, int fd_order, margins_t *m)
{
    const int M = order + 1;
    const double c = ORC_C_LIGHT;
    m->m1 = iceil(1.02 * (d->R_m + d->arm_m) / c / d->dt) + M / 2;
    m->m2 = iceil((gen == ORC_GEN_20 ? 7.2 : 3.1) * (d->arm_m / c) / d->dt) + M / 2;
    m->w = fd_order / 2;
    m->lo = m->m1 + m->m2 + 2 * m->w;
    m->hi = m->m1 + M / 2 + 2 * m->w;
}

/* ---------------------------------------------------------------------------------- */
/* O5  single-link response, Eq. (2.5) with delays (2.6) (readings G3, G4)             */
/* ---------------------------------------------------------------------------------- */
static void links_full_at(const orbit_ctx *o, const frame_t *f, const double *hp, const double *hc,
                          int64_t n, int order, real y[6])
{
    const real c = ORC_C_LIGHT, dt = o->d.dt;
    geom_t g;
    orbit_geometry(o, n, &g);
    for (int l = 0; l < 6; ++l) {
        const int s = LINK_S[l], r = LINK_R[l];
        real Fp, Fc;
        antenna(f, g.nh[l], &Fp, &Fc);
        const real kn = dot3(f->k, g.nh[l]);
        const real delta_s = g.L[l] + dot3(f->k, g.R[s]) / c; /* (2.6a) */
        const real delta_r = dot3(f->k, g.R[r]) / c;          /* (2.6b) */
        const real Hs = Fp * interp_input(hp, o->d.n, n, delta_s, dt, order) +
                        Fc * interp_input(hc, o->d.n, n, delta_s, dt, order);
        const real Hr = Fp * interp_input(hp, o->d.n, n, delta_r, dt, order) +
                        Fc * interp_input(hc, o->d.n, n, delta_r, dt, order);
        y[l] = (Hs - Hr) / (2 * (1 - kn)); /* (2.5) */
    }
}

/* LFA single link, Eq. (3.1) = (B10), retarded time (B1) (readings G14, G16); only l = +1,+2,+3 */
static void links_lfa_at(const orbit_ctx *o, const frame_t *f, const real *gp, const real *gc,
                         int64_t g0, int64_t glen, int64_t n, int order, real y[6])
{
    const real c = ORC_C_LIGHT, dt = o->d.dt;
    geom_t g;
    orbit_geometry(o, n, &g);
    for (int l = 0; l < 6; ++l) y[l] = 0; /* "the rest are set to zero" */
    for (int l = 0; l < 3; ++l) {
        const int s = LINK_S[l], r = LINK_R[l];
        real Fp, Fc;
        antenna(f, g.nh[l], &Fp, &Fc);
        const real tau = g.L[l] / 2 + (dot3(f->k, g.R[s]) + dot3(f->k, g.R[r])) / (2 * c); /* (B1) */
        const real dHp = interp_series(gp, g0, glen, n, tau, dt, order);
        const real dHc = interp_series(gc, g0, glen, n, tau, dt, order);
        y[l] = -(g.L[l] / 2) * (Fp * dHp + Fc * dHc); /* (B10), L_l in seconds */
    }
}

/* Extended LFA single link, l = +1,+2,+3:
 *   point = 0: central, tau of (B1), series (B4) truncated after `terms` terms (terms = 1 is (B10)):
 *       y = -(L_l / 2) { dH/dt + (1/6) [ (L_l / 2)(1 - k.n_l) ]^2 d^3H/dt^3 } (tau),   tau-derivatives = t-derivatives (B7)
 *   point = 1: backward (epsilon = 0), Eq. (B13):  y = -(L_l / 2) dH/dt (t - L_l - k.R_s / c)      leading order
 *   point = 2: forward  (epsilon = 1), Eq. (B14):  y = -(L_l / 2) dH/dt (t - k.R_r / c)            leading order
 * with H = F+ h+ + Fx hx and the antenna patterns at reception time (B9), (G3, G17).  g1 = dh/dt, g3 = d^3h/dt^3 on
 * the grid. */
enum { ORC_LFA_CENTRAL = 0, ORC_LFA_BACKWARD = 1, ORC_LFA_FORWARD = 2 };
static void links_lfa_ext_at(const orbit_ctx *o, const frame_t *f, const real *gp, const real *gc, const real *g3p,
                             const real *g3c, int64_t g0, int64_t glen, int64_t n, int order, int terms, int point,
                             real y[6])
{
    const real c = ORC_C_LIGHT, dt = o->d.dt;
    geom_t g;
    orbit_geometry(o, n, &g);
    for (int l = 0; l < 6; ++l) y[l] = 0;
    for (int l = 0; l < 3; ++l) {
        const int s = LINK_S[l], r = LINK_R[l];
        real Fp, Fc;
        antenna(f, g.nh[l], &Fp, &Fc);
        const real ds = g.L[l] + dot3(f->k, g.R[s]) / c, dr = dot3(f->k, g.R[r]) / c; /* (2.6) */
        real tau;
        if (point == ORC_LFA_CENTRAL) tau = g.L[l] / 2 + (dot3(f->k, g.R[s]) + dot3(f->k, g.R[r])) / (2 * c); /* (B1) */
        else if (point == ORC_LFA_BACKWARD) tau = ds;                                                          /* tau_0 */
        else tau = dr;                                                                                         /* tau_1 */
        real dH = Fp * interp_series(gp, g0, glen, n, tau, dt, order) + Fc * interp_series(gc, g0, glen, n, tau, dt, order);
        if (point == ORC_LFA_CENTRAL && terms >= 2) {
            const real half = (g.L[l] / 2) * (1 - dot3(f->k, g.nh[l]));   /* (delta_s - delta_r) / 2 with L n = R_r - R_s */
            const real d3H = Fp * interp_series(g3p, g0, glen, n, tau, dt, order) +
                             Fc * interp_series(g3c, g0, glen, n, tau, dt, order);
            dH += half * half / 6 * d3H;                                  /* m = 1 term of (B4) */
        }
        y[l] = -(g.L[l] / 2) * dH;
    }
}

/* all six LFA links (O14): Eq. (B10) at the retarded time (B1) of each link with ITS OWN light time L_l (l = -1, -2, -3
 * differ from +1, +2, +3 by L_-l != L_l only: the antenna patterns are even in n_l and R_s + R_r is symmetric) */
static void links_lfa6_at(const orbit_ctx *o, const frame_t *f, const real *gp, const real *gc, int64_t g0,
                          int64_t glen, int64_t n, int order, real y[6])
{
    const real c = ORC_C_LIGHT, dt = o->d.dt;
    geom_t g;
    orbit_geometry(o, n, &g);
    for (int l = 0; l < 6; ++l) {
        const int s = LINK_S[l], r = LINK_R[l];
        real Fp, Fc;
        antenna(f, g.nh[l], &Fp, &Fc);
        const real tau = g.L[l] / 2 + (dot3(f->k, g.R[s]) + dot3(f->k, g.R[r])) / (2 * c); /* (B1) */
        const real dH = Fp * interp_series(gp, g0, glen, n, tau, dt, order) + Fc * interp_series(gc, g0, glen, n, tau, dt, order);
        y[l] = -(g.L[l] / 2) * dH;                                                          /* (B10) */
    }
}

/* ---------------------------------------------------------------------------------- */
/* O6  Michelson TDI, Eqs. (2.7), (2.8) with G8, G9, G12; ch = 0,1,2 -> X,Y,Z          */
/* ---------------------------------------------------------------------------------- */
static int cyc(int label, int times) /* 1->2->3->1 on |l|, sign kept */
{
    int a = label > 0 ? label : -label;
    for (int i = 0; i < times; ++i) a = a % 3 + 1;
    return label > 0 ? a : -a;
}

typedef struct { const real *y[6]; int64_t y0, ylen; } yseries_t;

static real ydel(const yseries_t *ys, int label, int64_t n, real delay, real dt, int order)
{
    const int l = link_index(label);
    if (delay == 0) { /* undelayed terms are taken from the grid */
        const int64_t i = n - ys->y0;
        return (i >= 0 && i < ys->ylen) ? ys->y[l][i] : (real)0;
    }
    return interp_series(ys->y[l], ys->y0, ys->ylen, n, delay, dt, order);
}

static real michelson_at(const yseries_t *ys, const real Lsec[6], int ch, int gen, int64_t n, real dt,
                         int order)
{
    /* X uses |l| = 2, 3; Y and Z by cyclic permutation */
    const int p2 = cyc(2, ch), p3 = cyc(3, ch);
    const real Lp2 = Lsec[link_index(p2)], Lm2 = Lsec[link_index(-p2)];
    const real Lp3 = Lsec[link_index(p3)], Lm3 = Lsec[link_index(-p3)];
#define Y(label, delay) ydel(ys, (label), n, (delay), dt, order)
    /* Eq. (2.7), term by term in the printed order (y_1-32, y_231, y_123, y_3-21 for X) */
    real X = Y(-p3, Lm2 + Lp2 + Lp3) - Y(-p3, Lp3)
           + Y(+p3, Lp2 + Lm2)       - Y(+p3, (real)0)
           + Y(+p2, Lm2)             - Y(+p2, Lm2 + Lm3 + Lp3)
           + Y(-p2, (real)0)         - Y(-p2, Lm3 + Lp3);
    if (gen == ORC_GEN_20) {
        /* Eq. (2.8); the 7th term with reading G9 (L_-2 + L_2 + 2 L_3 + 2 L_-3) */
        X += Y(-p3, Lm2 + Lp2 + 2 * Lp3 + Lm3)         - Y(-p3, 2 * Lp3 + Lm3 + 2 * Lm2 + 2 * Lp2)
           + Y(+p3, Lm2 + Lp2 + Lp3 + Lm3)             - Y(+p3, Lp3 + Lm3 + 2 * Lm2 + 2 * Lp2)
           + Y(+p2, 2 * Lm2 + Lp2 + 2 * Lp3 + 2 * Lm3) - Y(+p2, Lp3 + Lm3 + 2 * Lm2 + Lp2)
           + Y(-p2, Lm2 + Lp2 + 2 * Lp3 + 2 * Lm3)     - Y(-p2, Lp3 + Lm3 + Lm2 + Lp2);
    }
#undef Y
    return X;
}

/* O15 Sagnac-type combinations alpha, beta, gamma ("Sagnac-type observables emulate the interference
 * pattern generated by photons propagating in clockwise and counterclockwise directions around the constellation"; the
 * paper prints no equation for them -- reading G33 -- so the textbook definition is written out in the link labelling of
 * P:81, where link +1 runs 3 -> 2, +2: 1 -> 3, +3: 2 -> 1 and -1: 2 -> 3, -2: 3 -> 1, -3: 1 -> 2).
 * The beam that leaves spacecraft 1, goes round 1 -> 3 -> 2 -> 1 and is read at t, and the one going round 1 -> 2 -> 3 -> 1:
 *     S+ = y_{+3} + D_{+3} y_{+1} + D_{+3} D_{+1} y_{+2},          S- = y_{-2} + D_{-2} y_{-1} + D_{-2} D_{-1} y_{-3}
 * In laser-noise terms y_l(t) = p_s(t - L_l) - p_r(t) each telescopes to p_1(t - T+-) - p_1(t) with the round-trip times
 * T+ = L_3 + L_1 + L_2, T- = L_-2 + L_-1 + L_-3.  Then
 *     gen 1.5:  alpha = S+ - S-                                     (6 terms; free of laser noise where T+ = T-)
 *     gen 2.0:  alpha = (S+ + D_{T+} S-) - (S- + D_{T-} S+)         (12 terms; free of laser noise for any constant L_l != L_-l)
 * beta, gamma by the cyclic permutation 1 -> 2 -> 3 -> 1 of the link labels.  Every delay is evaluated at t, as in
 * O6, so the operators commute and a product of delays is the sum of the light times. */
static real sagnac_at(const yseries_t *ys, const real Lsec[6], int ch, int gen, int64_t n, real dt, int order)
{
    const int c3 = cyc(3, ch), c1 = cyc(1, ch), c2 = cyc(2, ch);   /* the links +3, +1, +2 of alpha, permuted */
    const real Lp3 = Lsec[link_index(c3)], Lp1 = Lsec[link_index(c1)], Lp2 = Lsec[link_index(c2)];
    const real Lm2 = Lsec[link_index(-c2)], Lm1 = Lsec[link_index(-c1)], Lm3 = Lsec[link_index(-c3)];
    const real Tp = Lp3 + Lp1 + Lp2, Tm = Lm2 + Lm1 + Lm3;
#define Y(label, delay) ydel(ys, (label), n, (delay), dt, order)
    real a = Y(+c3, (real)0) + Y(+c1, Lp3) + Y(+c2, Lp3 + Lp1)
           - Y(-c2, (real)0) - Y(-c1, Lm2) - Y(-c3, Lm2 + Lm1);
    if (gen == ORC_GEN_20) {
        a += Y(-c2, Tp) + Y(-c1, Tp + Lm2) + Y(-c3, Tp + Lm2 + Lm1)
           - Y(+c3, Tm) - Y(+c1, Tm + Lp3) - Y(+c2, Tm + Lp3 + Lp1);
    }
#undef Y
    return a;
}

/* O12 properly nested delays (the comparison case of P:151 -- the paper itself evaluates every L_l at t).
 * Delay operators act as (D_l f)(t) = f(t - L_l(t)), so D_a D_b f (t) = f(t - L_a(t) - L_b(t - L_a(t))): walking a
 * chain of links c_1 c_2 .. c_m backwards from the reception time,
 *     d_0 = 0,   d_j = d_{j-1} + L_{c_j}(t - d_{j-1}),
 * and the term is y(t - d_m).  With a = D_{-2} D_2, b = D_3 D_{-3} (for X; cyclic for Y, Z) and P = y_123, Q = y_3-21,
 * U = y_1-32, W = y_231:
 *     X_1.5 = (1 - b)(Q + D_{-2} P) - (1 - a)(W + D_3 U)
 *     X_2.0 = (1 - b - b a + a b b)(Q + D_{-2} P) - (1 - a - a b + b a a)(W + D_3 U)
 * which for commuting (un-nested) delays are Eqs. (2.7) and (2.8) term by term (with G9).  The light travel time at
 * an off-grid time is the centred Lagrange interpolation of order p_L of the sampled series L_l(t_n) (reading G29);
 * the link series are interpolated once per term at the accumulated delay, as in O6. */
typedef struct { const real *L[6]; int64_t l0, llen; } lseries_t;

static real chain_delay(const lseries_t *Ls, int64_t n, real dt, int order_L, int len, const int *labels)
{
    real d = 0;
    for (int j = 0; j < len; ++j) {
        const int l = link_index(labels[j]);
        if (d == 0) d += Ls->L[l][n - Ls->l0];                                           /* on the grid */
        else d += interp_series(Ls->L[l], Ls->l0, Ls->llen, n, d, dt, order_L);
    }
    return d;
}

static real michelson_nested_at(const yseries_t *ys, const lseries_t *Ls, int ch, int gen, int64_t n, real dt,
                                int order, int order_L)
{
    const int p2 = cyc(2, ch), p3 = cyc(3, ch);
#define CH(...) chain_delay(Ls, n, dt, order_L, (int)(sizeof((int[]){ __VA_ARGS__ }) / sizeof(int)), (int[]){ __VA_ARGS__ })
#define Y(label, delay) ydel(ys, (label), n, (delay), dt, order)
    /* (1 - b)(Q + D_-2 P) - (1 - a)(W + D_3 U) */
    real X = Y(-p2, (real)0) + Y(+p2, CH(-p2))
           - Y(-p2, CH(+p3, -p3)) - Y(+p2, CH(+p3, -p3, -p2))
           - Y(+p3, (real)0) - Y(-p3, CH(+p3))
           + Y(+p3, CH(-p2, +p2)) + Y(-p3, CH(-p2, +p2, +p3));
    if (gen == ORC_GEN_20) {
        /* (- b a + a b b)(Q + D_-2 P) - (- a b + b a a)(W + D_3 U) */
        X += -Y(-p2, CH(+p3, -p3, -p2, +p2)) - Y(+p2, CH(+p3, -p3, -p2, +p2, -p2))
           + Y(-p2, CH(-p2, +p2, +p3, -p3, +p3, -p3)) + Y(+p2, CH(-p2, +p2, +p3, -p3, +p3, -p3, -p2))
           + Y(+p3, CH(-p2, +p2, +p3, -p3)) + Y(-p3, CH(-p2, +p2, +p3, -p3, +p3))
           - Y(+p3, CH(+p3, -p3, -p2, +p2, -p2, +p2)) - Y(-p3, CH(+p3, -p3, -p2, +p2, -p2, +p2, +p3));
    }
#undef Y
#undef CH
    return X;
}

/* the sampled light travel times on [l0, l0 + len) in working precision */
static int lseries_alloc(const orbit_ctx *o, int64_t l0, int64_t len, real *buf[6], lseries_t *Ls)
{
    for (int l = 0; l < 6; ++l)
        if (!(buf[l] = (real *)calloc((size_t)(len > 0 ? len : 1), sizeof(real)))) return ORC_EINVAL;
#pragma omp parallel for
    for (int64_t i = 0; i < len; ++i) {
        geom_t g;
        orbit_geometry(o, l0 + i, &g);
        for (int l = 0; l < 6; ++l) buf[l][i] = g.L[l];
    }
    for (int l = 0; l < 6; ++l) Ls->L[l] = buf[l];
    Ls->l0 = l0;
    Ls->llen = len;
    return ORC_OK;
}

/* LFA Michelson, Eq. (B25) (gen 1.5) / (B33) (gen 2.0); dy[l] = FD1 or FD2 of y_l, l = +1,+2,+3 */
static real michelson_lfa_at(const yseries_t *dys, const real Lsec[6], int ch, int gen, int64_t n,
                             real dt, int order)
{
    const int p2 = cyc(2, ch), p3 = cyc(3, ch);
    const real L2 = Lsec[link_index(p2)], L3 = Lsec[link_index(p3)]; /* positive-link values, G14 */
    /* y_123 is link +2 (p2), y_231 is link +3 (p3) */
    if (gen == ORC_GEN_15)
        return 4 * (L3 * ydel(dys, +p2, n, L3 + L2 / 2, dt, order) -
                    L2 * ydel(dys, +p3, n, L2 + L3 / 2, dt, order));
    return 8 * (L2 + L3) * (L3 * ydel(dys, +p2, n, 2 * L3 + 3 * L2 / 2, dt, order) -
                            L2 * ydel(dys, +p3, n, 2 * L2 + 3 * L3 / 2, dt, order));
}

/* O14: the Michelson variables Taylor-expanded WITHOUT the link-reversal symmetry, Eq. (B20)
 * (gen 1.5) and Eq. (B30) P:894 (gen 2.0): all six LFA links, first and second (second and third) time derivatives of
 * each, evaluated at the mid-points (B18) / (B31) of the two arms (reading G13: the printed (B21) / (B32) disagree with
 * them; d/dtau = d/dt as in (B7)).  For X, with P = y_123 (+p2), Q = y_3-21 (-p2), U = y_1-32 (-p3), W = y_231 (+p3),
 * a = L_-p2 + L_p2, b = L_-p3 + L_p3:
 *   X_1.5 = b [P' - (L_-p2 / 2) P''](tau_2) + b [Q' + (L_-p2 / 2) Q''](tau_2) - a [U' - (L_p3 / 2) U''](tau_3) - a [W' + (L_p3 / 2) W''](tau_3)
 *     tau_2 = t - (L_-p3 + L_-p2 + L_p3) / 2,   tau_3 = t - (L_-p2 + L_p2 + L_p3) / 2                              (B18)
 *   X_2.0 = (a + b) { b [P'' - (L_-p2 / 2) P'''](tau_2) + b [Q'' + (L_-p2 / 2) Q'''](tau_2)
 *                    - a [U'' - (L_p3 / 2) U'''](tau_3) - a [W'' + (L_p3 / 2) W'''](tau_3) }
 *     tau_2 = t - L_-p3 - L_-p2 - L_p3 - L_p2 / 2,   tau_3 = t - L_-p2 - L_p2 - L_p3 - L_-p3 / 2                    (B31)
 * dlo[l], dhi[l]: the lower and the higher of the two derivatives of link l on the grid. */
static real michelson_b20_at(const yseries_t *dlo, const yseries_t *dhi, const real Lsec[6], int ch, int gen, int64_t n,
                             real dt, int order)
{
    const int p2 = cyc(2, ch), p3 = cyc(3, ch);
    const real Lp2 = Lsec[link_index(p2)], Lm2 = Lsec[link_index(-p2)];
    const real Lp3 = Lsec[link_index(p3)], Lm3 = Lsec[link_index(-p3)];
    const real a = Lm2 + Lp2, b = Lm3 + Lp3;
    real d2, d3, pre;
    if (gen == ORC_GEN_15) {
        d2 = (Lm3 + Lm2 + Lp3) / 2;
        d3 = (Lm2 + Lp2 + Lp3) / 2;
        pre = 1;
    } else {
        d2 = Lm3 + Lm2 + Lp3 + Lp2 / 2;
        d3 = Lm2 + Lp2 + Lp3 + Lm3 / 2;
        pre = a + b;
    }
#define DLO(label, d) ydel(dlo, (label), n, (d), dt, order)
#define DHI(label, d) ydel(dhi, (label), n, (d), dt, order)
    return pre * (b * (DLO(+p2, d2) - (Lm2 / 2) * DHI(+p2, d2)) + b * (DLO(-p2, d2) + (Lm2 / 2) * DHI(-p2, d2))
                  - a * (DLO(-p3, d3) - (Lp3 / 2) * DHI(-p3, d3)) - a * (DLO(+p3, d3) + (Lp3 / 2) * DHI(+p3, d3)));
#undef DLO
#undef DHI
}

/* O7  Eq. (2.9) */
static void aet(real X, real Y, real Z, real *A, real *E, real *T)
{
    *A = (Z - X) / R_SQRT((real)2);
    *E = (X - 2 * Y + Z) / R_SQRT((real)6);
    *T = (X + Y + Z) / R_SQRT((real)3);
}

/* O9  hybrid weights, Eqs. (4.1), (4.5) (reading G18) and the raised-cosine taper (G20) */
static void hybrid_weights(const orc_hybrid *h, real t, real *w_lfa, real *w_full)
{
    const real th = h->t_hyb, T = h->window_s;
    if (h->taper == ORC_TAPER_SIGMOID) {
        const real sg = h->sigma_s;
        *w_lfa = (t <= th + T / 2) ? 1 / (1 + R_EXP((t - th) / sg)) : (real)0;   /* Sigma(+1) */
        *w_full = (t >= th - T / 2) ? 1 / (1 + R_EXP(-(t - th) / sg)) : (real)0; /* Sigma(-1) */
    } else {
        const real x = (t - th + T / 2) / T;
        if (x <= 0) *w_full = 0;
        else if (x >= 1) *w_full = 1;
        else *w_full = (real)0.5 * (1 - R_COS(R_PI * x));
        *w_lfa = 1 - *w_full;
    }
}

/* ---------------------------------------------------------------------------------- */
/* drivers: outputs for absolute samples [nb, ne) of every source, compact rows of      */
/* length ne - nb.  Any output pointer may be NULL.                                     */
/* ---------------------------------------------------------------------------------- */
typedef struct {
    real *y[6];      /* link series on [y0, y0 + ylen) */
    real *X[3];      /* Michelson on [nb, ne) */
    int64_t y0, ylen;
} work_t;

static int64_t imax(int64_t a, int64_t b) { return a > b ? a : b; }
static int64_t imin(int64_t a, int64_t b) { return a < b ? a : b; }

static int work_alloc(work_t *w, int64_t y0, int64_t ylen, int64_t nout)
{
    memset(w, 0, sizeof *w);
    w->y0 = y0;
    w->ylen = ylen;
    for (int l = 0; l < 6; ++l)
        if (!(w->y[l] = (real *)calloc((size_t)imax(ylen, 1), sizeof(real)))) return ORC_EINVAL;
    for (int c = 0; c < 3; ++c)
        if (!(w->X[c] = (real *)calloc((size_t)imax(nout, 1), sizeof(real)))) return ORC_EINVAL;
    return ORC_OK;
}
static void work_free(work_t *w)
{
    for (int l = 0; l < 6; ++l) free(w->y[l]);
    for (int c = 0; c < 3; ++c) free(w->X[c]);
}

/* full response for one source: y (6 links) on the halo range, X,Y,Z on [nb,ne) */
static int g_nested_order = 0; /* 0: every L_l at t (the paper); p_L > 0: nested delays (O12), set per call */
static int g_sagnac = 0;       /* 1: alpha, beta, gamma of O15 in place of X, Y, Z, set per call */

static int full_one(const orbit_ctx *o, const frame_t *f, const double *hp, const double *hc, int gen,
                    int order, const margins_t *mg, int64_t lo, int64_t hi, int64_t nb, int64_t ne,
                    work_t *w)
{
    const int64_t N = o->d.n;
    const int64_t y0 = imax(0, nb - mg->m2), y1 = imin(N, ne + (order + 1) / 2 + 1);
    if (work_alloc(w, y0, y1 - y0, ne - nb)) return ORC_EINVAL;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t m = y0; m < y1; ++m) {
        if (m < mg->m1 || m >= N - mg->m1) continue; /* margin: y = 0 (G11) */
        real y[6];
        links_full_at(o, f, hp, hc, m, order, y);
        for (int l = 0; l < 6; ++l) w->y[l][m - y0] = y[l];
    }
    yseries_t ys = { { w->y[0], w->y[1], w->y[2], w->y[3], w->y[4], w->y[5] }, y0, y1 - y0 };
    if (g_nested_order > 0) { /* O12 */
        real *buf[6];
        lseries_t Ls;
        if (lseries_alloc(o, y0, y1 - y0, buf, &Ls)) return ORC_EINVAL;
#pragma omp parallel for schedule(dynamic, 64)
        for (int64_t n = nb; n < ne; ++n) {
            if (n < lo || n >= N - hi) continue;
            for (int c = 0; c < 3; ++c)
                w->X[c][n - nb] = michelson_nested_at(&ys, &Ls, c, gen, n, (real)o->d.dt, order, g_nested_order);
        }
        for (int l = 0; l < 6; ++l) free(buf[l]);
        return ORC_OK;
    }
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t n = nb; n < ne; ++n) {
        if (n < lo || n >= N - hi) continue; /* margin: X = 0 */
        geom_t g;
        orbit_geometry(o, n, &g); /* every delay evaluated at t_n */
        for (int c = 0; c < 3; ++c)
            w->X[c][n - nb] = g_sagnac ? sagnac_at(&ys, g.L, c, gen, n, (real)o->d.dt, order)
                                       : michelson_at(&ys, g.L, c, gen, n, (real)o->d.dt, order);
    }
    return ORC_OK;
}

/* LFA response for one source */
/* half width of the widest stencil applied to the strain: the first derivative (w), or with the m = 1 term of (B4)
 * the third derivative (w + 1) */
static int64_t lfa_strain_width(int fd_order, int terms) { return fd_order / 2 + (terms >= 2 ? 1 : 0); }

static int lfa_one_ext(const orbit_ctx *o, const frame_t *f, const double *hp, const double *hc, int gen,
                       int order, int fd_order, int terms, int point, const margins_t *mg, int64_t nb, int64_t ne,
                       work_t *w)
{
    const int64_t N = o->d.n, wd = mg->w, ws = lfa_strain_width(fd_order, terms), extra = ws - wd;
    const real dt = o->d.dt;
    /* the same ranges as lfa_one; the link series is valid where the widest strain stencil fits: m1 + ws */
    const int64_t d0 = imax(0, nb - mg->m2), d1 = imin(N, ne + (order + 1) / 2 + 1);
    const int64_t y0 = imax(0, d0 - wd), y1 = imin(N, d1 + wd);
    const int64_t g0 = imax(0, y0 - mg->m1), g1 = imin(N, y1 + mg->m1);
    real *gp = (real *)calloc((size_t)imax(g1 - g0, 1), sizeof(real));
    real *gc = (real *)calloc((size_t)imax(g1 - g0, 1), sizeof(real));
    real *g3p = (real *)calloc((size_t)imax(g1 - g0, 1), sizeof(real));
    real *g3c = (real *)calloc((size_t)imax(g1 - g0, 1), sizeof(real));
    real *dy[3] = { 0, 0, 0 };
    for (int l = 0; l < 3; ++l) dy[l] = (real *)calloc((size_t)imax(d1 - d0, 1), sizeof(real));
    if (!gp || !gc || !g3p || !g3c || !dy[0] || !dy[1] || !dy[2] || work_alloc(w, y0, y1 - y0, ne - nb)) return ORC_EINVAL;
#pragma omp parallel for
    for (int64_t i = g0; i < g1; ++i) {
        if (i < ws || i >= N - ws) continue;
        gp[i - g0] = fd1_in(hp, i, dt, fd_order);
        gc[i - g0] = fd1_in(hc, i, dt, fd_order);
        if (terms >= 2) {
            g3p[i - g0] = fd3_in(hp, i, dt, fd_order);
            g3c[i - g0] = fd3_in(hc, i, dt, fd_order);
        }
    }
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t m = y0; m < y1; ++m) {
        if (m < mg->m1 + ws || m >= N - mg->m1 - ws) continue;
        real y[6];
        links_lfa_ext_at(o, f, gp, gc, g3p, g3c, g0, g1 - g0, m, order, terms, point, y);
        for (int l = 0; l < 6; ++l) w->y[l][m - y0] = y[l];
    }
#pragma omp parallel for
    for (int64_t i = d0; i < d1; ++i) {
        if (i < mg->m1 + ws + wd || i >= N - mg->m1 - ws - wd) continue;
        for (int l = 0; l < 3; ++l)
            dy[l][i - d0] = (gen == ORC_GEN_15) ? fd1_r(w->y[l], i - y0, dt, fd_order)
                                                : fd2_r(w->y[l], i - y0, dt, fd_order);
    }
    yseries_t dys = { { dy[0], dy[1], dy[2], 0, 0, 0 }, d0, d1 - d0 };
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t n = nb; n < ne; ++n) {
        if (n < mg->lo + extra || n >= N - mg->hi - extra) continue;
        geom_t g;
        orbit_geometry(o, n, &g);
        for (int c = 0; c < 3; ++c)
            w->X[c][n - nb] = michelson_lfa_at(&dys, g.L, c, gen, n, dt, order);
    }
    free(gp); free(gc); free(g3p); free(g3c);
    for (int l = 0; l < 3; ++l) free(dy[l]);
    return ORC_OK;
}

/* LFA response without the link-reversal symmetry (O14) for one source; xw = 1 for gen 2.0 (third-derivative stencil) */
static int lfa6_one(const orbit_ctx *o, const frame_t *f, const double *hp, const double *hc, int gen, int order,
                    int fd_order, const margins_t *mg, int64_t nb, int64_t ne, work_t *w)
{
    const int64_t N = o->d.n, wd = mg->w, xw = gen == ORC_GEN_20 ? 1 : 0, wy = wd + xw;
    const real dt = o->d.dt;
    const int64_t d0 = imax(0, nb - mg->m2), d1 = imin(N, ne + (order + 1) / 2 + 1);
    const int64_t y0 = imax(0, d0 - wy), y1 = imin(N, d1 + wy);
    const int64_t g0 = imax(0, y0 - mg->m1), g1 = imin(N, y1 + mg->m1);
    real *gp = (real *)calloc((size_t)imax(g1 - g0, 1), sizeof(real));
    real *gc = (real *)calloc((size_t)imax(g1 - g0, 1), sizeof(real));
    real *lo[6], *hi[6];
    for (int l = 0; l < 6; ++l) {
        lo[l] = (real *)calloc((size_t)imax(d1 - d0, 1), sizeof(real));
        hi[l] = (real *)calloc((size_t)imax(d1 - d0, 1), sizeof(real));
        if (!lo[l] || !hi[l]) return ORC_EINVAL;
    }
    if (!gp || !gc || work_alloc(w, y0, y1 - y0, ne - nb)) return ORC_EINVAL;
#pragma omp parallel for
    for (int64_t i = g0; i < g1; ++i) {
        if (i < wd || i >= N - wd) continue;
        gp[i - g0] = fd1_in(hp, i, dt, fd_order);
        gc[i - g0] = fd1_in(hc, i, dt, fd_order);
    }
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t m = y0; m < y1; ++m) {
        if (m < mg->m1 + wd || m >= N - mg->m1 - wd) continue;
        real y[6];
        links_lfa6_at(o, f, gp, gc, g0, g1 - g0, m, order, y);
        for (int l = 0; l < 6; ++l) w->y[l][m - y0] = y[l];
    }
#pragma omp parallel for
    for (int64_t i = d0; i < d1; ++i) {
        if (i < mg->m1 + wd + wy || i >= N - mg->m1 - wd - wy) continue;
        for (int l = 0; l < 6; ++l) {
            if (gen == ORC_GEN_15) {
                lo[l][i - d0] = fd1_r(w->y[l], i - y0, dt, fd_order);
                hi[l][i - d0] = fd2_r(w->y[l], i - y0, dt, fd_order);
            } else {
                lo[l][i - d0] = fd2_r(w->y[l], i - y0, dt, fd_order);
                hi[l][i - d0] = fd3_r(w->y[l], i - y0, dt, fd_order);
            }
        }
    }
    yseries_t slo = { { lo[0], lo[1], lo[2], lo[3], lo[4], lo[5] }, d0, d1 - d0 };
    yseries_t shi = { { hi[0], hi[1], hi[2], hi[3], hi[4], hi[5] }, d0, d1 - d0 };
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t n = nb; n < ne; ++n) {
        if (n < mg->lo + xw || n >= N - mg->hi - xw) continue;
        geom_t g;
        orbit_geometry(o, n, &g);
        for (int c = 0; c < 3; ++c) w->X[c][n - nb] = michelson_b20_at(&slo, &shi, g.L, c, gen, n, dt, order);
    }
    free(gp); free(gc);
    for (int l = 0; l < 6; ++l) { free(lo[l]); free(hi[l]); }
    return ORC_OK;
}

static int lfa_one(const orbit_ctx *o, const frame_t *f, const double *hp, const double *hc, int gen,
                   int order, int fd_order, const margins_t *mg, int64_t nb, int64_t ne, work_t *w)
{
    const int64_t N = o->d.n, wd = mg->w;
    const real dt = o->d.dt;
    /* ranges, innermost last: X on [nb,ne) <- dy on [d0,d1) <- y on [y0,y1) <- g on [g0,g1) */
    const int64_t d0 = imax(0, nb - mg->m2), d1 = imin(N, ne + (order + 1) / 2 + 1);
    const int64_t y0 = imax(0, d0 - wd), y1 = imin(N, d1 + wd);
    const int64_t g0 = imax(0, y0 - mg->m1), g1 = imin(N, y1 + mg->m1);
    real *gp = (real *)calloc((size_t)imax(g1 - g0, 1), sizeof(real));
    real *gc = (real *)calloc((size_t)imax(g1 - g0, 1), sizeof(real));
    real *dy[3] = { 0, 0, 0 };
    for (int l = 0; l < 3; ++l) dy[l] = (real *)calloc((size_t)imax(d1 - d0, 1), sizeof(real));
    if (!gp || !gc || !dy[0] || !dy[1] || !dy[2] || work_alloc(w, y0, y1 - y0, ne - nb)) return ORC_EINVAL;
    /* g = d h / dt by the central stencil on the grid */
#pragma omp parallel for
    for (int64_t i = g0; i < g1; ++i) {
        if (i < wd || i >= N - wd) continue;
        gp[i - g0] = fd1_in(hp, i, dt, fd_order);
        gc[i - g0] = fd1_in(hc, i, dt, fd_order);
    }
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t m = y0; m < y1; ++m) {
        if (m < mg->m1 + wd || m >= N - mg->m1 - wd) continue;
        real y[6];
        links_lfa_at(o, f, gp, gc, g0, g1 - g0, m, order, y);
        for (int l = 0; l < 6; ++l) w->y[l][m - y0] = y[l];
    }
    /* dy = first (gen 1.5) or second (gen 2.0) time derivative of y_l, l = +1,+2,+3 */
#pragma omp parallel for
    for (int64_t i = d0; i < d1; ++i) {
        if (i < mg->m1 + 2 * wd || i >= N - mg->m1 - 2 * wd) continue;
        for (int l = 0; l < 3; ++l)
            dy[l][i - d0] = (gen == ORC_GEN_15) ? fd1_r(w->y[l], i - y0, dt, fd_order)
                                                : fd2_r(w->y[l], i - y0, dt, fd_order);
    }
    yseries_t dys = { { dy[0], dy[1], dy[2], 0, 0, 0 }, d0, d1 - d0 };
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t n = nb; n < ne; ++n) {
        if (n < mg->lo || n >= N - mg->hi) continue;
        geom_t g;
        orbit_geometry(o, n, &g);
        for (int c = 0; c < 3; ++c)
            w->X[c][n - nb] = michelson_lfa_at(&dys, g.L, c, gen, n, dt, order);
    }
    free(gp); free(gc);
    for (int l = 0; l < 3; ++l) free(dy[l]);
    return ORC_OK;
}

static void emit(const work_t *w, int64_t nb, int64_t ne, int64_t b, int64_t batch, double *A, double *E,
                 double *T, double *XYZ, double *y)
{
    const int64_t len = ne - nb;
    for (int64_t i = 0; i < len; ++i) {
        real a, e, t;
        aet(w->X[0][i], w->X[1][i], w->X[2][i], &a, &e, &t);
        if (A) A[b * len + i] = (double)a;
        if (E) E[b * len + i] = (double)e;
        if (T) T[b * len + i] = (double)t;
        if (XYZ)
            for (int c = 0; c < 3; ++c) XYZ[(c * batch + b) * len + i] = (double)w->X[c][i];
        if (y)
            for (int l = 0; l < 6; ++l) {
                const int64_t m = nb + i - w->y0;
                y[(l * batch + b) * len + i] = (m >= 0 && m < w->ylen) ? (double)w->y[l][m] : 0.0;
            }
    }
}

static int check_args(const orc_orbit_desc *d, int gen, int order, int fd_order, int need_fd, int64_t ld,
                      int64_t nb, int64_t ne)
{
    if (!d || d->n <= 0 || d->dt <= 0) return ORC_EINVAL;
    if (gen != ORC_GEN_15 && gen != ORC_GEN_20) return ORC_EINVAL;
    if (order < 1 || order > 63 || order % 2 == 0) return ORC_EINVAL;
    if (need_fd && fd_order != 2 && fd_order != 4) return ORC_EINVAL;
    if (ld < d->n || nb < 0 || ne > d->n || nb > ne) return ORC_EINVAL;
    return ORC_OK;
}

/* ---- exported API ---------------------------------------------------------------- */

int orc_real_bits(void) { return (int)(sizeof(real) * 8); }
#ifdef _OPENMP
#include <omp.h>
int orc_num_threads(void) { return omp_get_max_threads(); }
#else
int orc_num_threads(void) { return 1; }
#endif
int orc_real_mant_dig(void)
{
#ifdef ORC_REAL_LD
    return __LDBL_MANT_DIG__;
#else
    return __DBL_MANT_DIG__;
#endif
}

int orc_margins(const orc_orbit_desc *d, int gen, int order, int fd_order, int64_t *lo, int64_t *hi)
{
    margins_t m;
    if (!d || !lo || !hi) return ORC_EINVAL;
    margins(d, gen, order, fd_order, &m);
    *lo = m.lo;
    *hi = m.hi;
    return ORC_OK;
}

/* margins of the link series y itself (valid on [ylo, n - yhi)) */
int orc_link_margins(const orc_orbit_desc *d, int order, int fd_order, int64_t *ylo, int64_t *yhi)
{
    margins_t m;
    if (!d || !ylo || !yhi) return ORC_EINVAL;
    margins(d, ORC_GEN_15, order, fd_order, &m);
    *ylo = m.m1 + m.w;
    *yhi = m.m1 + m.w;
    return ORC_OK;
}

/* Eq. (4.2): t_hyb = t_c - 5 (8 pi f_hyb)^(-8/3) (G Mc / c^3)^(-5/3) */
double orc_hyb_time(double f_hyb_hz, double mchirp_s, double t_c)
{
    return (double)((real)t_c - 5 * R_POW(8 * R_PI * (real)f_hyb_hz, -(real)8 / 3) *
                                    R_POW((real)mchirp_s, -(real)5 / 3));
}

/* Eq. (4.3) */
double orc_lfa_fraction(double f_hyb, double f_min, double f_max)
{
    const real e = -(real)8 / 3;
    return (double)((R_POW((real)f_min, e) - R_POW((real)f_hyb, e)) /
                    (R_POW((real)f_min, e) - R_POW((real)f_max, e)));
}

void orc_lagrange_weights(double eps, int order, double *w)
{
    real wr[64];
    lagrange_weights((real)eps, order, wr);
    for (int i = 0; i <= order; ++i) w[i] = (double)wr[i];
}

/* I[x](n, d): value of x at t_n - d (O4) */
double orc_interp(const double *x, int64_t len, int64_t n, double d, double dt, int order)
{
    return (double)interp_input(x, len, n, (real)d, (real)dt, order);
}

/* derivative stencils on a double series, which = 1 (FD1) or 2 (FD2); out[i] for i in [w, len-w) */
void orc_stencil(const double *x, int64_t len, double dt, int fd_order, int which, double *out)
{
    const int64_t w = fd_order / 2;
    real *xr = (real *)malloc(sizeof(real) * (size_t)len);
    for (int64_t i = 0; i < len; ++i) { xr[i] = x[i]; out[i] = 0; }
    for (int64_t i = w; i < len - w; ++i)
        out[i] = (double)(which == 1 ? fd1_r(xr, i, (real)dt, fd_order) : fd2_r(xr, i, (real)dt, fd_order));
    free(xr);
}

/* source frame: out = k[3], u[3], v[3], cos 2psi, sin 2psi */
void orc_source_frame(const orc_source *s, double *out)
{
    frame_t f;
    source_frame(s, &f);
    for (int a = 0; a < 3; ++a) { out[a] = (double)f.k[a]; out[3 + a] = (double)f.u[a]; out[6 + a] = (double)f.v[a]; }
    out[9] = (double)f.c2;
    out[10] = (double)f.s2;
}

/* orbit tables for samples [nb, ne): R [3][3][len], nhat [6][3][len], L [6][len] */
int orc_orbit_tables(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, int64_t nb,
                     int64_t ne, double *R, double *nhat, double *L)
{
    if (!d || nb < 0 || ne > d->n || nb > ne) return ORC_EINVAL;
    if (d->mode == ORC_ORBIT_TABLES && (!Rtab || !Ltab)) return ORC_EINVAL;
    orbit_ctx o = { *d, Rtab, Ltab };
    const int64_t len = ne - nb;
#pragma omp parallel for
    for (int64_t n = nb; n < ne; ++n) {
        geom_t g;
        orbit_geometry(&o, n, &g);
        for (int i = 0; i < 3; ++i)
            for (int a = 0; a < 3; ++a)
                if (R) R[(i * 3 + a) * len + (n - nb)] = (double)g.R[i][a];
        for (int l = 0; l < 6; ++l) {
            for (int a = 0; a < 3; ++a)
                if (nhat) nhat[(l * 3 + a) * len + (n - nb)] = (double)g.nh[l][a];
            if (L) L[l * len + (n - nb)] = (double)g.L[l];
        }
    }
    return ORC_OK;
}

/* the same link quantities split as hi + lo doubles (hi = the value rounded to double, lo = the remainder of the
 * working precision): lets the tests see the digits of n_l and L_l beyond fp64 that the CUDA orbit kernel stores
 * as low parts.  nhat_hi / nhat_lo [6][3][len], L_hi / L_lo [6][len]. */
int orc_orbit_tables_split(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, int64_t nb,
                           int64_t ne, double *nhat_hi, double *nhat_lo, double *L_hi, double *L_lo)
{
    if (!d || nb < 0 || ne > d->n || nb > ne || !nhat_hi || !nhat_lo || !L_hi || !L_lo) return ORC_EINVAL;
    if (d->mode == ORC_ORBIT_TABLES && (!Rtab || !Ltab)) return ORC_EINVAL;
    orbit_ctx o = { *d, Rtab, Ltab };
    const int64_t len = ne - nb;
#pragma omp parallel for
    for (int64_t n = nb; n < ne; ++n) {
        geom_t g;
        orbit_geometry(&o, n, &g);
        for (int l = 0; l < 6; ++l) {
            for (int a = 0; a < 3; ++a) {
                const double hi = (double)g.nh[l][a];
                nhat_hi[(l * 3 + a) * len + (n - nb)] = hi;
                nhat_lo[(l * 3 + a) * len + (n - nb)] = (double)(g.nh[l][a] - (real)hi);
            }
            const double hi = (double)g.L[l];
            L_hi[l * len + (n - nb)] = hi;
            L_lo[l * len + (n - nb)] = (double)(g.L[l] - (real)hi);
        }
    }
    return ORC_OK;
}

/* antenna patterns F^+_l, F^x_l and k.n_l of one source at sample n: out[6][3] */
int orc_antenna(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, const orc_source *s,
                int64_t n, double *out)
{
    orbit_ctx o = { *d, Rtab, Ltab };
    frame_t f;
    geom_t g;
    source_frame(s, &f);
    orbit_geometry(&o, n, &g);
    for (int l = 0; l < 6; ++l) {
        real Fp, Fc;
        antenna(&f, g.nh[l], &Fp, &Fc);
        out[l * 3 + 0] = (double)Fp;
        out[l * 3 + 1] = (double)Fc;
        out[l * 3 + 2] = (double)dot3(f.k, g.nh[l]);
    }
    return ORC_OK;
}

void orc_hybrid_weights(const orc_hybrid *h, const double *t, int64_t len, double *w_lfa, double *w_full)
{
    for (int64_t i = 0; i < len; ++i) {
        real a, b;
        hybrid_weights(h, (real)t[i], &a, &b);
        w_lfa[i] = (double)a;
        w_full[i] = (double)b;
    }
}

/* Michelson X, Y, Z of Eq. (2.7) / (2.8) from CALLER-SUPPLIED link series y [6][n] (link order +1,+2,+3,-1,-2,-3):
 * michelson_at() on every sample of the valid range [lo, n - hi) of margins(); XYZ [3][n], zero in the margins.
 * Lets a test plant sentinels in the margin samples of y and see that no valid output reads them (O10, G11). */
int orc_michelson_from_links(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, const double *y,
                             int gen, int order, double *XYZ)
{
    if (check_args(d, gen, order, 0, 0, d ? d->n : 0, 0, d ? d->n : 0) || !y || !XYZ) return ORC_EINVAL;
    orbit_ctx o = { *d, Rtab, Ltab };
    margins_t mg;
    margins(d, gen, order, 0, &mg);
    const int64_t N = d->n;
    real *yr[6];
    for (int l = 0; l < 6; ++l) {
        if (!(yr[l] = (real *)malloc(sizeof(real) * (size_t)N))) return ORC_EINVAL;
        for (int64_t i = 0; i < N; ++i) yr[l][i] = y[(int64_t)l * N + i];
    }
    yseries_t ys = { { yr[0], yr[1], yr[2], yr[3], yr[4], yr[5] }, 0, N };
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t n = 0; n < N; ++n) {
        for (int c = 0; c < 3; ++c) XYZ[(int64_t)c * N + n] = 0.0;
        if (n < mg.lo || n >= N - mg.hi) continue;
        geom_t g;
        orbit_geometry(&o, n, &g);
        for (int c = 0; c < 3; ++c)
            XYZ[(int64_t)c * N + n] = (double)michelson_at(&ys, g.L, c, gen, n, (real)d->dt, order);
    }
    for (int l = 0; l < 6; ++l) free(yr[l]);
    return ORC_OK;
}

/* alpha, beta, gamma of O15 from caller-supplied link series y [6][n]: sagnac_at() on the valid range of margins() (the
 * Michelson margins of the same generation: the Sagnac delays, 2 and 5 light times, are shorter than the Michelson ones) */
int orc_sagnac_from_links(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, const double *y,
                          int gen, int order, double *abc)
{
    if (check_args(d, gen, order, 0, 0, d ? d->n : 0, 0, d ? d->n : 0) || !y || !abc) return ORC_EINVAL;
    orbit_ctx o = { *d, Rtab, Ltab };
    margins_t mg;
    margins(d, gen, order, 0, &mg);
    const int64_t N = d->n;
    real *yr[6];
    for (int l = 0; l < 6; ++l) {
        if (!(yr[l] = (real *)malloc(sizeof(real) * (size_t)N))) return ORC_EINVAL;
        for (int64_t i = 0; i < N; ++i) yr[l][i] = y[(int64_t)l * N + i];
    }
    yseries_t ys = { { yr[0], yr[1], yr[2], yr[3], yr[4], yr[5] }, 0, N };
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t n = 0; n < N; ++n) {
        for (int c = 0; c < 3; ++c) abc[(int64_t)c * N + n] = 0.0;
        if (n < mg.lo || n >= N - mg.hi) continue;
        geom_t g;
        orbit_geometry(&o, n, &g);
        for (int c = 0; c < 3; ++c)
            abc[(int64_t)c * N + n] = (double)sagnac_at(&ys, g.L, c, gen, n, (real)d->dt, order);
    }
    for (int l = 0; l < 6; ++l) free(yr[l]);
    return ORC_OK;
}

/*
 * Full response (O5-O7).  hp, hc: [batch][ld]; outputs: A,E,T [batch][ne-nb],
 * XYZ [3][batch][ne-nb], y [6][batch][ne-nb]; any may be NULL.
 */
int orc_response_full(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, const double *hp,
                      const double *hc, int64_t ld, int64_t batch, const orc_source *src, int gen,
                      int order, int64_t nb, int64_t ne, double *A, double *E, double *T, double *XYZ,
                      double *y)
{
    if (check_args(d, gen, order, 0, 0, ld, nb, ne) || !hp || !hc || !src) return ORC_EINVAL;
    orbit_ctx o = { *d, Rtab, Ltab };
    margins_t mg;
    margins(d, gen, order, 0, &mg);
    for (int64_t b = 0; b < batch; ++b) {
        frame_t f;
        work_t w;
        source_frame(&src[b], &f);
        if (full_one(&o, &f, hp + b * ld, hc + b * ld, gen, order, &mg, mg.lo, mg.hi, nb, ne, &w)) return ORC_EINVAL;
        emit(&w, nb, ne, b, batch, A, E, T, XYZ, y);
        work_free(&w);
    }
    return ORC_OK;
}

/* LFA response (O8) */
/* Full response with the Sagnac combinations (O15): alpha, beta, gamma where orc_response_full has X, Y, Z, and Eq. (2.9)
 * applied to them for A, E, T */
int orc_response_full_sagnac(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, const double *hp,
                             const double *hc, int64_t ld, int64_t batch, const orc_source *src, int gen,
                             int order, int64_t nb, int64_t ne, double *A, double *E, double *T,
                             double *XYZ, double *y)
{
    g_sagnac = 1;
    const int rc = orc_response_full(d, Rtab, Ltab, hp, hc, ld, batch, src, gen, order, nb, ne, A, E, T, XYZ, y);
    g_sagnac = 0;
    return rc;
}

/* Full response with properly nested TDI delays (O12); nested_order = p_L, the Lagrange order of the light-time lookups */
int orc_response_full_nested(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, const double *hp,
                             const double *hc, int64_t ld, int64_t batch, const orc_source *src, int gen,
                             int order, int nested_order, int64_t nb, int64_t ne, double *A, double *E, double *T,
                             double *XYZ, double *y)
{
    if (nested_order < 1 || nested_order > 63 || nested_order % 2 == 0) return ORC_EINVAL;
    g_nested_order = nested_order;
    const int rc = orc_response_full(d, Rtab, Ltab, hp, hc, ld, batch, src, gen, order, nb, ne, A, E, T, XYZ, y);
    g_nested_order = 0;
    return rc;
}

/* X, Y, Z with nested delays from caller-supplied link series y [6][n] (for the pins: laser-noise cancellation) */
int orc_michelson_nested_from_links(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, const double *y,
                                    int gen, int order, int nested_order, double *XYZ)
{
    if (check_args(d, gen, order, 0, 0, d ? d->n : 0, 0, d ? d->n : 0) || !y || !XYZ) return ORC_EINVAL;
    if (nested_order < 1 || nested_order > 63 || nested_order % 2 == 0) return ORC_EINVAL;
    orbit_ctx o = { *d, Rtab, Ltab };
    margins_t mg;
    margins(d, gen, order, 0, &mg);
    const int64_t N = d->n;
    real *yr[6], *buf[6];
    lseries_t Ls;
    for (int l = 0; l < 6; ++l) {
        if (!(yr[l] = (real *)malloc(sizeof(real) * (size_t)N))) return ORC_EINVAL;
        for (int64_t i = 0; i < N; ++i) yr[l][i] = y[(int64_t)l * N + i];
    }
    if (lseries_alloc(&o, 0, N, buf, &Ls)) return ORC_EINVAL;
    yseries_t ys = { { yr[0], yr[1], yr[2], yr[3], yr[4], yr[5] }, 0, N };
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t n = 0; n < N; ++n) {
        for (int c = 0; c < 3; ++c) XYZ[(int64_t)c * N + n] = 0.0;
        if (n < mg.lo || n >= N - mg.hi) continue;
        for (int c = 0; c < 3; ++c)
            XYZ[(int64_t)c * N + n] = (double)michelson_nested_at(&ys, &Ls, c, gen, n, (real)d->dt, order, nested_order);
    }
    for (int l = 0; l < 6; ++l) { free(yr[l]); free(buf[l]); }
    return ORC_OK;
}

int orc_response_lfa(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, const double *hp,
                     const double *hc, int64_t ld, int64_t batch, const orc_source *src, int gen,
                     int order, int fd_order, int64_t nb, int64_t ne, double *A, double *E, double *T,
                     double *XYZ, double *y)
{
    if (check_args(d, gen, order, fd_order, 1, ld, nb, ne) || !hp || !hc || !src) return ORC_EINVAL;
    orbit_ctx o = { *d, Rtab, Ltab };
    margins_t mg;
    margins(d, gen, order, fd_order, &mg);
    for (int64_t b = 0; b < batch; ++b) {
        frame_t f;
        work_t w;
        source_frame(&src[b], &f);
        if (lfa_one(&o, &f, hp + b * ld, hc + b * ld, gen, order, fd_order, &mg, nb, ne, &w)) return ORC_EINVAL;
        emit(&w, nb, ne, b, batch, A, E, T, XYZ, y);
        work_free(&w);
    }
    return ORC_OK;
}

/* Extended LFA response: `terms` terms of the single-link series (B4) (1 | 2) about the expansion
 * point `point` (0 central (B1), 1 backward (B13), 2 forward (B14); terms = 2 only with the central point), then the
 * Michelson combination (B25) / (B33) as in orc_response_lfa.  The output margins grow by one sample per side when
 * terms = 2 (the third-derivative stencil is one sample wider): orc_margins_lfa_ext. */
int orc_margins_lfa_ext(const orc_orbit_desc *d, int gen, int order, int fd_order, int terms, int64_t *lo, int64_t *hi)
{
    margins_t m;
    if (!d || !lo || !hi) return ORC_EINVAL;
    margins(d, gen, order, fd_order, &m);
    *lo = m.lo + (terms >= 2 ? 1 : 0);
    *hi = m.hi + (terms >= 2 ? 1 : 0);
    return ORC_OK;
}

int orc_response_lfa_ext(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, const double *hp,
                         const double *hc, int64_t ld, int64_t batch, const orc_source *src, int gen,
                         int order, int fd_order, int terms, int point, int64_t nb, int64_t ne, double *A, double *E,
                         double *T, double *XYZ, double *y)
{
    if (check_args(d, gen, order, fd_order, 1, ld, nb, ne) || !hp || !hc || !src) return ORC_EINVAL;
    if (terms < 1 || terms > 2 || point < 0 || point > 2 || (terms == 2 && point != ORC_LFA_CENTRAL)) return ORC_EINVAL;
    orbit_ctx o = { *d, Rtab, Ltab };
    margins_t mg;
    margins(d, gen, order, fd_order, &mg);
    for (int64_t b = 0; b < batch; ++b) {
        frame_t f;
        work_t w;
        source_frame(&src[b], &f);
        if (lfa_one_ext(&o, &f, hp + b * ld, hc + b * ld, gen, order, fd_order, terms, point, &mg, nb, ne, &w)) return ORC_EINVAL;
        emit(&w, nb, ne, b, batch, A, E, T, XYZ, y);
        work_free(&w);
    }
    return ORC_OK;
}

/* O14: six LFA links and the Michelson variables of Eq. (B20) / (B30); margins grow by one sample for gen 2.0 */
int orc_margins_lfa6(const orc_orbit_desc *d, int gen, int order, int fd_order, int64_t *lo, int64_t *hi)
{
    margins_t m;
    if (!d || !lo || !hi) return ORC_EINVAL;
    margins(d, gen, order, fd_order, &m);
    *lo = m.lo + (gen == ORC_GEN_20 ? 1 : 0);
    *hi = m.hi + (gen == ORC_GEN_20 ? 1 : 0);
    return ORC_OK;
}

int orc_response_lfa6(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, const double *hp, const double *hc,
                      int64_t ld, int64_t batch, const orc_source *src, int gen, int order, int fd_order, int64_t nb,
                      int64_t ne, double *A, double *E, double *T, double *XYZ, double *y)
{
    if (check_args(d, gen, order, fd_order, 1, ld, nb, ne) || !hp || !hc || !src) return ORC_EINVAL;
    orbit_ctx o = { *d, Rtab, Ltab };
    margins_t mg;
    margins(d, gen, order, fd_order, &mg);
    for (int64_t b = 0; b < batch; ++b) {
        frame_t f;
        work_t w;
        source_frame(&src[b], &f);
        if (lfa6_one(&o, &f, hp + b * ld, hc + b * ld, gen, order, fd_order, &mg, nb, ne, &w)) return ORC_EINVAL;
        emit(&w, nb, ne, b, batch, A, E, T, XYZ, y);
        work_free(&w);
    }
    return ORC_OK;
}

/* X, Y, Z of Eq. (B20) / (B30) from caller-supplied link series y [6][n] (for the pins): the derivatives by the stencils
 * of order fd_order, valid where they fit */
int orc_michelson_b20_from_links(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, const double *y, int gen,
                                 int order, int fd_order, double *XYZ)
{
    if (check_args(d, gen, order, fd_order, 1, d ? d->n : 0, 0, d ? d->n : 0) || !y || !XYZ) return ORC_EINVAL;
    orbit_ctx o = { *d, Rtab, Ltab };
    margins_t mg;
    margins(d, gen, order, fd_order, &mg);
    const int64_t N = d->n, wy = fd_order / 2 + 1;
    real *yr = (real *)malloc(sizeof(real) * (size_t)N), *lo[6], *hi[6];
    if (!yr) return ORC_EINVAL;
    for (int l = 0; l < 6; ++l) {
        lo[l] = (real *)calloc((size_t)N, sizeof(real));
        hi[l] = (real *)calloc((size_t)N, sizeof(real));
        if (!lo[l] || !hi[l]) return ORC_EINVAL;
        for (int64_t i = 0; i < N; ++i) yr[i] = y[(int64_t)l * N + i];
        for (int64_t i = wy; i < N - wy; ++i) {
            lo[l][i] = gen == ORC_GEN_15 ? fd1_r(yr, i, (real)d->dt, fd_order) : fd2_r(yr, i, (real)d->dt, fd_order);
            hi[l][i] = gen == ORC_GEN_15 ? fd2_r(yr, i, (real)d->dt, fd_order) : fd3_r(yr, i, (real)d->dt, fd_order);
        }
    }
    yseries_t slo = { { lo[0], lo[1], lo[2], lo[3], lo[4], lo[5] }, 0, N }, shi = { { hi[0], hi[1], hi[2], hi[3], hi[4], hi[5] }, 0, N };
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t n = 0; n < N; ++n) {
        for (int c = 0; c < 3; ++c) XYZ[(int64_t)c * N + n] = 0.0;
        if (n < mg.lo + 1 || n >= N - mg.hi - 1) continue;
        geom_t g;
        orbit_geometry(&o, n, &g);
        for (int c = 0; c < 3; ++c)
            XYZ[(int64_t)c * N + n] = (double)michelson_b20_at(&slo, &shi, g.L, c, gen, n, (real)d->dt, order);
    }
    free(yr);
    for (int l = 0; l < 6; ++l) { free(lo[l]); free(hi[l]); }
    return ORC_OK;
}

/* third-derivative stencil on a double series (for the pins): out[i] for i in [w, len - w), w = fd_order / 2 + 1 */
void orc_stencil3(const double *x, int64_t len, double dt, int fd_order, double *out)
{
    const int64_t w = fd_order / 2 + 1;
    for (int64_t i = 0; i < len; ++i) out[i] = 0;
    for (int64_t i = w; i < len - w; ++i) out[i] = (double)fd3_in(x, i, (real)dt, fd_order);
}

/* ---------------------------------------------------------------------------------- */
/* O13  on-device waveform generation fused with the projection (SURVEY 8(f)-3,        */
/*      step i of P:408): the leading-order chirp of Eq. (4.2)'s order joined to a      */
/*      damped-sinusoid ringdown -- the input recipe of configs 1-4 (DESIGN.md          */
/*      section 4) taken as a waveform MODEL with parameters, so that the strain can    */
/*      be evaluated at any time instead of being read from a sampled series.           */
/* ---------------------------------------------------------------------------------- */
/* tau = t_c - t, tau_in = max(tau, tau_cut), u = tau_in / (5 Mc):
 *   f     = (1 / pi) (5 / (256 tau_in))^(3/8) Mc^(-5/8)          (inverse of Eq. (4.2))
 *   amp   = 4 (Mc c / d_L) (pi f Mc)^(2/3) = 4 (Mc c / d_L) (5 Mc / (256 tau_in))^(1/4)
 *   Phi   = phi_c - 2 u^(5/8)
 * after the join (x = tau_cut - tau > 0): amp *= exp(-x / tau_rd),
 *   Phi  += 2 pi [ f_rd x - (f_rd - f_cut) tau_rd (1 - exp(-x / tau_rd)) ],   f_cut = f(tau_cut)
 * h+ = amp (1 + cos^2 iota) / 2 cos Phi,   hx = amp cos iota sin Phi.   Mc = G M_c / c^3 in seconds. */
typedef struct { double t_c, mc_s, dist_m, cos_iota, phi_c, tau_cut, f_rd, tau_rd; } orc_chirp;

static void chirp_at(const orc_chirp *w, real t, real *hp, real *hc)
{
    const real mc = w->mc_s, tau_cut = w->tau_cut;
    const real tau = (real)w->t_c - t;
    const real tau_in = tau > tau_cut ? tau : tau_cut;
    const real f_cut = (1 / R_PI) * R_POW(5 / (256 * tau_cut), (real)0.375) * R_POW(mc, (real)-0.625);
    const real f = (1 / R_PI) * R_POW(5 / (256 * tau_in), (real)0.375) * R_POW(mc, (real)-0.625);
    real amp = 4 * (mc * (real)ORC_C_LIGHT / (real)w->dist_m) * R_POW(R_PI * f * mc, (real)2 / 3);
    real phase = (real)w->phi_c - 2 * R_POW(tau_in / (5 * mc), (real)0.625);
    const real x = tau_cut - tau;
    if (x > 0) {
        const real decay = R_EXP(-x / (real)w->tau_rd);
        amp *= decay;
        phase += 2 * R_PI * ((real)w->f_rd * x - ((real)w->f_rd - f_cut) * (real)w->tau_rd * (1 - decay));
    }
    const real ci = w->cos_iota;
    *hp = amp * (real)0.5 * (1 + ci * ci) * R_COS(phase);
    *hc = amp * ci * R_SIN(phase);
}

/* the model sampled on the grid t_n = t0 + n dt, rounded to double: hp, hc [batch][ld] */
int orc_waveform_chirp(const orc_chirp *w, int64_t batch, double t0, double dt, int64_t n, int64_t ld, double *hp,
                       double *hc)
{
    if (!w || !hp || !hc || batch < 1 || n < 1 || ld < n || !(dt > 0)) return ORC_EINVAL;
    for (int64_t b = 0; b < batch; ++b) {
        if (!(w[b].mc_s > 0) || !(w[b].dist_m > 0) || !(w[b].tau_cut > 0) || !(w[b].tau_rd > 0)) return ORC_EINVAL;
#pragma omp parallel for
        for (int64_t i = 0; i < n; ++i) {
            real a, c;
            chirp_at(&w[b], (real)t0 + (real)i * (real)dt, &a, &c);
            hp[b * ld + i] = (double)a;
            hc[b * ld + i] = (double)c;
        }
    }
    return ORC_OK;
}

/* O13b: the harmonic-sum waveform of an eccentric inspiral (the input recipe of config 5, as a MODEL):
 * the orbital evolution table F, e, l and their time derivatives at nk knots (tab [7][nk]: t, F, e, l, dF/dt, de/dt,
 * dl/dt) is carried to time t by cubic Hermite interpolation on the knot interval that contains t, then
 *   h+ = sum_n [ -(1 + cos^2 iota)(a_n cos 2 gamma - b_n sin 2 gamma) + (1 - cos^2 iota) c_n ]
 *   hx = sum_n 2 cos iota (b_n cos 2 gamma + a_n sin 2 gamma),                                  n = 1 .. nharm
 *   a_n = -n A [J_{n-2} - 2 e J_{n-1} + (2 / n) J_n + 2 e J_{n+1} - J_{n+2}](n e) cos(n l)
 *   b_n = -n A sqrt(1 - e^2) [J_{n-2} - 2 J_n + J_{n+2}](n e) sin(n l),     c_n = 2 A J_n(n e) cos(n l)
 *   A = (2 pi F M)^(2/3) eta M c / d_L          (Peters & Mathews 1963 in the form of Barack & Cutler 2004, Eqs. 7-9)
 * par [6] = M [s], eta, d_L [m], cos iota, gamma, l0. */
static real hermite_at(const double *tk, const double *yk, const double *dyk, int64_t idx, real t)
{
    const real h = (real)tk[idx + 1] - (real)tk[idx];
    const real u = (t - (real)tk[idx]) / h;
    const real h00 = (1 + 2 * u) * (1 - u) * (1 - u), h10 = u * (1 - u) * (1 - u);
    const real h01 = u * u * (3 - 2 * u), h11 = u * u * (u - 1);
    return h00 * (real)yk[idx] + h10 * h * (real)dyk[idx] + h01 * (real)yk[idx + 1] + h11 * h * (real)dyk[idx + 1];
}

static void ecc_at(const double *tab, int64_t nk, const double *par, int nharm, real t, real *hp, real *hc)
{
    const double *tk = tab;
    int64_t lo = 0, hi = nk;                      /* upper bound: first knot > t */
    while (lo < hi) {
        const int64_t mid = (lo + hi) / 2;
        if ((real)tk[mid] <= t) lo = mid + 1; else hi = mid;
    }
    int64_t idx = lo - 1;
    if (idx < 0) idx = 0;
    if (idx > nk - 2) idx = nk - 2;
    const real F = hermite_at(tk, tab + nk, tab + 4 * nk, idx, t);
    const real e = hermite_at(tk, tab + 2 * nk, tab + 5 * nk, idx, t);
    const real ell = hermite_at(tk, tab + 3 * nk, tab + 6 * nk, idx, t) + (real)par[5];
    const real M = par[0], eta = par[1], ci = par[3], gam = par[4];
    const real A = R_POW(2 * R_PI * F * M, (real)2 / 3) * eta * M * (real)ORC_C_LIGHT / (real)par[2];
    const real c2g = R_COS(2 * gam), s2g = R_SIN(2 * gam), ci2 = ci * ci, sq = R_SQRT(1 - e * e);
    real sp = 0, sc = 0;
    for (int n = 1; n <= nharm; ++n) {
        const real x = n * e, cn = R_COS(n * ell), sn = R_SIN(n * ell);
        const real jm2 = R_JN(n - 2, x), jm1 = R_JN(n - 1, x), j0 = R_JN(n, x), jp1 = R_JN(n + 1, x), jp2 = R_JN(n + 2, x);
        const real an = -n * A * (jm2 - 2 * e * jm1 + ((real)2 / n) * j0 + 2 * e * jp1 - jp2) * cn;
        const real bn = -n * A * sq * (jm2 - 2 * j0 + jp2) * sn;
        const real cc = 2 * A * j0 * cn;
        sp += -(1 + ci2) * (an * c2g - bn * s2g) + (1 - ci2) * cc;
        sc += 2 * ci * (bn * c2g + an * s2g);
    }
    *hp = sp;
    *hc = sc;
}

/* the model sampled on t0 + i dt: tab [batch][7][nk], par [batch][6]; hp, hc [batch][ld] */
int orc_waveform_ecc(const double *tab, int64_t nk, const double *par, int nharm, int64_t batch, double t0, double dt,
                     int64_t n, int64_t ld, double *hp, double *hc)
{
    if (!tab || !par || !hp || !hc || nk < 2 || nharm < 1 || batch < 1 || n < 1 || ld < n || !(dt > 0)) return ORC_EINVAL;
    for (int64_t b = 0; b < batch; ++b) {
#pragma omp parallel for
        for (int64_t i = 0; i < n; ++i) {
            real a, c;
            ecc_at(tab + b * 7 * nk, nk, par + 6 * b, nharm, (real)t0 + (real)i * (real)dt, &a, &c);
            hp[b * ld + i] = (double)a;
            hc[b * ld + i] = (double)c;
        }
    }
    return ORC_OK;
}

/* Eq. (2.5) with the strain of the model evaluated AT the retarded times (no sampled series, no interpolation) */
static void links_full_chirp_at(const orbit_ctx *o, const frame_t *f, const orc_chirp *w, int64_t n, real y[6])
{
    const real c = ORC_C_LIGHT;
    const real t = (real)o->d.t0 + (real)n * (real)o->d.dt;
    geom_t g;
    orbit_geometry(o, n, &g);
    for (int l = 0; l < 6; ++l) {
        const int s = LINK_S[l], r = LINK_R[l];
        real Fp, Fc, hps, hcs, hpr, hcr;
        antenna(f, g.nh[l], &Fp, &Fc);
        const real kn = dot3(f->k, g.nh[l]);
        const real delta_s = g.L[l] + dot3(f->k, g.R[s]) / c; /* (2.6a) */
        const real delta_r = dot3(f->k, g.R[r]) / c;          /* (2.6b) */
        chirp_at(w, t - delta_s, &hps, &hcs);
        chirp_at(w, t - delta_r, &hpr, &hcr);
        y[l] = ((Fp * hps + Fc * hcs) - (Fp * hpr + Fc * hcr)) / (2 * (1 - kn)); /* (2.5) */
    }
}

/* Full response from waveform parameters: links by links_full_chirp_at on the same ranges as full_one (the link series
 * is still zero inside its margins, G11, so that it is the series the sampled path produces up to the interpolation
 * error), then O6 / O7 unchanged. */
int orc_response_full_chirp(const orc_orbit_desc *d, const double *Rtab, const double *Ltab, const orc_chirp *wav,
                            int64_t batch, const orc_source *src, int gen, int order, int64_t nb, int64_t ne, double *A,
                            double *E, double *T, double *XYZ, double *y)
{
    if (check_args(d, gen, order, 0, 0, d ? d->n : 0, nb, ne) || !wav || !src) return ORC_EINVAL;
    orbit_ctx o = { *d, Rtab, Ltab };
    margins_t mg;
    margins(d, gen, order, 0, &mg);
    const int64_t N = d->n;
    for (int64_t b = 0; b < batch; ++b) {
        frame_t f;
        work_t w;
        source_frame(&src[b], &f);
        const int64_t y0 = imax(0, nb - mg.m2), y1 = imin(N, ne + (order + 1) / 2 + 1);
        if (work_alloc(&w, y0, y1 - y0, ne - nb)) return ORC_EINVAL;
#pragma omp parallel for schedule(dynamic, 64)
        for (int64_t m = y0; m < y1; ++m) {
            if (m < mg.m1 || m >= N - mg.m1) continue;
            real yy[6];
            links_full_chirp_at(&o, &f, &wav[b], m, yy);
            for (int l = 0; l < 6; ++l) w.y[l][m - y0] = yy[l];
        }
        yseries_t ys = { { w.y[0], w.y[1], w.y[2], w.y[3], w.y[4], w.y[5] }, y0, y1 - y0 };
#pragma omp parallel for schedule(dynamic, 64)
        for (int64_t n = nb; n < ne; ++n) {
            if (n < mg.lo || n >= N - mg.hi) continue;
            geom_t g;
            orbit_geometry(&o, n, &g);
            for (int c = 0; c < 3; ++c) w.X[c][n - nb] = michelson_at(&ys, g.L, c, gen, n, (real)d->dt, order);
        }
        emit(&w, nb, ne, b, batch, A, E, T, XYZ, y);
        work_free(&w);
    }
    return ORC_OK;
}

/* Hybrid response (O9): both responses on the whole requested range, blended per Eqs. (4.5), (4.6);
 * hyb has n_hyb = 1 or batch entries. */
int orc_response_hybrid(const orc_orbit_desc *d, const double *Rtab, const double *Ltab,
                        const double *hp, const double *hc, int64_t ld, int64_t batch,
                        const orc_source *src, int gen, int order, int fd_order, const orc_hybrid *hyb,
                        int64_t n_hyb, int64_t nb, int64_t ne, double *A, double *E, double *T,
                        double *XYZ, double *y)
{
    if (check_args(d, gen, order, fd_order, 1, ld, nb, ne) || !hp || !hc || !src || !hyb) return ORC_EINVAL;
    if (n_hyb != 1 && n_hyb != batch) return ORC_EINVAL;
    orbit_ctx o = { *d, Rtab, Ltab };
    margins_t mg, mf;
    margins(d, gen, order, fd_order, &mg); /* hybrid margins = the (wider) LFA ones */
    margins(d, gen, order, 0, &mf);
    const int64_t N = d->n;
    for (int64_t b = 0; b < batch; ++b) {
        const orc_hybrid *h = &hyb[n_hyb == 1 ? 0 : b];
        frame_t f;
        work_t wl, wf, wh;
        source_frame(&src[b], &f);
        if (lfa_one(&o, &f, hp + b * ld, hc + b * ld, gen, order, fd_order, &mg, nb, ne, &wl)) return ORC_EINVAL;
        if (full_one(&o, &f, hp + b * ld, hc + b * ld, gen, order, &mf, mg.lo, mg.hi, nb, ne, &wf)) return ORC_EINVAL;
        if (work_alloc(&wh, nb, ne - nb, ne - nb)) return ORC_EINVAL;
        for (int64_t n = nb; n < ne; ++n) {
            real wa, wb;
            hybrid_weights(h, (real)d->t0 + (real)n * (real)d->dt, &wa, &wb);
            /* (4.5): links, valid where both link series are (the LFA link margins) */
            if (n >= mg.m1 + mg.w && n < N - mg.m1 - mg.w)
                for (int l = 0; l < 6; ++l)
                    wh.y[l][n - nb] = wa * wl.y[l][n - wl.y0] + wb * wf.y[l][n - wf.y0];
            /* (4.6): Michelson observables blended separately (G19) */
            for (int c = 0; c < 3; ++c) wh.X[c][n - nb] = wa * wl.X[c][n - nb] + wb * wf.X[c][n - nb];
        }
        emit(&wh, nb, ne, b, batch, A, E, T, XYZ, y);
        work_free(&wl); work_free(&wf); work_free(&wh);
    }
    return ORC_OK;
}
