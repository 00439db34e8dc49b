/*
 * lisatdi.h -- C ABI of the B200 (sm_100a) time-domain LISA response library.
 *
 * The operations are those of arXiv 2505.09600 (Valencia & Husa); "P:n" is line n of
 * PAPER.md, "G<k>" a reading listed in DESIGN.md.  Everything is fp64.
 *
 *   full response   P:85-161   Eqs. (2.2)-(2.9): projection of h+, hx onto the six links at
 *                               retarded times, Michelson TDI 1.5 / 2.0, A, E, T
 *   LFA             P:210-260, P:677-957  Eqs. (3.1), (B1), (B10), (B25), (B33)
 *   hybrid          P:263-315  Eqs. (4.1), (4.2), (4.5), (4.6)
 *
 * Conventions
 *   - Pointers named d_* are DEVICE memory, h_* are HOST memory; both are owned by the
 *     caller.  The library allocates no device memory and keeps no pointer after a call
 *     returns, except that an ltdi_orbits handle refers to the caller's table buffer.
 *   - Every call is asynchronous on `stream` (a cudaStream_t passed as void*, NULL = the
 *     legacy default stream); the small h_* parameter arrays are consumed before the call
 *     returns.  ltdi_response_hybrid forks part of its work onto one internal non-blocking
 *     stream and joins it back with events before it returns control of `stream`'s order:
 *     to the caller the call is ordered on `stream` like the others.
 *   - Return value: LTDI_OK or a negative LTDI_E* code.  Nothing throws or aborts.
 *   - Time grid: t_n = t0 + n dt, n = 0 .. n-1, shared by all sources of a batch.
 *   - Series layout: a series of source b starts at element b * ld (ld >= n).
 *   - Links are ordered l = +1, +2, +3, -1, -2, -3 (+1: 3->2, +2: 1->3, +3: 2->1,
 *     -1: 2->3, -2: 3->1, -3: 1->2), spacecraft 1, 2, 3.
 *   - Fractional delays use centred Lagrange interpolation of odd order p (p + 1 taps, G10).
 *   - Output samples n < lo or n >= n - hi (ltdi_margins) are written as exactly 0.0 (G11).
 */
#ifndef LISATDI_H
#define LISATDI_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { LTDI_OK = 0, LTDI_EINVAL = -1, LTDI_EUNSUPPORTED = -2, LTDI_ECUDA = -3, LTDI_EWORKSPACE = -4 };
enum { LTDI_GEN_15 = 15, LTDI_GEN_20 = 20 };                 /* Eq. (2.7) / Eq. (2.8) */
enum {
    LTDI_ORBIT_STATIC_EQUALARM = 0, /* Keplerian positions, L_l(t) = arm_m / c constant ("equal and constant") */
    LTDI_ORBIT_KEPLERIAN = 1,       /* Keplerian positions, first-order light times, L_l != L_-l (G6)         */
    LTDI_ORBIT_TABLES = 2,          /* caller-supplied positions and light times per sample                           */
    LTDI_ORBIT_KNOTS = 3            /* a numerical orbit file: positions tabulated at knots (ltdi_orbits_init_knots)    */
};
enum { LTDI_TAPER_SIGMOID = 0,      /* Eq. (4.1), the paper's weight                                  */
       LTDI_TAPER_COSINE = 1 };     /* raised cosine over the window (BASELINE.json configs 2, 4; G20) */
enum { LTDI_RESPONSE_FULL = 0, LTDI_RESPONSE_LFA = 1, LTDI_RESPONSE_HYBRID = 2 };
enum { LTDI_LFA_CENTRAL = 0,        /* expansion about tau of Eq. (B1), P:685 (the paper's choice)                 */
       LTDI_LFA_BACKWARD = 1,       /* epsilon = 0: about t - L_l - k.R_s / c, Eq. (B13)                    */
       LTDI_LFA_FORWARD = 2 };      /* epsilon = 1: about t - k.R_r / c, Eq. (B14), P:778 (the choice of Ref. [46]) */

/* Time grid and orbit model (first-order Keplerian orbits, G5). */
typedef struct {
    double t0, dt;   /* t_n = t0 + n dt [s], dt > 0 */
    int64_t n;       /* samples, > 0 */
    double arm_m;    /* nominal arm length L [m] (2.5e9) */
    double R_m;      /* orbital radius [m] (1 AU) */
    double period_s; /* orbital period [s] (Omega = 2 pi / period) */
    double alpha0;   /* orbital phase at t = 0 [rad] */
    double rot0;     /* constellation rotation phase [rad] */
    int32_t mode;    /* LTDI_ORBIT_* */
} ltdi_orbit_desc;

typedef struct { double beta, lambda, psi; } ltdi_source; /* ecliptic latitude, longitude, polarisation [rad] */

/* Hybridisation window: centre t_hyb [s], width window_s (T), sigmoid scale sigma_s. */
typedef struct { double t_hyb, window_s, sigma_s; int32_t taper; } ltdi_hybrid;

typedef struct ltdi_orbits ltdi_orbits; /* opaque; changed only by ltdi_orbits_prepare() after init */

/* Rows of the device orbit table: 9 positions R_i [m] (i*3+axis), 9 unit vectors n_l for
 * l = +1,+2,+3 (n_-l = -n_l), 6 light travel times L_l [s]; row stride = ltdi_orbits_stride(). */
#define LTDI_TABLE_ROWS 24

/* ---- S0: orbit / delay tables (Eq. (B22)) -------------------------------- */

/* Bytes of the device buffer that ltdi_orbits_init* fills for this grid. */
int ltdi_orbits_workspace_bytes(const ltdi_orbit_desc *desc, size_t *bytes);

/* Launch the orbit/delay kernel: spacecraft positions, link unit vectors and light travel
 * times per sample into d_tables (>= workspace bytes, 16-byte aligned).  mode must be
 * STATIC_EQUALARM or KEPLERIAN.  *out receives a host handle (free with ltdi_orbits_destroy). */
int ltdi_orbits_init(const ltdi_orbit_desc *desc, void *d_tables, size_t bytes, void *stream,
                     ltdi_orbits **out);

/* Same from caller-supplied device tables: d_R [3][3][n] positions [m], d_L [6][n] light travel
 * times [s]; the unit vectors are derived (n_l = (R_r - R_s) / |R_r - R_s|).  desc->mode
 * must be LTDI_ORBIT_TABLES; arm_m and R_m still size the margins. */
int ltdi_orbits_init_tables(const ltdi_orbit_desc *desc, const double *d_R, const double *d_L,
                            void *d_tables, size_t bytes, void *stream, ltdi_orbits **out);

/* SURVEY.md 8(f)-4, numerical orbits ("realistic ESA orbits"; reading G28): d_knots [3][3][nk] (device; spacecraft,
 * component, knot) holds the spacecraft positions [m] at the times knot_t0 + j knot_dt.  They are brought to every
 * sample time by centred Lagrange interpolation of odd order knot_order <= 15 on the knot grid (taps
 * k = -(M/2-1) .. M/2 around the knot at or before t, M = knot_order + 1), the velocities are the time derivative of
 * that interpolant, n_l = (R_r - R_s) / |R_r - R_s| and L_l = (|R_r - R_s| / c)(1 + n_l . V_s / c) as for the Keplerian
 * mode (G6).  desc->mode must be LTDI_ORBIT_KNOTS; arm_m and R_m size the margins.  The knots must cover the grid:
 * knot_t0 + (M/2 - 1) knot_dt <= t0 and t0 + (n - 1) dt <= knot_t0 + (nk - 1 - M/2) knot_dt, else LTDI_EINVAL.
 * d_knots is read by the kernel only (stream-ordered); the handle keeps no reference to it. */
int ltdi_orbits_init_knots(const ltdi_orbit_desc *desc, const double *d_knots, int64_t nk, double knot_t0,
                           double knot_dt, int knot_order, void *d_tables, size_t bytes, void *stream,
                           ltdi_orbits **out);

/* Optional: the TDI delays of Eqs. (2.7) / (2.8) and (B25) / (B33) are sums of L_l(t_n), so the
 * Lagrange weights of the TDI stage depend on the orbit object, the generation and the order only, not on
 * the sources.  ltdi_orbits_prepare() computes them once into d_buf (device, 16-byte aligned, >=
 * ltdi_orbits_prepare_bytes() bytes, owned by the caller, referenced by the handle until the next prepare or
 * destroy); responses called with the same gen and lagrange_order then skip their own weight kernel.  The
 * results are bitwise the same with or without it.  Orders other than 9 and 31 need 0 bytes (no-op). */
int ltdi_orbits_prepare_bytes(const ltdi_orbit_desc *desc, int lagrange_order, size_t *bytes);
int ltdi_orbits_prepare(ltdi_orbits *orb, int gen, int lagrange_order, void *d_buf, size_t bytes, void *stream);

int ltdi_orbits_destroy(ltdi_orbits *orb);               /* frees the handle only */
int64_t ltdi_orbits_stride(const ltdi_orbits *orb);      /* elements between table rows */
const double *ltdi_orbits_tables(const ltdi_orbits *orb); /* the caller's d_tables */

/* ---- helpers ------------------------------------------------------------------------------ */

/* Output margins (G11): response samples n < *lo and n >= n - *hi are 0.  fd_order = 0 for the
 * full response, 2 or 4 for LFA / hybrid. */
int ltdi_margins(const ltdi_orbit_desc *desc, int gen, int lagrange_order, int fd_order, int64_t *lo,
                 int64_t *hi);
/* Margins of the link series y_slr themselves. */
int ltdi_link_margins(const ltdi_orbit_desc *desc, int lagrange_order, int fd_order, int64_t *lo,
                      int64_t *hi);
/* Eq. (4.2): t_hyb = t_c - 5 (8 pi f_hyb)^(-8/3) (G Mc / c^3)^(-5/3); mchirp_s = G Mc / c^3 [s]. */
int ltdi_hyb_time(double f_hyb_hz, double mchirp_s, double t_c, double *t_hyb);

/* Bytes of d_work needed by ltdi_response_* (which = LTDI_RESPONSE_*). */
int ltdi_workspace_bytes(int which, int64_t n, int64_t batch, int gen, int lagrange_order, size_t *bytes);

/* ---- S1-S8: the three responses ------------------------------------------------------------- */
/*
 * Common arguments
 *   orb             orbit tables for the time grid (n samples)
 *   d_hp, d_hc      h+, hx sampled on the grid, [batch][ld], source frame
 *   h_src           [batch] sky position and polarisation
 *   gen             LTDI_GEN_15 or LTDI_GEN_20
 *   lagrange_order  odd, 1 .. 63
 *   d_A, d_E, d_T   [batch][ld] outputs, Eq. (2.9); required
 *   d_XYZ           [3][batch][ld] Michelson X, Y, Z, or NULL
 *   d_y             [6][batch][ld] single-link responses y_slr, or NULL
 *   d_work          scratch of ltdi_workspace_bytes() bytes, 16-byte aligned
 * Errors: LTDI_EINVAL for NULL required pointers, bad gen / order / fd_order, ld < n, batch < 1;
 * LTDI_EWORKSPACE if work_bytes is too small; LTDI_ECUDA if a CUDA call fails (set LTDI_DEBUG in the
 * environment to have the CUDA error printed); LTDI_EUNSUPPORTED if the link series one tile needs do not fit
 * the 227 KB of shared memory (sampling steps far below the light travel time: dt < L / (c 250) for the hybrid,
 * TDI 2.0) or batch x tiles exceeds 2^31.
 */

/* Full response: Eqs. (2.2)-(2.6) projection (S2, S3), Eq. (2.7)/(2.8) TDI (S4), Eq. (2.9) (S5). */
int ltdi_response_full(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld,
                       int64_t batch, const ltdi_source *h_src, int gen, int lagrange_order, double *d_A,
                       double *d_E, double *d_T, double *d_XYZ, double *d_y, void *d_work,
                       size_t work_bytes, void *stream);

/* SURVEY.md 8(f)-4, properly nested delays (the comparison case of P:151; the paper itself evaluates every L_l at t).
 * Delay operators act as (D_l f)(t) = f(t - L_l(t)); with a = D_-2 D_2, b = D_3 D_-3 (for X; cyclic for Y, Z),
 *   X_1.5 = (1 - b)(y_3-21 + D_-2 y_123) - (1 - a)(y_231 + D_3 y_1-32)
 *   X_2.0 = (1 - b - b a + a b b)(y_3-21 + D_-2 y_123) - (1 - a - a b + b a a)(y_231 + D_3 y_1-32),
 * i.e. Eqs. (2.7) / (2.8) term by term, but the delay of every term is accumulated along its chain of links,
 * d_j = d_{j-1} + L_cj(t - d_{j-1}), the light travel time at an off-grid time being the centred Lagrange interpolation
 * of order nested_order of the sampled L_l(t_n) (reading G29).  nested_order must be 3; Lagrange orders 9 and 31 only
 * (LTDI_EUNSUPPORTED otherwise).  Everything else as ltdi_response_full. */
int ltdi_response_full_nested(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld,
                              int64_t batch, const ltdi_source *h_src, int gen, int lagrange_order, int nested_order,
                              double *d_A, double *d_E, double *d_T, double *d_XYZ, double *d_y, void *d_work,
                              size_t work_bytes, void *stream);

/* waveform generation on the device, fused with the projection (step i of P:408).
 * The chirp + ringdown MODEL (the recipe of BASELINE.json configs 1-4; leading-order chirp of the order of Eq. (4.2),
 * P:283): with tau = t_c - t, Mc = G M_c / c^3 [s],
 *   tau > tau_cut:  Phi = phi_c - 2 (tau / 5 Mc)^(5/8),  amp = 4 (Mc c / d_L)(5 Mc / (256 tau))^(1/4)
 *   x = tau_cut - tau >= 0:  Phi = Phi(tau_cut) + 2 pi [f_rd x - (f_rd - f_cut) tau_rd (1 - exp(-x / tau_rd))],
 *                            amp = amp(tau_cut) exp(-x / tau_rd),   f_cut = (1 / pi)(5 / (256 tau_cut))^(3/8) Mc^(-5/8)
 *   h+ = amp (1 + cos^2 iota) / 2 cos Phi,   hx = amp cos iota sin Phi.
 * A source without ringdown takes a tiny tau_cut (the join then lies outside the segment). */
typedef struct {
    double t_c;      /* coalescence time [s] (same clock as the time grid) */
    double mc_s;     /* chirp mass G M_c / c^3 [s] */
    double dist_m;   /* luminosity distance [m] */
    double cos_iota; /* cosine of the inclination */
    double phi_c;    /* phase at coalescence [rad] */
    double tau_cut;  /* the ringdown joins tau_cut seconds before t_c, > 0 */
    double f_rd;     /* ringdown frequency [Hz] */
    double tau_rd;   /* ringdown damping time [s], > 0 */
} ltdi_chirp;

/* The model sampled on t0 + i dt, i < n: d_hp, d_hc [batch][ld] (device).  d_work: >= 160 bytes per source, 16-byte aligned. */
int ltdi_waveform_chirp(const ltdi_chirp *h_wav, int64_t batch, double t0, double dt, int64_t n, int64_t ld,
                        double *d_hp, double *d_hc, void *d_work, size_t work_bytes, void *stream);

/* The harmonic-sum waveform of an eccentric inspiral (the recipe of BASELINE.json config 5 as a model) on t0 + i dt, i < n:
 * d_tab [batch][7][nk] (device) is the orbital evolution table of every source -- knot times t_k (increasing), orbital
 * frequency F, eccentricity e, mean anomaly l and dF/dt, de/dt, dl/dt at the knots --, carried to the sample time by cubic
 * Hermite interpolation on the knot interval that contains it (the first / last interval outside the table); then
 *   h+ = sum_n [ -(1 + cos^2 iota)(a_n cos 2 gamma - b_n sin 2 gamma) + (1 - cos^2 iota) c_n ],
 *   hx = sum_n 2 cos iota (b_n cos 2 gamma + a_n sin 2 gamma),   n = 1 .. nharm (<= 64),
 *   a_n = -n A [J_{n-2} - 2 e J_{n-1} + (2 / n) J_n + 2 e J_{n+1} - J_{n+2}](n e) cos(n l),
 *   b_n = -n A sqrt(1 - e^2) [J_{n-2} - 2 J_n + J_{n+2}](n e) sin(n l),   c_n = 2 A J_n(n e) cos(n l),
 *   A = (2 pi F M)^(2/3) eta M c / d_L   (Peters & Mathews harmonics in the form of Barack & Cutler 2004, Eqs. 7-9; App. F of
 * the paper uses eccentric signals of this kind).  h_par [batch][6] (host): M = G M_tot / c^3 [s], eta, d_L [m], cos iota,
 * gamma, l0.  n e must stay below 8 (power series of the Bessel functions).  d_hp, d_hc [batch][ld] (device);
 * d_work: >= 64 bytes per source, 16-byte aligned. */
int ltdi_waveform_ecc(const double *d_tab, int64_t nk, const double *h_par, int nharm, int64_t batch, double t0,
                      double dt, int64_t n, int64_t ld, double *d_hp, double *d_hc, void *d_work, size_t work_bytes,
                      void *stream);

/* Full response straight from the model parameters: Eq. (2.5) with h+, hx EVALUATED at the retarded times t - delta_s,
 * t - delta_r (no sampled strain is read and the first interpolation level is gone), then Eq. (2.7) / (2.8) and (2.9) as
 * ltdi_response_full.  h_wav [batch]; ld = row stride of the outputs (>= n); Lagrange orders 9 and 31 (the order only
 * acts in the TDI stage).  The result differs from ltdi_response_full on the sampled model by the interpolation error of
 * the latter (largest where the model's envelope has its kink at the join). */
int ltdi_response_full_chirp(const ltdi_orbits *orb, const ltdi_chirp *h_wav, int64_t ld, int64_t batch,
                             const ltdi_source *h_src, int gen, int lagrange_order, double *d_A, double *d_E,
                             double *d_T, double *d_XYZ, double *d_y, void *d_work, size_t work_bytes, void *stream);

/* Low-frequency approximation: Eq. (B10) links at the retarded time (B1) from central-difference
 * derivatives of h+, hx (S6), Eq. (B25) (gen 1.5) / (B33) (gen 2.0) Michelson (S7).  fd_order 2 | 4.
 * Links -1, -2, -3 are zero. */
int ltdi_response_lfa(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld,
                      int64_t batch, const ltdi_source *h_src, int gen, int lagrange_order, int fd_order,
                      double *d_A, double *d_E, double *d_T, double *d_XYZ, double *d_y, void *d_work,
                      size_t work_bytes, void *stream);

/* higher-order and alternative LFA of the single link.
 *   terms = 1, point = LTDI_LFA_CENTRAL: identical to ltdi_response_lfa (bitwise).
 *   terms = 2 (central point only): the m = 1 term of the odd-derivative series Eq. (B4), P:704,
 *       y = -(L_l / 2) { dH/dt + (1/6) [(L_l / 2)(1 - k.n_l)]^2 d^3H/dt^3 }(tau),
 *     d^3h/dt^3 from the central stencil of accuracy order fd_order (2: (x[2] - 2 x[1] + 2 x[-1] - x[-2]) / (2 dt^3),
 *     4: (-x[3] + 8 x[2] - 13 x[1] + 13 x[-1] - 8 x[-2] + x[-3]) / (8 dt^3)); its stencil is one sample wider than the
 *     first derivative's, so the output margins grow by one sample per side (ltdi_margins_lfa_ext).
 *   point = LTDI_LFA_BACKWARD / LTDI_LFA_FORWARD (terms = 1): the leading-order expressions (B13) / (B14) about the
 *     emission / reception ends of the link, whose residual is first order in the expansion parameter.
 * The Michelson stage is (B25) / (B33) as in ltdi_response_lfa.  Errors as there; LTDI_EINVAL for other terms / point. */
int ltdi_response_lfa_ext(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld,
                          int64_t batch, const ltdi_source *h_src, int gen, int lagrange_order, int fd_order,
                          int terms, int point, double *d_A, double *d_E, double *d_T, double *d_XYZ, double *d_y,
                          void *d_work, size_t work_bytes, void *stream);
int ltdi_margins_lfa_ext(const ltdi_orbit_desc *desc, int gen, int lagrange_order, int fd_order, int terms,
                         int64_t *lo, int64_t *hi);

/* SURVEY.md 8(f)-2, second part: the Michelson variables Taylor-expanded WITHOUT the link-reversal symmetry
 * (L_l = L_-l, y_slr = y_r-ls) that (B25) / (B33) assume -- Eq. (B20) P:832 (gen 1.5) and Eq. (B30) P:894 (gen 2.0): all six
 * LFA links, each from (B10) at its own retarded time (B1), their first and second (gen 2.0: second and third) time
 * derivatives by the central stencils of order fd_order, evaluated at the mid-points (B18) / (B31) of the two arms
 * (reading G13; d/dtau = d/dt).  With P = y_123, Q = y_3-21, U = y_1-32, W = y_231, a = L_-2 + L_2, b = L_-3 + L_3:
 *   X_1.5 = b [P' - (L_-2 / 2) P''] + b [Q' + (L_-2 / 2) Q''] - a [U' - (L_3 / 2) U''] - a [W' + (L_3 / 2) W'']
 *   X_2.0 = (a + b) { the same with one more derivative on every link }.
 * d_y returns all six LFA links.  Output margins grow by one sample for gen 2.0 (ltdi_margins_lfa6).  Runs on the
 * library's generic tile kernel (per-sample weights, plain fp64) for every Lagrange order. */
int ltdi_response_lfa6(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld, int64_t batch,
                       const ltdi_source *h_src, int gen, int lagrange_order, int fd_order, double *d_A, double *d_E,
                       double *d_T, double *d_XYZ, double *d_y, void *d_work, size_t work_bytes, void *stream);
int ltdi_margins_lfa6(const ltdi_orbit_desc *desc, int gen, int lagrange_order, int fd_order, int64_t *lo, int64_t *hi);

/* SURVEY.md 8(f)-4, third part: the full response in the Sagnac-type combinations alpha, beta, gamma ("photons
 * propagating in clockwise and counterclockwise directions around the constellation"; the paper prints no equation, so
 * the textbook form is taken, reading G33).  In the link labelling of P:81 (+1: 3 -> 2, +2: 1 -> 3, +3: 2 -> 1,
 * -1: 2 -> 3, -2: 3 -> 1, -3: 1 -> 2), with the two beams read at spacecraft 1
 *   S+ = y_{+3} + D_{+3} y_{+1} + D_{+3} D_{+1} y_{+2},   S- = y_{-2} + D_{-2} y_{-1} + D_{-2} D_{-1} y_{-3}
 * and the round-trip times T+ = L_3 + L_1 + L_2, T- = L_-2 + L_-1 + L_-3:
 *   gen LTDI_GEN_15: alpha = S+ - S-                             (6 terms: free of laser noise where T+ = T-)
 *   gen LTDI_GEN_20: alpha = (S+ + D_{T+} S-) - (S- + D_{T-} S+) (12 terms: free of laser noise for constant L_l != L_-l)
 * beta, gamma by the cyclic permutation 1 -> 2 -> 3 -> 1; every delay evaluated at t; links from Eq. (2.5).
 * d_abc [3][batch][ld] returns alpha, beta, gamma; d_A, d_E, d_T are Eq. (2.9) applied to them; the margins are those of
 * ltdi_margins for the same generation (the Sagnac delays, 2 and 5 light times, are shorter than the Michelson ones).
 * Arguments, layout and errors as ltdi_response_full.  Runs on the library's generic tile kernel (per-sample weights)
 * for every Lagrange order. */
int ltdi_response_full_sagnac(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld, int64_t batch,
                              const ltdi_source *h_src, int gen, int lagrange_order, double *d_A, double *d_E,
                              double *d_T, double *d_abc, double *d_y, void *d_work, size_t work_bytes, void *stream);

/* Hybrid: LFA for t <= t_hyb + T/2, full for t >= t_hyb - T/2, links blended by Eq. (4.5) and
 * X, Y, Z blended separately by Eq. (4.6) (S8).  h_hyb has n_hyb = 1 or batch entries. */
int ltdi_response_hybrid(const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld,
                         int64_t batch, const ltdi_source *h_src, int gen, int lagrange_order,
                         int fd_order, const ltdi_hybrid *h_hyb, int64_t n_hyb, double *d_A, double *d_E,
                         double *d_T, double *d_XYZ, double *d_y, void *d_work, size_t work_bytes,
                         void *stream);

/* The three responses for callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): the same computation as ltdi_response_full / _lfa / _hybrid (which = LTDI_RESPONSE_*; fd_order and
 * h_hyb / n_hyb as there, ignored where they do not apply), but the caller passes NO workspace -- the scratch (source frames,
 * TDI weight anchors, link series) lives in a file-scope device array of the library of LTDI_STATIC_SCRATCH_BYTES (64 MiB),
 * which every GPU that loads the library holds until the process exits.  The call allocates nothing: no cudaMalloc, cudaFree
 * or allocating library routine, on any call (the first call on a device looks up the array's device address and uploads the
 * library's constant tables: make one call outside a graph capture first).  d_A, d_E, d_T [batch][ld] are the caller's.
 * Limit: ltdi_workspace_bytes(which, n, batch, gen, lagrange_order) must not exceed LTDI_STATIC_SCRATCH_BYTES, else
 * LTDI_EWORKSPACE and nothing is launched (config 2's single source of 518 400 samples fits for all three responses; 4096
 * sources do not: use the calls above with a workspace of the caller's).  Every call on a device shares the one array, which
 * keeps the contents of the last call; nothing in it has to start at zero (each region is written by the call before the
 * call reads it).  Calls that overlap on the GPU -- two streams, two host threads -- RACE on it: serialise them.  Other
 * errors as ltdi_response_full. */
#define LTDI_STATIC_SCRATCH_BYTES ((size_t)64 << 20)
int ltdi_response_static(int which, const ltdi_orbits *orb, const double *d_hp, const double *d_hc, int64_t ld,
                         int64_t batch, const ltdi_source *h_src, int gen, int lagrange_order, int fd_order,
                         const ltdi_hybrid *h_hyb, int64_t n_hyb, double *d_A, double *d_E, double *d_T, void *stream);

/* End-to-end variant (the call a host application makes): h_hp, h_hc [batch][ld] and h_A, h_E, h_T
 * [batch][ld] are HOST buffers (pinned memory makes the copies asynchronous).  The call enqueues, on
 * `stream`, the host->device copies of the strain, the response `which` (LTDI_RESPONSE_*; fd_order and
 * h_hyb / n_hyb as in the calls above, ignored where they do not apply) and the device->host copies of
 * A, E, T.  d_scratch: device scratch of ltdi_host_scratch_bytes() bytes, 256-byte aligned.  Results
 * are valid after the stream is synchronised.  A batch of more than 128 MiB per series is cut into up to 16 pieces of
 * whole sources that pass through upload, kernels and download as a pipeline (the copies on two streams of the
 * library's own, chained to `stream` by events), so that one call keeps both directions of PCIe and the SMs busy; the
 * results are bitwise those of the one-piece call. */
int ltdi_host_scratch_bytes(int64_t ld, int64_t batch, size_t *bytes);
int ltdi_response_host(int which, const ltdi_orbits *orb, const double *h_hp, const double *h_hc, int64_t ld,
                       int64_t batch, const ltdi_source *h_src, int gen, int lagrange_order, int fd_order,
                       const ltdi_hybrid *h_hyb, int64_t n_hyb, double *h_A, double *h_E, double *h_T,
                       void *d_scratch, size_t scratch_bytes, void *stream);

/* ---- SURVEY.md 8(f)-1 (first "next" row): FFT -> noise-weighted inner product, overlap, mismatch, SNR --------- */
/*
 * Steps iv-v of the paper's likelihood evaluation.  Noise model: the analytic "Sangria" PSDs of Sec. II C,
 * Eqs. (2.10)-(2.13): proof-mass and optical-path noise, galactic foreground (2.11) with T_obs in years
 * (2.12), S_n^{A,E} and S_n^T for equal arms with Lambda = 4 sin^2(2x) (TDI 2.0) or 1 (TDI 1.5), x = 2 pi f L / c.
 */
typedef struct {
    double arm_m;     /* L [m] */
    double t_obs_yr;  /* observation time of Eq. (2.12) [yr] (1 in the paper) */
    int32_t gen;      /* LTDI_GEN_15 | LTDI_GEN_20 */
    int32_t galactic; /* 0: without S_gal (lower panel of Fig. 2), 1: with it */
} ltdi_noise_desc;

/* d_psd [2][nf] (device): row 0 = S_n^{A,E}(f_k), row 1 = S_n^T(f_k), f_k = k df; entry k = 0 is +inf. */
int ltdi_noise_psd(const ltdi_noise_desc *desc, double df, int64_t nf, double *d_psd, void *stream);

/* Plan for series of n samples (2 <= n <= 2^27, row stride ld, batch sources): a host object with the lengths and the
 * chunking of the library's own Fourier transform (csrc/fft.cuh: Stockham passes for powers of two, Bluestein's chirp-z
 * for every other n); its device work area is part of the caller's d_work.  Returns the bytes of d_work that
 * ltdi_overlap_products needs. */
typedef struct ltdi_overlap ltdi_overlap;
int ltdi_overlap_create(int64_t n, int64_t ld, int64_t batch, ltdi_overlap **out, size_t *work_bytes);
int ltdi_overlap_destroy(ltdi_overlap *ovl);

/* Two responses a and b (e.g. full and hybrid) as device series A, E, T [batch][ld] each.  Per source and channel
 * c = A, E, T: x~_k = dt DFT(x)_k over all n samples (margins are zero, no window), f_k = k / (n dt), and
 *   <x|y> = 4 Re sum_{fmin <= f_k <= fmax, k > 0} conj(x~_k) y~_k / S_n(f_k) / (n dt)        Eq. (5.1)
 * with S_n = d_psd row 0 for A and E, row 1 for T (nf = n / 2 + 1 entries per row).
 * d_out [batch][3][5]: <a|a>, <b|b>, <a|b>, overlap O = <a|b> / sqrt(<a|a> <b|b>) (5.2), mismatch 1 - |O|.
 * d_snr [batch][3] or NULL: rho = sqrt(<A|A> + <E|E> + <T|T>) of a and of b, Eq. (6.1), and the Gaussian
 * log-likelihood ln L = -1/2 sum_c <a_c - b_c|a_c - b_c> = -1/2 sum_c (<a|a> + <b|b> - 2 <a|b>) of Eq. (D4)
 * with a in the role of the data d and b of the template h.
 * d_work: 256-byte aligned device scratch of work_bytes.  Asynchronous on stream. */
int ltdi_overlap_products(ltdi_overlap *ovl, const double *d_aA, const double *d_aE, const double *d_aT,
                          const double *d_bA, const double *d_bE, const double *d_bT, double dt, const double *d_psd,
                          double fmin, double fmax, double *d_out, double *d_snr, void *d_work, size_t work_bytes,
                          void *stream);

const char *ltdi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LISATDI_H */
