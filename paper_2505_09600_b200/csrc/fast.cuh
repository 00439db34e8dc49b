// fast.cuh -- the tuned sm_100a path for Lagrange orders 9 and 31 (M = 10, 32 taps).
//
// Three kernels per response, the link series y_slr travelling through a scratch buffer (48 B per sample written
// and read once: 0.25 TB/s at the speed of these kernels, far from the HBM roofline):
//
//   anchor_kernel   per time tile of the TDI stage and per distinct TDI delay: integer shift q, and the
//                   Lagrange weights w_k(eps_c) with their first derivative at the tile-centre delay.  The TDI
//                   delays (sums of L_l(t_n)) drift by ~1e-7 samples over a tile, so w_k(eps_n) =
//                   w_k(eps_c) + D w_k' with D = eps_n - eps_c: the neglected term (D^2 / 2) sum_k w_k'' x_k =
//                   (D^2 / 2) dt^2 x''(t) is <= 1.3e-13 (omega dt)^2 |x| for the checked bound |D| <= 5e-7
//                   (a tile that fails the check, or whose q changes, takes the exact
//                   per-sample weights instead).  The weights do not depend on the source: a batch shares them.
//   link_kernel     S2 + S3 (Eq. 2.4-2.6) resp. S6 (Eq. B10): one thread owns TWO consecutive samples, builds
//                   the per-sample weights of each of the 9 (3) retarded times from the symmetric pair form
//                   below, and streams the shared 33-sample window of h+ / hx out of shared memory once for
//                   both samples (the shared-memory pipe, not the FP64 pipe, limits a one-sample-per-thread
//                   kernel: SURVEY.md section 7, hard part 4).
//   tdi_kernel      S4 + S5 (Eq. 2.7-2.9) resp. S7 (B25/B33) and S8 (4.5/4.6): one thread owns SEVEN
//                   consecutive samples of one Michelson channel and slides a 7-sample register window over
//                   the link series (stride-7 shared-memory reads are conflict free), weights broadcast from
//                   the anchors.
//
// Symmetric pair form of the Lagrange weights.  Taps k = -(H-1) .. H (M = 2H), eps in [0,1).  Pair j = 0..H-1
// holds taps k = j+1 and k = -j, nodes +-(j+1/2) about u = eps - 1/2:
//   prod_{m != k}(eps - m) = (eps + j) G_j      (k = j+1),      ((j+1) - eps) G_j * (-1)   (k = -j)
//   G_j = prod_{i != j} g_i,   g_i = u^2 - (i+1/2)^2 = (eps + i)(eps - i - 1)
// and 1 / prod_{m != k}(k - m) = +-c_j.  Scaling g_i by lambda_i with prod_{i != j} lambda_i = c_j folds the
// denominators into the products: w_{j+1} = Gt_j (eps + j), w_{-j} = Gt_j (j + 1 - eps), Gt_j = prod_{i != j}
// lambda_i g_i  -- 3.4 M flops per weight set instead of 5 M for prefix x suffix over all taps.
#pragma once
#include "common.cuh"
#include "dd.cuh"
#include "chirp.cuh"

#define FAST_TC_R 7                       /* samples per thread in the TDI kernel */
#define FAST_TCA 448                      /* samples per anchor tile */
/* TDI tile geometry per response: G thread groups per channel, 7 G samples per tile, 3 G threads.  Full: one warp
 * per Michelson channel (224 samples, 96 threads, four CTAs per SM at 168 registers).  LFA: 448 samples, 192
 * threads, four CTAs per SM at 80 registers (its tiles are latency-bound: two interpolations per channel).
 * Hybrid: 448 samples, 192 threads, two CTAs per SM (it needs the shared memory of both responses). */
__host__ __device__ constexpr int tdi_g(int which) { return which == LTDI_RESPONSE_FULL ? 32 : 64; }
__host__ __device__ constexpr int tdi_tc(int which) { return FAST_TC_R * tdi_g(which); }
__host__ __device__ constexpr int tdi_threads(int which) { return 3 * tdi_g(which); }
#define FAST_TA_THREADS 128
#define FAST_TA (2 * FAST_TA_THREADS)     /* 256 samples per link tile, three CTAs per SM */
#define FAST_TAL (FAST_TA - 4)            /* LFA link tiles: 256 link samples give the time derivative of 252 (two samples of rim
                                           * on either side serve the widest stencil and keep the tile start even) */
#define FAST_NA_FULL 39                   /* anchors per tile: 3 channels x 13 delays */
#define FAST_NA_LFA 12                    /* 2 generations x 3 channels x 2 delays (gen 1.5 first) */
#define FAST_NA_LFA_GEN 6                 /* those of one generation */
#define FAST_NA (FAST_NA_FULL + FAST_NA_LFA)
#define FAST_DMAX 5.0e-7                  /* |eps_n - eps_c| bound for the first-order weights */
#define FAST_DMAX2 5.0e-5                 /* bound for the second-order weights: the neglected (D^3 / 6)(omega dt)^3 |x| <= 2e-14 |x| */
/* one anchor = [M] double2 {w_k, w_k'}, in doubles */
#define FAST_ANC_DOUBLES(M) (2 * (M))

/* lambda_i and kappa_i = -lambda_i (i + 1/2)^2 for H = 5 (row 0) and H = 16 (row 1) */
__constant__ double c_sym_lam[2][16];
__constant__ double c_sym_kap[2][16];

struct FastParams {
    const double *tab;
    int64_t stride, n;
    double t0, dt, inv_dt;
    double inv_fd1, inv_fd2; /* 1 / (2 dt) | 1 / (12 dt) and 1 / dt^2 | 1 / (12 dt^2): stencil denominators (fd 2 | 4) */
    const double *hp, *hc;
    int64_t ld, batch;       /* batch = sources of this launch (a chunk) */
    const double *frames;    /* [batch][LTDI_FRAME_STRIDE] of this chunk (use_small == 0) */
    int use_small;           /* batch_all <= 32: sources and hybrid windows travel in `small` as kernel arguments and
                              * every CTA derives its source frame itself (no parameter kernel in front of the call) */
    double small[32 * 7];    /* [32][3] beta, lambda, psi, then [32][4] t_hyb, window, sigma, taper (by absolute source) */
    double small_fr[32 * 11]; /* [32][11] source frames k, u, v, cos 2psi, sin 2psi (S1, formed on the host in long double: as
                              * one thread's three sincos in front of every CTA it cost the single-source configs ~1 us per tile) */
    const double *hyb;       /* [n_hyb][4] of this chunk (t_hyb, window, sigma, taper) */
    int64_t n_hyb;
    int which, gen, fd;
    int lfa_terms, lfa_point, xw;   /* terms of Eq. (B4), expansion point LTDI_LFA_*, xw = terms - 1 */
    double inv_fd3;                 /* 1 / (2 dt^3) | 1 / (8 dt^3): third-derivative stencil denominator (fd 2 | 4) */
    int64_t m1, m2, w, lo, hi;
    int64_t m2_15, m2_20;    /* anchor kernel: backward TDI reach of either generation (the anchors serve both) */
    int qmax;
    double *yF, *yL;         /* scratch [6][batch][lds]: full links; [3][batch][lds]: TIME DERIVATIVE (gen 1.5: first, gen 2.0:
                              * second) of the LFA links, formed by the link kernel itself */
    double *yLraw;           /* [3][batch][lds] the LFA links themselves, written only when the caller asks for d_y */
    int64_t lds;
    double *A, *E, *T, *XYZ, *Y; /* outputs of this chunk ([batch][ld] ...), XYZ / Y strides use batch_all */
    int64_t batch_all, b0;   /* full batch and first source of the chunk (for the [3][batch][ld] outputs) */
    const double *anc;       /* [anchor tiles][FAST_NA][M][2] */
    const double *anc_hdr;   /* [anchor tiles][FAST_NA][4]: d_c [s], q, eps_c, valid (0 no, 1 first order, 2 second order only) */
    const double *anc2;      /* [anchor tiles][FAST_NA][M]: w_k'' (second-order instances; nullptr otherwise) */
    int nested;              /* properly nested TDI delays (full response; second-order instance) */
    int64_t ntilesA, ntilesC;
    /* hybrid: compact work lists built by hybrid_plan_kernel (x = source of the chunk, y = tile); a launch runs exactly
     * the tiles of its class.  work == nullptr: every tile of every source (id = tile * batch + source). */
    const int2 *work;
    int64_t nwork;           /* items of this launch */
    int64_t nwork_full;      /* link_hybrid_kernel: the first nwork_full items are full-link tiles, the rest LFA-link tiles */
};

/* item id -> (source of the chunk, tile) */
__device__ __forceinline__ void work_item(const FastParams &p, int64_t id, int64_t &b, int64_t &tile)
{
    if (p.work) {
        const int2 it = p.work[id];
        b = it.x;
        tile = it.y;
    } else {
        b = id % p.batch;
        tile = id / p.batch;
    }
}

// ---------------------------------------------------------------------------------------------
// helpers
// ---------------------------------------------------------------------------------------------
// Ampere-style asynchronous copies (LDGSTS): the staging loops issue all their loads at once and wait once
__device__ __forceinline__ void cp_async8(void *dst_smem, const void *src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async16(void *dst_smem, const void *src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// TMA 1-D bulk copies (cp.async.bulk) completing on an mbarrier: ONE thread moves a whole row, the other threads
// spend no instruction on staging (the per-element cp.async loops of the TDI kernel were a third of its executed
// instructions, ncu r02a).  Addresses and sizes are multiples of 16 bytes.
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    unsigned ok;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok)
                     : "r"(smem_u32(bar)), "r"(parity)
                     : "memory");
    } while (!ok);
}

// s = d / dt to within one rounding of the correctly rounded quotient (one Newton correction)
__device__ __forceinline__ double div_dt(double d, double dt, double inv_dt)
{
    const double s0 = d * inv_dt;
    const double r = fma(-s0, dt, d);
    return fma(r, inv_dt, s0);
}

__device__ __forceinline__ void split_delay_fast(double d, double dt, double inv_dt, int &q, double &eps)
{
    const double s = div_dt(d, dt, inv_dt);
    const double qc = ceil(s);
    q = (int)qc;
    eps = qc - s;
}

// generic exact weights (prefix x suffix over all taps), used by the rare slow paths
template <int M>
__device__ __noinline__ void lagrange_exact(double eps, double *w)
{
    const double *c = c_lag_inv_den + (M / 2 - 1) * LTDI_MAX_TAPS;
    const int kmin = -(M / 2 - 1);
    double run = 1.0;
    for (int i = 0; i < M; ++i) {
        w[i] = run;
        run *= eps - (double)(kmin + i);
    }
    run = 1.0;
    for (int i = M - 1; i >= 0; --i) {
        w[i] = (w[i] * run) * c[i];
        run *= eps - (double)(kmin + i);
    }
}

// ---------------------------------------------------------------------------------------------
// the pair interpolator of the link kernel
// ---------------------------------------------------------------------------------------------
// Window W[i] = x[js + i], i = 0 .. M: sample 0 uses W[0..M-1], sample 1 uses W[1..M].  The staged series are
// split by parity (even samples / odd samples), so that lanes that own consecutive sample PAIRS read
// consecutive addresses.  W[i] = (i odd ? p1[(i-1)/2] : p0[i/2]).
//
// DIFF: the dot products run over x_k - x_ref (x_ref = the window's centre sample, returned in pref / cref) and the
// caller adds x_ref back: sum_k w_k x_k = x_ref + sum_k w_k (x_k - x_ref) because the weights sum to 1.  The
// differences of neighbouring samples are exact or nearly so, and the rounding errors of the weights and of the
// accumulation now scale with |x_k - x_ref| ~ 16 omega dt |x| instead of |x|: for the low-frequency signals whose
// LFA response amplifies the noise of y by 1 / (omega dt)^2 (Eq. (B33)) the interpolation stops contributing to it.
template <int H, bool DIFF>
__device__ __forceinline__ void interp_pair(double e0, double e1, const double *__restrict__ P0,
                                            const double *__restrict__ P1, const double *__restrict__ C0,
                                            const double *__restrict__ C1, double &ap0, double &ac0, double &ap1,
                                            double &ac1, double &pref, double &cref)
{
    constexpr int row = (H == 16) ? 1 : 0;
    const double uu0 = (e0 - 0.5) * (e0 - 0.5), uu1 = (e1 - 0.5) * (e1 - 0.5);
    // suffix products S[j] = prod_{i > j} lambda_i g_i
    double S0[H], S1[H];
    S0[H - 1] = 1.0;
    S1[H - 1] = 1.0;
#pragma unroll
    for (int j = H - 2; j >= 0; --j) {
        const double g0 = fma(c_sym_lam[row][j + 1], uu0, c_sym_kap[row][j + 1]);
        const double g1 = fma(c_sym_lam[row][j + 1], uu1, c_sym_kap[row][j + 1]);
        S0[j] = S0[j + 1] * g0;
        S1[j] = S1[j + 1] * g1;
    }
    // centre of the window
#define W_AT(Q0, Q1, i) (((i) & 1) ? (Q1)[((i) - 1) >> 1] : (Q0)[(i) >> 1])
    double plo = W_AT(P0, P1, H), clo = W_AT(C0, C1, H);
    pref = DIFF ? plo : 0.0;
    cref = DIFF ? clo : 0.0;
    if (DIFF) { plo = 0.0; clo = 0.0; }
    double phi = plo, chi = clo;
    double a_p0 = 0.0, a_c0 = 0.0, a_p1 = 0.0, a_c1 = 0.0;
    double pre0 = 1.0, pre1 = 1.0;
#pragma unroll
    for (int j = 0; j < H; ++j) {
        const double G0 = pre0 * S0[j], G1 = pre1 * S1[j];
        const double t0 = G0 * e0, t1 = G1 * e1;
        const double w0p = fma(G0, (double)j, t0), w0m = fma(G0, (double)(j + 1), -t0); /* taps k = j+1, k = -j */
        const double w1p = fma(G1, (double)j, t1), w1m = fma(G1, (double)(j + 1), -t1);
        const double pl = W_AT(P0, P1, H - 1 - j) - pref, ph = W_AT(P0, P1, H + 1 + j) - pref;
        const double cl = W_AT(C0, C1, H - 1 - j) - cref, ch = W_AT(C0, C1, H + 1 + j) - cref;
        a_p0 = fma(w0m, pl, a_p0);
        a_p0 = fma(w0p, phi, a_p0);
        a_c0 = fma(w0m, cl, a_c0);
        a_c0 = fma(w0p, chi, a_c0);
        a_p1 = fma(w1m, plo, a_p1);
        a_p1 = fma(w1p, ph, a_p1);
        a_c1 = fma(w1m, clo, a_c1);
        a_c1 = fma(w1p, ch, a_c1);
        plo = pl; phi = ph; clo = cl; chi = ch;
        if (j + 1 < H) {
            if (j == 0) {
                pre0 = c_sym_lam[row][0] * (e0 * (e0 - 1.0)); /* g_0 = eps (eps - 1): no cancellation near 0, 1 */
                pre1 = c_sym_lam[row][0] * (e1 * (e1 - 1.0));
            } else {
                pre0 *= fma(c_sym_lam[row][j], uu0, c_sym_kap[row][j]);
                pre1 *= fma(c_sym_lam[row][j], uu1, c_sym_kap[row][j]);
            }
        }
    }
#undef W_AT
    ap0 = a_p0; ac0 = a_c0; ap1 = a_p1; ac1 = a_c1;
}

// one sample, taps ascending, exact weights: the pair's two samples have different integer shifts
template <int H>
__device__ __noinline__ void interp_single(double eps, const double *he_p, const double *ho_p, const double *he_c,
                                           const double *ho_c, int js /* window start relative to the staged origin */,
                                           double &ap, double &ac)
{
    double w[2 * H];
    lagrange_exact<2 * H>(eps, w);
    double sp = 0.0, sc = 0.0;
    for (int i = 0; i < 2 * H; ++i) {
        const int g = js + i;
        const double xp = (g & 1) ? ho_p[g >> 1] : he_p[g >> 1];
        const double xc = (g & 1) ? ho_c[g >> 1] : he_c[g >> 1];
        sp = fma(w[i], xp, sp);
        sc = fma(w[i], xc, sc);
    }
    ap = sp;
    ac = sc;
}

// interpolate both series at the two samples m0, m0+1 of a pair with delays d0, d1 [s]
template <int H, bool DIFF>
__device__ __forceinline__ void interp_delays(const FastParams &p, double d0, double d1, int rel0 /* m0 - origin */,
                                              const double *he_p, const double *ho_p, const double *he_c,
                                              const double *ho_c, double &ap0, double &ac0, double &ap1, double &ac1,
                                              double &pref, double &cref)
{
    int q0, q1;
    double e0, e1;
    split_delay_fast(d0, p.dt, p.inv_dt, q0, e0);
    split_delay_fast(d1, p.dt, p.inv_dt, q1, e1);
    q0 = max(-p.qmax, min(p.qmax, q0));
    q1 = max(-p.qmax, min(p.qmax, q1));
    const int js = rel0 - q0 - (H - 1); /* >= 0 by the margin bound */
    if (q0 == q1) {
        const int c = js >> 1;
        const double *P0, *P1, *C0, *C1;
        if (js & 1) { P0 = ho_p + c; P1 = he_p + c + 1; C0 = ho_c + c; C1 = he_c + c + 1; }
        else        { P0 = he_p + c; P1 = ho_p + c;     C0 = he_c + c; C1 = ho_c + c; }
        interp_pair<H, DIFF>(e0, e1, P0, P1, C0, C1, ap0, ac0, ap1, ac1, pref, cref);
    } else {
        pref = 0.0;
        cref = 0.0;
        interp_single<H>(e0, he_p, ho_p, he_c, ho_c, js, ap0, ac0);
        interp_single<H>(e1, he_p, ho_p, he_c, ho_c, rel0 + 1 - q1 - (H - 1), ap1, ac1);
    }
}

// ---------------------------------------------------------------------------------------------
// accurate antenna patterns of the LFA links.  F+ = n^T P+ n and Fx = n^T Px n with the symmetric matrices
//   P+ = (u u^T - v v^T) cos 2psi + (u v^T + v u^T) sin 2psi,   Px = (u v^T + v u^T) cos 2psi - (u u^T - v v^T) sin 2psi
// of the source (Eqs. (2.2)-(2.4) with G17 written as quadratic forms).  A quadratic form expands EXACTLY about the
// link vector n_c of the tile centre:  F(n_c + d) = F(n_c) + (2 P n_c) . d + d^T P d.  F(n_c) is evaluated once per
// tile, link and source in double-double from the dd link vector of the table; d = n - n_c is ~1e-4 over a tile
// (the constellation turns by 2e-7 rad/s), so the bracket is evaluated in plain fp64 with an absolute error of
// 1e-20, and F(n) = hi + (lo + bracket) is a double-double value for ~40 flops per sample and link.  (Rounding
// errors of P itself are constant in time: a smooth relative offset of 1e-16, which no stencil amplifies.)
// anchor layout (doubles): 0-1 F+_c hi lo, 2-3 Fx_c hi lo, 4-6 g+ = 2 P+ n_c, 7-9 gx, 10-12 n_c hi, 13-15 n_c lo,
// 16-21 P+ (xx yy zz xy xz yz), 22-27 Px
// ---------------------------------------------------------------------------------------------
#define LFA_ANC_DOUBLES 28
#define LFA_LO_ROWS 12
/* a staged low-part row: floats of samples a0 - 2 .. a0 + FAST_TA + 1 (+ padding), so that the copy starts on a 16-byte
 * boundary although an LFA tile starts at a0 = 2 (mod 4); sample a0 + i sits at element 2 + i */
#define LFA_TLW (FAST_TA + 8)
/* doubles of the raw-strain region of the LFA link kernel: two series of 2 hw2 + 2 LFA_RAW_HALO samples, and at least the
 * three link rows of the tile that take its place after the stencil pass */
__host__ __device__ constexpr int lfa_raw_doubles(int hw2) { return 2 * (2 * hw2 + 8) > 3 * FAST_TA ? 2 * (2 * hw2 + 8) : 3 * FAST_TA; }
#define LFA_RAW_HALO 4   /* raw strain staged beyond the FD series on either side: the widest stencil (d^3/dt^3, order 4) needs 3;
                          * even, so that the staged run starts on a 16-byte boundary for the bulk copy */

// One warp per link: lanes 0..15 = (polarisation = lane >> 3, element e = lane & 7); e < 6 holds one element P_e of the
// symmetric matrix and its term (1 | 2) P_e n_a n_b of the quadratic form in double-double, summed over the eight lanes
// of the polarisation by a shuffle tree; lanes 16..21 form g = 2 P n_c, lanes 22..24 store n_c.  (As three serial
// threads this was a fifth of the kernel's time: everybody else waited at the barrier behind ~600 dependent flops.)
__device__ __forceinline__ void lfa_anchor_warp(const double *fr, const double *tb, const float *tl, int l, int ic,
                                                double *s_anc, int lane)
{
    double *an = s_anc + l * LFA_ANC_DOUBLES;
    const double *u = fr + 3, *v = fr + 6;
    const double c2 = fr[9], s2 = fr[10];
    const int pol = (lane >> 3) & 1, e = lane & 7;
    const int ia = e < 3 ? e : (e == 5 ? 1 : 0), ib = e < 3 ? e : (e == 3 ? 1 : 2);   /* xx yy zz xy xz yz */
    const bool term = lane < 16 && e < 6;
    const int ja = term ? ia : 0, jb = term ? ib : 0;
    const double dp = u[ja] * u[jb] - v[ja] * v[jb];     /* (2.4a) as a matrix */
    const double dc = u[ja] * v[jb] + v[ja] * u[jb];     /* (2.4b) */
    const double P = pol == 0 ? dp * c2 + dc * s2 : dc * c2 - dp * s2;   /* (2.2) + (2.3), G17 */
    const dd na = dd_make(tb[(ROW_N + 3 * l + ja) * FAST_TA + ic], (double)tl[(LO_N + 3 * l + ja) * LFA_TLW + 2 + ic]);
    const dd nb = dd_make(tb[(ROW_N + 3 * l + jb) * FAST_TA + ic], (double)tl[(LO_N + 3 * l + jb) * LFA_TLW + 2 + ic]);
    dd t = dd_mul_d(dd_mul(na, nb), e < 3 ? P : 2.0 * P);
    if (!term) t = dd_make(0.0, 0.0);
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) {
        const dd q = dd_make(__shfl_xor_sync(0xffffffffu, t.hi, o), __shfl_xor_sync(0xffffffffu, t.lo, o));
        t = dd_add(t, q);
    }
    if (lane < 16 && e == 0) { an[2 * pol] = t.hi; an[2 * pol + 1] = t.lo; }
    if (term) an[16 + 6 * pol + e] = P;
    /* g[a] = 2 sum_b P_ab n_b: lanes 16..21 = (polarisation, a) */
    const int gl = lane - 16, gpol = gl >= 3 ? 1 : 0, ga = gl - 3 * gpol;
    const int a_ = (gl >= 0 && gl < 6) ? ga : 0;
    const int e0 = a_ == 0 ? 0 : (a_ == 1 ? 3 : 4), e1 = a_ == 0 ? 3 : (a_ == 1 ? 1 : 5), e2 = a_ == 0 ? 4 : (a_ == 1 ? 5 : 2);
    const int base = 8 * ((gl >= 0 && gl < 6) ? gpol : 0);
    const double P0 = __shfl_sync(0xffffffffu, P, base + e0), P1 = __shfl_sync(0xffffffffu, P, base + e1),
                 P2 = __shfl_sync(0xffffffffu, P, base + e2);
    if (gl >= 0 && gl < 6) {
        const double n0 = tb[(ROW_N + 3 * l) * FAST_TA + ic], n1 = tb[(ROW_N + 3 * l + 1) * FAST_TA + ic],
                     n2 = tb[(ROW_N + 3 * l + 2) * FAST_TA + ic];
        an[4 + 3 * gpol + ga] = 2.0 * (P0 * n0 + P1 * n1 + P2 * n2);
    }
    if (lane >= 22 && lane < 25) {
        const int a = lane - 22;
        an[10 + a] = tb[(ROW_N + 3 * l + a) * FAST_TA + ic];
        an[13 + a] = (double)tl[(LO_N + 3 * l + a) * LFA_TLW + 2 + ic];
    }
}

// y^LFA of one sample: n = (nx, ny, nz) + (lx, ly, lz), L = L_hi + L_lo, dh/dt numerators (pref + ap), (cref + ac)
__device__ __forceinline__ double lfa_link_value(const double *an, double nx, double ny, double nz, double lx, double ly,
                                                 double lz, double L_hi, double L_lo, double kscale, double pref, double ap,
                                                 double cref, double ac)
{
    const double dx = (nx - an[10]) + (lx - an[13]), dy = (ny - an[11]) + (ly - an[14]), dz = (nz - an[12]) + (lz - an[15]);
    const double *P = an + 16, *Q = an + 22;
    const double tp0 = fma(P[0], dx, fma(P[3], dy, P[4] * dz)), tp1 = fma(P[3], dx, fma(P[1], dy, P[5] * dz)),
                 tp2 = fma(P[4], dx, fma(P[5], dy, P[2] * dz));
    const double tc0 = fma(Q[0], dx, fma(Q[3], dy, Q[4] * dz)), tc1 = fma(Q[3], dx, fma(Q[1], dy, Q[5] * dz)),
                 tc2 = fma(Q[4], dx, fma(Q[5], dy, Q[2] * dz));
    const double Fp_lo = an[1] + fma(an[4] + tp0, dx, fma(an[5] + tp1, dy, (an[6] + tp2) * dz));
    const double Fc_lo = an[3] + fma(an[7] + tc0, dx, fma(an[8] + tc1, dy, (an[9] + tc2) * dz));
    const double Fp_hi = an[0], Fc_hi = an[2];
    const dd Sp = two_sum(pref, ap), Sc = two_sum(cref, ac);
    dd a = two_prod(Fp_hi, Sp.hi), b = two_prod(Fc_hi, Sc.hi);
    a.lo = fma(Fp_lo, Sp.hi, fma(Fp_hi, Sp.lo, a.lo));
    b.lo = fma(Fc_lo, Sc.hi, fma(Fc_hi, Sc.lo, b.lo));
    dd sum = two_sum(a.hi, b.hi);
    sum.lo += a.lo + b.lo;
    dd c = two_prod(L_hi, kscale);
    c.lo = fma(L_lo, kscale, c.lo);
    const dd y = two_prod(sum.hi, c.hi);
    return y.hi + fma(sum.lo, c.hi, fma(sum.hi, c.lo, y.lo));
}

// ---------------------------------------------------------------------------------------------
// link kernel: LFA == false: Eq. (2.5), six links;  LFA == true: Eq. (B10) at (B1), links +1, +2, +3
// ---------------------------------------------------------------------------------------------
template <int H, bool LFA>
__device__ __forceinline__ void link_body(const FastParams &p, int64_t bid)
{
    extern __shared__ double smem[];
    int64_t b, tile;
    work_item(p, bid, b, tile);
    /* first link sample of the tile (even).  LFA: the tile also differentiates its links in time (G15) and stores the
     * derivative of its inner FAST_TAL samples, so consecutive tiles overlap by the rim of the stencil */
    const int64_t a0 = LFA ? tile * FAST_TAL - 2 : tile * FAST_TA;
    const int tid = threadIdx.x;
    const int w = LFA ? (int)p.w : 0;

    __shared__ double fr[LTDI_FRAME_STRIDE];
    __shared__ double s_anc[LFA ? 3 * LFA_ANC_DOUBLES : 1];
    if (p.use_small) {
        if (tid < 11) fr[tid] = p.small_fr[11 * (p.b0 + b) + tid];   /* S1, Eq. (2.1) with G1, (2.3) */
    } else if (tid < LTDI_FRAME_STRIDE) fr[tid] = p.frames[b * LTDI_FRAME_STRIDE + tid];

    /* staged strain: samples [org, org + 2 * hw2), org even; parity split; LFA: FD1 numerators of the strain */
    const int64_t org = a0 - p.m1 - (p.m1 & 1);
    const int hw2 = (int)((FAST_TA + 2 * p.m1 + 4) / 2);   /* pairs */
    double *he_p = smem, *ho_p = he_p + hw2, *he_c = ho_p + hw2, *ho_c = he_c + hw2;
    const double *gp = p.hp + b * p.ld, *gc = p.hc + b * p.ld;
    /* orbit-table rows of the tile: rows 0..23 (full) or 0..20 (LFA: R, n, L_+l), [row][FAST_TA].  Contiguous runs go
     * through TMA bulk copies on an mbarrier, issued by the lanes of warp 0 (one row each): as per-element cp.async
     * loops the staging was a fifth of the LFA kernel's executed instructions (ncu r02a).  A row is copied up to the
     * table stride; what lies beyond (a tail tile) is only read by samples >= n, whose outputs are never stored. */
    constexpr int NROWS = LFA ? ROW_L + 3 : LTDI_TABLE_ROWS;
    double *tb = ho_c + hw2;
    __shared__ uint64_t s_bar, s_bar2;   /* s_bar2 (LFA): the table rows, which the stencil pass does not need */
    const int64_t tl0 = max(a0, (int64_t)0), tl1 = min(a0 + FAST_TA, p.stride);       /* table samples of the tile */
    const unsigned nl = (unsigned)max(tl1 - tl0, (int64_t)0);                          /* even */
    const int toff = (int)(tl0 - a0);                                                  /* 0, or 2 in the first LFA tile */
    float *tl = nullptr;   /* LFA: low parts of the dd table entries of the tile */
    double *he3_p = nullptr; /* LFA, terms = 2: [4][hw2] third-derivative numerators (even +, odd +, even x, odd x) */
    if (!LFA) {
        if (tid == 0) {
            mbar_init(&s_bar, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            mbar_expect_tx(&s_bar, NROWS * nl * 8u);
        }
        __syncthreads();   /* the barrier is initialised: every fourth thread issues one row (all four warps issue) */
        if ((tid & 3) == 0 && (tid >> 2) < NROWS)
            bulk_g2s(tb + (tid >> 2) * FAST_TA + toff, p.tab + (int64_t)(tid >> 2) * p.stride + tl0, nl * 8u, &s_bar);
        for (int i = tid; i < 2 * hw2; i += FAST_TA_THREADS) {
            const int64_t g = org + i;
            double *dp = ((i & 1) ? ho_p : he_p) + (i >> 1), *dc = ((i & 1) ? ho_c : he_c) + (i >> 1);
            if (g >= 0 && g < p.n) {
                cp_async8(dp, gp + g);
                cp_async8(dc, gc + g);
            } else {
                *dp = 0.0;
                *dc = 0.0;
            }
        }
        cp_async_wait_all();
        __syncthreads();
        mbar_wait(&s_bar, 0);
    } else {
        /* raw strain of samples org - 4 .. org + 2 hw2 + 3, then the FD1 numerators (G15); low parts of n_l (9 rows)
         * and of L_+l (3 rows): float rows LO_N .. LO_L + 2 of the table */
        const int nraw = 2 * hw2 + 2 * LFA_RAW_HALO;
        double *raw_p = tb + NROWS * FAST_TA, *raw_c = raw_p + nraw;
        tl = reinterpret_cast<float *>(raw_p + lfa_raw_doubles(hw2));   /* the raw region later holds the tile's links */
        const int64_t rs = org - LFA_RAW_HALO;                                   /* even */
        const int64_t g_lo = max(rs, (int64_t)0), g_hi = min(rs + nraw, p.n);
        const int ncopy = (int)max(g_hi - g_lo, (int64_t)0);
        /* one bulk copy per series needs 16-byte aligned ends (an odd ld or n falls back to element copies) */
        const int64_t f0 = max(a0 - 2, (int64_t)0), f1 = min(a0 + FAST_TA + 2, p.stride);   /* low-part samples, multiples of 4 */
        const unsigned nf = (unsigned)max(f1 - f0, (int64_t)0);
        const bool bulk = ncopy > 0 && !(ncopy & 1) &&
                          !((reinterpret_cast<uintptr_t>(gp + g_lo) | reinterpret_cast<uintptr_t>(gc + g_lo)) & 15);
        if (tid == 0) {
            mbar_init(&s_bar, 1);
            mbar_init(&s_bar2, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            mbar_expect_tx(&s_bar, bulk ? 2u * ncopy * 8u : 0u);
            mbar_expect_tx(&s_bar2, NROWS * nl * 8u + LFA_LO_ROWS * nf * 4u);
        }
        __syncthreads();   /* the barriers are initialised */
        if (tid % 3 == 0) {   /* 35 copies, one per issuing thread, spread over the four warps; the raw strain first */
            const int id = tid / 3;
            if (id < 2) {
                if (bulk) bulk_g2s((id == 0 ? raw_p : raw_c) + (g_lo - rs), (id == 0 ? gp : gc) + g_lo, ncopy * 8u, &s_bar);
            } else if (id < 2 + NROWS) {
                const int r = id - 2;
                bulk_g2s(tb + r * FAST_TA + toff, p.tab + (int64_t)r * p.stride + tl0, nl * 8u, &s_bar2);
            } else if (id < 2 + NROWS + LFA_LO_ROWS) {   /* float rows from sample a0 - 2 (a multiple of 4) on: see LFA_TLW */
                const int r = id - 2 - NROWS;
                const float *glo = reinterpret_cast<const float *>(p.tab + (int64_t)LTDI_TABLE_ROWS * p.stride);
                bulk_g2s(tl + r * LFA_TLW + (f0 - (a0 - 2)), glo + (int64_t)r * p.stride + f0, nf * 4u, &s_bar2);
            }
        }
        if (!bulk || ncopy < nraw)   /* interior tiles (all but two per source) have nothing to fill and nothing to copy by element */
            for (int j = tid; j < nraw; j += FAST_TA_THREADS) {
                const int64_t g = rs + j;
                if (g < g_lo || g >= g_hi) {
                    raw_p[j] = 0.0;
                    raw_c[j] = 0.0;
                } else if (!bulk) {
                    cp_async8(raw_p + j, gp + g);
                    cp_async8(raw_c + j, gc + g);
                }
            }
        /* SURVEY 8(f)-2, terms = 2: the d^3h/dt^3 numerators, parity-split like the first-derivative series */
        he3_p = reinterpret_cast<double *>(tl + LFA_LO_ROWS * LFA_TLW);
        cp_async_wait_all();
        __syncthreads();
        mbar_wait(&s_bar, 0);      /* the raw strain: the stencil pass runs while the table rows are still arriving */
        const int ws = w + p.xw;   /* the widest stencil applied to the strain */
        for (int i = tid; i < 2 * hw2; i += FAST_TA_THREADS) {
            const int64_t g = org + i;
            double vp = 0.0, vc = 0.0;
            if (g >= ws && g < p.n - ws) {
                const double *xp = raw_p + i + LFA_RAW_HALO, *xc = raw_c + i + LFA_RAW_HALO;
                if (w == 1) {
                    vp = xp[1] - xp[-1];
                    vc = xc[1] - xc[-1];
                } else {
                    vp = 8.0 * (xp[1] - xp[-1]) - (xp[2] - xp[-2]);
                    vc = 8.0 * (xc[1] - xc[-1]) - (xc[2] - xc[-2]);
                }
                if (p.lfa_terms >= 2) {
                    const double p1 = xp[1] - xp[-1], p2 = xp[2] - xp[-2], c1 = xc[1] - xc[-1], c2 = xc[2] - xc[-2];
                    double tp, tc;
                    if (w == 1) { tp = p2 - 2.0 * p1; tc = c2 - 2.0 * c1; }
                    else { tp = 8.0 * p2 - 13.0 * p1 - (xp[3] - xp[-3]); tc = 8.0 * c2 - 13.0 * c1 - (xc[3] - xc[-3]); }
                    he3_p[((i & 1) ? hw2 : 0) + (i >> 1)] = tp;
                    he3_p[((i & 1) ? 3 * hw2 : 2 * hw2) + (i >> 1)] = tc;
                }
            } else if (p.lfa_terms >= 2) {
                he3_p[((i & 1) ? hw2 : 0) + (i >> 1)] = 0.0;
                he3_p[((i & 1) ? 3 * hw2 : 2 * hw2) + (i >> 1)] = 0.0;
            }
            ((i & 1) ? ho_p : he_p)[i >> 1] = vp;
            ((i & 1) ? ho_c : he_c)[i >> 1] = vc;
        }
        mbar_wait(&s_bar2, 0);     /* the table rows and their low parts */
        /* tile anchors of the antenna patterns: warp l builds the anchor of link l */
        if (tid < 96) lfa_anchor_warp(fr, tb, tl, tid >> 5, (int)max(min((int64_t)(FAST_TA / 2), p.n - 1 - a0), (int64_t)toff), s_anc, tid & 31);
        __syncthreads();
    }

    const int64_t m0 = a0 + 2 * tid;
    if (!LFA && m0 >= p.n) return;
    const int rel0 = (int)(m0 - org);
    const int64_t vlo = p.m1 + w + (LFA ? p.xw : 0), vhi = p.n - vlo;   /* valid link samples */
    const bool in0 = m0 >= vlo && m0 < vhi, in1 = m0 + 1 >= vlo && m0 + 1 < vhi;
    double *yout = p.yF + b * p.lds + m0;                /* full links: straight to the scratch */
    double *ysm = LFA ? tb + NROWS * FAST_TA : nullptr;  /* LFA links of the tile [3][FAST_TA], on top of the raw strain (done with) */
    const int64_t ystride = p.batch * p.lds;
    if (!in0 && !in1) {
        if (!LFA) {
#pragma unroll
            for (int l = 0; l < 6; ++l) *reinterpret_cast<double2 *>(yout + l * ystride) = make_double2(0.0, 0.0);
            return;
        }
#pragma unroll
        for (int l = 0; l < 3; ++l) *reinterpret_cast<double2 *>(ysm + l * FAST_TA + 2 * tid) = make_double2(0.0, 0.0);
    } else {

    const double *t = tb + 2 * tid;
    const double inv_c = 1.0 / LTDI_C_LIGHT;
    auto row2 = [&](int r) { return *reinterpret_cast<const double2 *>(t + r * FAST_TA); };
    /* k . R_i / c [s] of the two samples; i may be a run-time index (rows come from shared memory) */
    auto kdotR = [&](int i, double &k0, double &k1) {
        const double2 x = row2(ROW_R + 3 * i), y = row2(ROW_R + 3 * i + 1), z = row2(ROW_R + 3 * i + 2);
        k0 = (fr[0] * x.x + fr[1] * y.x + fr[2] * z.x) * inv_c;
        k1 = (fr[0] * x.y + fr[1] * y.y + fr[2] * z.y) * inv_c;
    };
    /* F^+, F^x (2.2)-(2.4) with G17 and k . n of link |l| = a + 1 for the two samples */
    auto patterns = [&](int a, double &Fp0, double &Fc0, double &kn0, double &Fp1, double &Fc1, double &kn1) {
        const double2 nx = row2(ROW_N + 3 * a), ny = row2(ROW_N + 3 * a + 1), nz = row2(ROW_N + 3 * a + 2);
        {
            const double un = fr[3] * nx.x + fr[4] * ny.x + fr[5] * nz.x;
            const double vn = fr[6] * nx.x + fr[7] * ny.x + fr[8] * nz.x;
            kn0 = fr[0] * nx.x + fr[1] * ny.x + fr[2] * nz.x;
            const double xip = un * un - vn * vn, xic = 2.0 * un * vn;   /* (2.4) */
            Fp0 = xip * fr[9] + xic * fr[10];                              /* (2.2) + (2.3), G17 */
            Fc0 = xic * fr[9] - xip * fr[10];
        }
        {
            const double un = fr[3] * nx.y + fr[4] * ny.y + fr[5] * nz.y;
            const double vn = fr[6] * nx.y + fr[7] * ny.y + fr[8] * nz.y;
            kn1 = fr[0] * nx.y + fr[1] * ny.y + fr[2] * nz.y;
            const double xip = un * un - vn * vn, xic = 2.0 * un * vn;
            Fp1 = xip * fr[9] + xic * fr[10];
            Fc1 = xic * fr[9] - xip * fr[10];
        }
    };

    /* ONE instance of the pair interpolator in a rolled loop: the kernel stays small enough for the instruction
     * cache (nine inlined copies made 113 KB of code and "no instruction" the top stall reason). */
    if (!LFA) {
        /* step = 3 r + s: receiver spacecraft r, then the two links it receives: s = 1: link +((r+2)%3 + 1) sent by
         * spacecraft (r+1)%3, s = 2: link -((r+1)%3 + 1) sent by spacecraft (r+2)%3 */
        double rp0 = 0.0, rc0 = 0.0, rp1 = 0.0, rc1 = 0.0; /* h+, hx at the receiver time t - k.R_r / c (2.6b) */
#pragma unroll 1
        for (int step = 0; step < 9; ++step) {
            const int r = step / 3, s = step - 3 * r;
            const int a = s == 1 ? (r + 2) % 3 : (r + 1) % 3;   /* |l| - 1 */
            const int l = s == 2 ? a + 3 : a;
            const int sc = s == 0 ? r : (s == 1 ? (r + 1) % 3 : (r + 2) % 3);
            double k0, k1;
            kdotR(sc, k0, k1);
            double d0 = k0, d1 = k1;
            if (s != 0) {
                const double2 L = row2(ROW_L + l);
                d0 = L.x + k0;                                           /* (2.6a) */
                d1 = L.y + k1;
            }
            double ap0, ac0, ap1, ac1, pref, cref;
            interp_delays<H, false>(p, d0, d1, rel0, he_p, ho_p, he_c, ho_c, ap0, ac0, ap1, ac1, pref, cref);
            if (s == 0) {
                rp0 = ap0; rc0 = ac0; rp1 = ap1; rc1 = ac1;
            } else {
                double Fp0, Fc0, kn0, Fp1, Fc1, kn1;
                patterns(a, Fp0, Fc0, kn0, Fp1, Fc1, kn1);
                const double e0 = 2.0 * (1.0 - (s == 2 ? -kn0 : kn0)), e1 = 2.0 * (1.0 - (s == 2 ? -kn1 : kn1));
                const double y0 = (Fp0 * (ap0 - rp0) + Fc0 * (ac0 - rc0)) / e0;   /* (2.5) */
                const double y1 = (Fp1 * (ap1 - rp1) + Fc1 * (ac1 - rc1)) / e1;
                *reinterpret_cast<double2 *>(yout + l * ystride) = make_double2(in0 ? y0 : 0.0, in1 ? y1 : 0.0);
            }
        }
    } else {
        /* (B10): y = -(L_l / 2) (F+ dh+/dt + Fx dhx/dt) with every factor that multiplies the result carried as a
         * double-double pair and one rounding at the end (dd.cuh: Eq. (B33) amplifies white noise of y by
         * 2.45 / (omega dt)^2).  The stencil denominator 1 / (2 dt) is a constant factor (its rounding is a constant
         * relative offset of 1e-16, not noise). */
        const double kscale = -0.5 * p.inv_fd1;
        const float *tlo = tl + 2 + 2 * tid;
#pragma unroll 1
        for (int l = 0; l < 3; ++l) {
            const int s = link_sender(l), r = link_receiver(l);
            double ks0, ks1, kr0, kr1;
            kdotR(s, ks0, ks1);
            kdotR(r, kr0, kr1);
            const double2 L = row2(ROW_L + l);
            double ap0, ac0, ap1, ac1, pref, cref;
            double d0, d1;
            if (p.lfa_point == LTDI_LFA_CENTRAL) { d0 = 0.5 * L.x + 0.5 * (ks0 + kr0); d1 = 0.5 * L.y + 0.5 * (ks1 + kr1); }   /* (B1) */
            else if (p.lfa_point == LTDI_LFA_BACKWARD) { d0 = L.x + ks0; d1 = L.y + ks1; }                                    /* (B13) */
            else { d0 = kr0; d1 = kr1; }                                                                                       /* (B14) */
            interp_delays<H, true>(p, d0, d1, rel0, he_p, ho_p, he_c, ho_c, ap0, ac0, ap1, ac1, pref, cref);
            if (p.lfa_terms >= 2) {
                /* m = 1 term of Eq. (B4): + (1/6) [(L_l / 2)(1 - k.n_l)]^2 d^3H/dt^3 at the same retarded time;
                 * relative to dH/dt it is (omega Delta / 2)^2 / 6, so plain fp64 serves: it joins the small part of the
                 * (reference + difference) pair of the first-derivative numerators */
                double bp0, bc0, bp1, bc1, p3, c3;
                interp_delays<H, true>(p, d0, d1, rel0, he3_p, he3_p + hw2, he3_p + 2 * hw2, he3_p + 3 * hw2, bp0, bc0, bp1, bc1, p3, c3);
                const double2 nx = row2(ROW_N + 3 * l), ny = row2(ROW_N + 3 * l + 1), nz = row2(ROW_N + 3 * l + 2);
                const double h0 = (0.5 * L.x) * (1.0 - (fr[0] * nx.x + fr[1] * ny.x + fr[2] * nz.x));
                const double h1 = (0.5 * L.y) * (1.0 - (fr[0] * nx.y + fr[1] * ny.y + fr[2] * nz.y));
                const double r31 = p.inv_fd3 / p.inv_fd1 / 6.0;
                const double f0 = h0 * h0 * r31, f1 = h1 * h1 * r31;
                ap0 = fma(f0, p3 + bp0, ap0); ac0 = fma(f0, c3 + bc0, ac0);
                ap1 = fma(f1, p3 + bp1, ap1); ac1 = fma(f1, c3 + bc1, ac1);
            }
            const double *an = s_anc + l * LFA_ANC_DOUBLES;
            const double2 nx = row2(ROW_N + 3 * l), ny = row2(ROW_N + 3 * l + 1), nz = row2(ROW_N + 3 * l + 2);
            const float2 lx = *reinterpret_cast<const float2 *>(tlo + (LO_N + 3 * l) * LFA_TLW);
            const float2 ly = *reinterpret_cast<const float2 *>(tlo + (LO_N + 3 * l + 1) * LFA_TLW);
            const float2 lz = *reinterpret_cast<const float2 *>(tlo + (LO_N + 3 * l + 2) * LFA_TLW);
            const float2 lL = *reinterpret_cast<const float2 *>(tlo + (LO_L + l) * LFA_TLW);
            const double y0 = lfa_link_value(an, nx.x, ny.x, nz.x, (double)lx.x, (double)ly.x, (double)lz.x, L.x,
                                             (double)lL.x, kscale, pref, ap0, cref, ac0);
            const double y1 = lfa_link_value(an, nx.y, ny.y, nz.y, (double)lx.y, (double)ly.y, (double)lz.y, L.y,
                                             (double)lL.y, kscale, pref, ap1, cref, ac1);
            *reinterpret_cast<double2 *>(ysm + l * FAST_TA + 2 * tid) = make_double2(in0 ? y0 : 0.0, in1 ? y1 : 0.0);
        }
    }
    }   /* in0 || in1 */
    if (LFA) {
        /* time derivative of the tile's links (G15; gen 1.5: first, gen 2.0: second; zero outside its valid range), which is
         * what the Michelson stage interpolates, Eq. (B25) / (B33): the TDI kernel stages it directly and has no stencil pass */
        __syncthreads();
        if (tid == 0 || tid == FAST_TA_THREADS - 1 || m0 >= p.n) return;   /* the rim pairs belong to the neighbouring tiles */
        const bool g15 = p.gen == LTDI_GEN_15;
        const double scale = g15 ? p.inv_fd1 : p.inv_fd2;
        const int64_t dlo = p.m1 + 2 * w + p.xw;
#pragma unroll
        for (int l = 0; l < 3; ++l) {
            const double *v = ysm + l * FAST_TA + 2 * tid;   /* v[j] = link sample m0 + j */
            double d[2];
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                double x;
                if (w == 1) x = g15 ? (v[j + 1] - v[j - 1]) : ((v[j + 1] - v[j]) - (v[j] - v[j - 1]));
                else if (g15) x = 8.0 * (v[j + 1] - v[j - 1]) - (v[j + 2] - v[j - 2]);
                else {
                    const double d1 = (v[j + 1] - v[j]) - (v[j] - v[j - 1]);
                    const double d2 = (v[j + 2] - v[j]) - (v[j] - v[j - 2]);
                    x = 16.0 * d1 - d2;
                }
                const int64_t m = m0 + j;
                d[j] = (m >= dlo && m < p.n - dlo) ? x * scale : 0.0;
            }
            *reinterpret_cast<double2 *>(p.yL + b * p.lds + l * ystride + m0) = make_double2(d[0], d[1]);
            if (p.yLraw) *reinterpret_cast<double2 *>(p.yLraw + b * p.lds + l * ystride + m0) = make_double2(v[0], v[1]);
        }
    }
}

#ifndef LINK_MINB
#define LINK_MINB 3
#endif
template <int H, bool LFA>
__global__ void __launch_bounds__(FAST_TA_THREADS, LINK_MINB) link_kernel(const __grid_constant__ FastParams p)
{
    link_body<H, LFA>(p, blockIdx.x);
}

// Eq. (2.5) with the strain of the chirp + ringdown model evaluated AT the nine retarded times of a sample
// (chirp.cuh) instead of interpolated from a sampled series: no strain is read, nothing is staged but the source frame;
// a thread owns two consecutive samples and reads its table entries straight from global memory (coalesced double2).
// The link series go to the same scratch as link_kernel's: the TDI stage is unchanged.
__global__ void __launch_bounds__(FAST_TA_THREADS, 3) link_chirp_kernel(const __grid_constant__ FastParams p,
                                                                       const ChirpDev *__restrict__ wav /* of the chunk */)
{
    const int64_t b = (int64_t)blockIdx.x % p.batch, tile = (int64_t)blockIdx.x / p.batch;
    const int64_t a0 = tile * FAST_TA;
    const int tid = threadIdx.x;
    __shared__ double fr[LTDI_FRAME_STRIDE];
    __shared__ ChirpDev sw;
    if (p.use_small) {
        if (tid < 11) fr[tid] = p.small_fr[11 * (p.b0 + b) + tid];
    } else if (tid < LTDI_FRAME_STRIDE) fr[tid] = p.frames[b * LTDI_FRAME_STRIDE + tid];
    if (tid >= 32 && tid < 32 + LTDI_CHIRP_STRIDE) reinterpret_cast<double *>(&sw)[tid - 32] = reinterpret_cast<const double *>(wav + b)[tid - 32];
    __syncthreads();
    const int64_t m0 = a0 + 2 * tid;
    if (m0 >= p.n) return;
    const int64_t vlo = p.m1, vhi = p.n - p.m1;
    const bool in0 = m0 >= vlo && m0 < vhi, in1 = m0 + 1 >= vlo && m0 + 1 < vhi;
    double *yout = p.yF + b * p.lds + m0;
    const int64_t ystride = p.batch * p.lds;
    if (!in0 && !in1) {
#pragma unroll
        for (int l = 0; l < 6; ++l) *reinterpret_cast<double2 *>(yout + l * ystride) = make_double2(0.0, 0.0);
        return;
    }
    const double *t = p.tab + m0;
    const double inv_c = 1.0 / LTDI_C_LIGHT;
    auto row2 = [&](int r) { return *reinterpret_cast<const double2 *>(t + (int64_t)r * p.stride); };
    const dd s0 = two_prod((double)m0, p.dt), s1 = two_prod((double)(m0 + 1), p.dt);   /* t_n - t0 */
    double rp0 = 0.0, rc0 = 0.0, rp1 = 0.0, rc1 = 0.0;
#pragma unroll 1
    for (int step = 0; step < 9; ++step) {   /* receiver r, then the two links it receives (as link_body) */
        const int r = step / 3, s = step - 3 * r;
        const int a = s == 1 ? (r + 2) % 3 : (r + 1) % 3;
        const int l = s == 2 ? a + 3 : a;
        const int sc = s == 0 ? r : (s == 1 ? (r + 1) % 3 : (r + 2) % 3);
        const double2 x = row2(ROW_R + 3 * sc), y = row2(ROW_R + 3 * sc + 1), z = row2(ROW_R + 3 * sc + 2);
        double d0 = (fr[0] * x.x + fr[1] * y.x + fr[2] * z.x) * inv_c;
        double d1 = (fr[0] * x.y + fr[1] * y.y + fr[2] * z.y) * inv_c;
        if (s != 0) {
            const double2 L = row2(ROW_L + l);
            d0 = L.x + d0;                                           /* (2.6a) */
            d1 = L.y + d1;
        }
        double ap0, ac0, ap1, ac1;
        chirp_eval(sw, dd_add_d(s0, -d0), ap0, ac0);
        chirp_eval(sw, dd_add_d(s1, -d1), ap1, ac1);
        if (s == 0) {
            rp0 = ap0; rc0 = ac0; rp1 = ap1; rc1 = ac1;
        } else {
            const double2 nx = row2(ROW_N + 3 * a), ny = row2(ROW_N + 3 * a + 1), nz = row2(ROW_N + 3 * a + 2);
            double y01[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const double n0 = h ? nx.y : nx.x, n1 = h ? ny.y : ny.x, n2 = h ? nz.y : nz.x;
                const double un = fr[3] * n0 + fr[4] * n1 + fr[5] * n2, vn = fr[6] * n0 + fr[7] * n1 + fr[8] * n2;
                const double kn = fr[0] * n0 + fr[1] * n1 + fr[2] * n2;
                const double xip = un * un - vn * vn, xic = 2.0 * un * vn;   /* (2.4) */
                const double Fp = xip * fr[9] + xic * fr[10], Fc = xic * fr[9] - xip * fr[10];   /* (2.2) + (2.3), G17 */
                const double e = 2.0 * (1.0 - (s == 2 ? -kn : kn));
                y01[h] = (Fp * ((h ? ap1 : ap0) - (h ? rp1 : rp0)) + Fc * ((h ? ac1 : ac0) - (h ? rc1 : rc0))) / e;   /* (2.5) */
            }
            *reinterpret_cast<double2 *>(yout + l * ystride) = make_double2(in0 ? y01[0] : 0.0, in1 ? y01[1] : 0.0);
        }
    }
}

// hybrid: both kinds of link tiles in ONE launch -- the few full-link tiles (first in the grid: they are the heavy
// ones) run beside the LFA-link tiles instead of as a launch of their own that leaves most SMs idle
template <int H>
__global__ void __launch_bounds__(FAST_TA_THREADS, LINK_MINB) link_hybrid_kernel(const __grid_constant__ FastParams p)
{
    if ((int64_t)blockIdx.x < p.nwork_full) link_body<H, false>(p, blockIdx.x);
    else link_body<H, true>(p, blockIdx.x);
}

// ---------------------------------------------------------------------------------------------
// TDI delays.  Channel ch = 0,1,2 (X,Y,Z; cyclic): i2 = (1+ch)%3, i3 = (2+ch)%3,
// dP = L[i2+3], dU = L[i3], a = L[i2+3] + L[i2], b = L[i3] + L[i3+3].  The 13 distinct delays of a channel are
// base + i a + j b with base in {0, dP, dU}:
// ---------------------------------------------------------------------------------------------
struct DelayDef { signed char base, i, j; };   /* base: 0 none, 1 dP, 2 dU */
__constant__ DelayDef c_delay_def[13] = {
    {1, 0, 0}, {1, 0, 1}, {0, 0, 1}, {2, 0, 0}, {2, 1, 0}, {0, 1, 0}, {1, 1, 1},
    {1, 1, 2}, {0, 1, 1}, {0, 1, 2}, {2, 1, 1}, {2, 2, 1}, {0, 2, 1}};
/* The 14 interpolated terms of Eq. (2.7) / (2.8): series (0 P, 1 Q, 2 U, 3 W), delay id, sign, and the link whose light
 * time the term adds to the delay of the term before it (0: +p3, 1: -p3, 2: -p2, 3: +p2).  They are ordered along the
 * two chains of delay operators that generate them (oracle O12; a = D_-p2 D_p2, b = D_p3 D_-p3):
 *   terms 0..6:  D_p3 U, b Q, b D_-p2 P, b a Q, b a D_-p2 P, b a a W, b a a D_p3 U      (all with sign -)
 *   terms 7..13: D_-p2 P, a W, a D_p3 U, a b W, a b D_p3 U, a b b Q, a b b D_-p2 P      (all with sign +)
 * so that with nested delays every term extends the delay of its predecessor by one light time.  TDI 1.5 uses the
 * first three of either chain. */
struct TermDef { signed char series, delay, sign, link; };
__constant__ TermDef c_term_def[14] = {
    {2, 3, -1, 0}, {1, 2, -1, 1}, {0, 1, -1, 2}, {1, 8, -1, 3}, {0, 6, -1, 2}, {3, 12, -1, 3}, {2, 11, -1, 0},
    {0, 0, +1, 2}, {3, 5, +1, 3}, {2, 4, +1, 0}, {3, 8, +1, 1}, {2, 10, +1, 0}, {1, 9, +1, 1}, {0, 7, +1, 2}};

__device__ __forceinline__ double tdi_delay(int id, double dP, double dU, double a, double b)
{
    /* the same expressions, in the same order, as the slow path and the oracle use */
    switch (id) {
    case 0: return dP;
    case 1: return dP + b;
    case 2: return b;
    case 3: return dU;
    case 4: return dU + a;
    case 5: return a;
    case 6: return dP + a + b;
    case 7: return dP + a + 2.0 * b;
    case 8: return a + b;
    case 9: return a + 2.0 * b;
    case 10: return dU + a + b;
    case 11: return dU + 2.0 * a + b;
    default: return 2.0 * a + b;
    }
}
/* LFA delays (B25) / (B33): id 0: arm i2 term (series d123-like), id 1: arm i3 term */
__device__ __forceinline__ double lfa_delay(int gen, int id, double L2, double L3)
{
    if (gen == LTDI_GEN_15) return id == 0 ? L3 + 0.5 * L2 : L2 + 0.5 * L3;
    return id == 0 ? 2.0 * L3 + 1.5 * L2 : 2.0 * L2 + 1.5 * L3;
}

// ---------------------------------------------------------------------------------------------
// anchor kernel: one block per TDI tile; thread a < FAST_NA builds the anchor of delay a
// ---------------------------------------------------------------------------------------------
template <int M>
__global__ void __launch_bounds__(64) anchor_kernel(const __grid_constant__ FastParams p, double *anc, double *hdr, double *anc2 /* w'' or nullptr */)
{
    const int64_t tile = blockIdx.x;
    const int64_t n0 = tile * FAST_TCA, n1 = min(n0 + (int64_t)FAST_TCA, p.n);
    const int64_t nc = min(n0 + FAST_TCA / 2, p.n - 1);
    const int tid = threadIdx.x;
    __shared__ double dev[6]; /* max |L_l(n) - L_l(nc)| over the tile */
    __shared__ double Lc[6];
    /* warp w < 2 reduces rows 3w .. 3w+2: coalesced sweeps over the tile, then a shuffle tree */
    {
        const int warp = tid >> 5, lane = tid & 31;
#pragma unroll
        for (int r = 0; r < 3; ++r) {
            const double *row = p.tab + (int64_t)(ROW_L + 3 * warp + r) * p.stride;
            const double c = row[nc];
            double v[FAST_TCA / 32];   /* all loads of the sweep in flight at once (index clamped: max is idempotent) */
#pragma unroll
            for (int k = 0; k < FAST_TCA / 32; ++k) v[k] = row[min(n0 + lane + 32 * k, n1 - 1)];
            double d = 0.0;
#pragma unroll
            for (int k = 0; k < FAST_TCA / 32; ++k) d = fmax(d, fabs(v[k] - c));
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) d = fmax(d, __shfl_xor_sync(0xffffffffu, d, o));
            if (lane == 0) {
                dev[3 * warp + r] = d;
                Lc[3 * warp + r] = c;
            }
        }
    }
    __syncthreads();
    if (tid >= FAST_NA) return;
    double d, bound;
    int64_t m2;   /* the halo of the generation that uses this delay */
    if (tid < FAST_NA_FULL) {
        const int ch = tid / 13, id = tid % 13;
        const int i2 = (1 + ch) % 3, i3 = (2 + ch) % 3;
        const double dP = Lc[i2 + 3], dU = Lc[i3], a = Lc[i2 + 3] + Lc[i2], b = Lc[i3] + Lc[i3 + 3];
        d = tdi_delay(id, dP, dU, a, b);
        const DelayDef df = c_delay_def[id];
        bound = (df.base == 1 ? dev[i2 + 3] : df.base == 2 ? dev[i3] : 0.0) + df.i * (dev[i2 + 3] + dev[i2]) +
                df.j * (dev[i3] + dev[i3 + 3]);
        m2 = id < 6 ? p.m2_15 : p.m2_20;   /* delays 0..5 are the ones of Eq. (2.7), used by both generations */
    } else {
        const int k = tid - FAST_NA_FULL, gen = k < FAST_NA_LFA_GEN ? LTDI_GEN_15 : LTDI_GEN_20;
        const int ch = (k % FAST_NA_LFA_GEN) / 2, id = k % 2;
        const int i2 = (1 + ch) % 3, i3 = (2 + ch) % 3;
        d = lfa_delay(gen, id, Lc[i2], Lc[i3]);
        bound = 2.0 * (dev[i2] + dev[i3]);
        m2 = gen == LTDI_GEN_15 ? p.m2_15 : p.m2_20;
    }
    bound *= p.inv_dt;
    /* properly nested delays (oracle O12) differ from the sums of L_l(t_n) by at most sum_j |dL_cj/dt| d, and the rates
     * are bounded by the deviations over the half tile: an allowance of 2 d / (half tile) on top */
    bound *= 1.0 + 2.0 * d / (fmax((double)max(nc - n0, n1 - 1 - nc), 1.0) * p.dt);
    int q;
    double eps;
    split_delay_fast(d, p.dt, p.inv_dt, q, eps);
    /* usable if the Taylor remainder is below rounding (first-order weights: FAST_DMAX; with w'' stored: FAST_DMAX2), the
     * integer shift cannot change inside the tile and the stencil stays inside the staged halo */
    const bool ok = bound <= (anc2 ? FAST_DMAX2 : FAST_DMAX) && eps - bound >= 0.0 && eps + bound < 1.0 && q >= 0 &&
                    q + M / 2 <= m2;
    double *h = hdr + (tile * FAST_NA + tid) * 4;
    h[0] = d; h[1] = (double)q; h[2] = eps; h[3] = ok ? (bound <= FAST_DMAX ? 1.0 : 2.0) : 0.0;

    /* w_k = c_k pre_k suf_k with pre_k = prod_{m<k}(eps - m), suf_k = prod_{m>k}(eps - m); the first (and second)
     * derivative by the product rule carried along the same sweeps */
    double2 *out = reinterpret_cast<double2 *>(anc + (tile * FAST_NA + tid) * (int64_t)FAST_ANC_DOUBLES(M));
    double *out2 = anc2 ? anc2 + (tile * FAST_NA + tid) * (int64_t)M : nullptr;
    const double *c = c_lag_inv_den + (M / 2 - 1) * LTDI_MAX_TAPS;
    constexpr int kmin = -(M / 2 - 1);
    double pf[M], pf1[M], pf2[M];
    {
        double f = 1.0, f1 = 0.0, f2 = 0.0;
#pragma unroll
        for (int i = 0; i < M; ++i) {
            pf[i] = f; pf1[i] = f1; pf2[i] = f2;
            const double e = eps - (double)(kmin + i);
            f2 = f2 * e + 2.0 * f1;
            f1 = f1 * e + f;
            f = f * e;
        }
    }
    double g = 1.0, g1 = 0.0, g2 = 0.0;
#pragma unroll
    for (int i = M - 1; i >= 0; --i) {
        double2 o;
        o.x = c[i] * (pf[i] * g);
        o.y = c[i] * (pf1[i] * g + pf[i] * g1);
        out[i] = o;
        if (out2) out2[i] = c[i] * (pf2[i] * g + 2.0 * pf1[i] * g1 + pf[i] * g2);
        const double e = eps - (double)(kmin + i);
        g2 = g2 * e + 2.0 * g1;
        g1 = g1 * e + g;
        g = g * e;
    }
}

// ---------------------------------------------------------------------------------------------
// TDI kernel
// ---------------------------------------------------------------------------------------------
// staged link window of a TDI tile: it starts tdi_back(m2) >= m2 samples before the tile (even, so that the
// rows can be copied in 16-byte pieces) and holds tdi_yr<M>(m2) samples (even)
__host__ __device__ __forceinline__ int tdi_back(int64_t m2) { return (int)((m2 + 1) & ~(int64_t)1); }
template <int M>
__host__ __device__ __forceinline__ int tdi_yr(int tc, int64_t m2) { return (tc + tdi_back(m2) + M / 2 + 2 + 1) & ~1; }

// exact per-sample interpolation of a staged series (slow path): ys[0] = sample y0, length len
template <int M>
__device__ __noinline__ double slow_delayed(const double *ys, int len, int idx /* n - y0 */, double delay, double dt,
                                            double inv_dt)
{
    int q;
    double eps;
    split_delay_fast(delay, dt, inv_dt, q, eps);
    double w[M];
    lagrange_exact<M>(eps, w);
    const int j = idx - q - (M / 2 - 1);
    double acc = 0.0;
    for (int i = 0; i < M; ++i) {
        const int jj = j + i;
        if (jj >= 0 && jj < len) acc = fma(w[i], ys[jj], acc);
    }
    return acc;
}

// Eqs. (4.1), (4.5) with G18; raised cosine, G20
__device__ __forceinline__ void hybrid_weights_fast(const double *h, double t, double &w_lfa, double &w_full)
{
    const double x0 = t - h[0], T = h[1];
    if (h[3] == (double)LTDI_TAPER_SIGMOID) {
        w_lfa = (x0 <= 0.5 * T) ? 1.0 / (1.0 + exp(x0 / h[2])) : 0.0;
        w_full = (x0 >= -0.5 * T) ? 1.0 / (1.0 + exp(-x0 / h[2])) : 0.0;
    } else {
        const double x = (x0 + 0.5 * T) / T;
        if (x <= 0.0) w_full = 0.0;
        else if (x >= 1.0) w_full = 1.0;
        else w_full = 0.5 * (1.0 - cospi(x));
        w_lfa = 1.0 - w_full;
    }
}


// FAST_TC_R consecutive outputs of one interpolated term.  With D = eps_n - eps_c,
//   sum_k w_k(eps_c + D) x_k = S0 + D S1,   S_m = sum_k w_k^(m)(eps_c) x_k :
// two constant-coefficient FIR filters over the tile, 2 DFMA per tap and sample in FAST_TC_R x 2 independent
// chains; the weights are broadcast reads, the samples slide through a register window.
// ORD2 (orbits whose light times drift by more than FAST_DMAX over a tile: numerical orbit files, caller's tables):
// every thread first moves the weights to the delay of ITS OWN centre sample with the second-order Taylor step
//   w_k(eps_c + Dt) = w_k + Dt (w_k' + Dt w_k'' / 2),   w_k'(eps_c + Dt) = w_k' + Dt w_k''
// (3 DFMA per tap and thread) and the caller applies the first-order step for the remaining eps_n - eps_c - Dt of its
// seven samples (three samples of drift: < 1e-7); neglected: Dt^3 / 6 times the third derivative of the weights and
// (eps_n - eps_c - Dt)^2 / 2 times the second.
/* (tile, channel) pairs that took the exact per-sample weights instead of the anchors (ltdi_profile_slow_tiles) */
__device__ unsigned long long d_slow_tiles;

/* header code of an anchor: 1 = first-order weights suffice, 2 = second-order weights needed, 0 = neither */
template <bool ORD2>
__device__ __forceinline__ bool anchor_ok(double code) { return ORD2 ? code != 0.0 : code == 1.0; }

template <int M, bool ORD2>
__device__ __forceinline__ void term7(const double *__restrict__ anc, const double *__restrict__ anc2, double Dt,
                                      const double *__restrict__ x, double (&s0)[FAST_TC_R], double (&s1)[FAST_TC_R])
{
    const double2 *w01 = reinterpret_cast<const double2 *>(anc);
    double win[FAST_TC_R];
#pragma unroll
    for (int r = 0; r < FAST_TC_R; ++r) { s0[r] = 0.0; s1[r] = 0.0; }
#pragma unroll
    for (int r = 0; r < FAST_TC_R - 1; ++r) win[r] = x[r];
    const double hDt = 0.5 * Dt;
#pragma unroll
    for (int k = 0; k < M; ++k) {
        double2 w = w01[k];
        if (ORD2) {
            const double w2 = anc2[k];
            w.x = fma(Dt, fma(hDt, w2, w.y), w.x);
            w.y = fma(Dt, w2, w.y);
        }
        win[(k + FAST_TC_R - 1) % FAST_TC_R] = x[k + FAST_TC_R - 1];
#pragma unroll
        for (int r = 0; r < FAST_TC_R; ++r) {
            const double xv = win[(k + r) % FAST_TC_R];
            s0[r] = fma(w.x, xv, s0[r]);
            s1[r] = fma(w.y, xv, s1[r]);
        }
    }
}

// Light travel time of a staged row (element 0 = sample y0 of the tile window) at t_i - d: centred Lagrange
// interpolation of order 3 (reading G29, oracle O12): taps k = -1 .. 2 about sample i - ceil(d / dt)
__device__ __forceinline__ double light_time_at(const double *__restrict__ Lrow, int i, double d, double dt, double inv_dt)
{
    int q;
    double e;
    split_delay_fast(d, dt, inv_dt, q, e);
    q = max(0, min(q, i - 1));   /* samples past the end of the series carry no light times: stay inside the row */
    const double *x = Lrow + (i - q);
    const double em1 = e - 1.0, em2 = e - 2.0, ep1 = e + 1.0;
    const double wm = -(e * em1) * em2 * (1.0 / 6.0), w0 = (ep1 * em1) * em2 * 0.5, w1 = -(ep1 * e) * em2 * 0.5,
                 w2 = (ep1 * e) * em1 * (1.0 / 6.0);
    return fma(wm, x[-1], fma(w0, x[0], fma(w1, x[1], w2 * x[2])));
}

// WHICH = LTDI_RESPONSE_*: the full-only and LFA-only instances carry no code or registers of the other branch.
// ORD2: second-order weights (see term7) and, for the full response, optionally nested delays (p.nested).
#ifndef TDI_LFA_MINB
#define TDI_LFA_MINB 4
#endif
template <int M, int WHICH, bool ORD2>
__global__ void __launch_bounds__(tdi_threads(WHICH), WHICH == LTDI_RESPONSE_HYBRID ? 2 : (WHICH == LTDI_RESPONSE_LFA ? TDI_LFA_MINB : (ORD2 ? 3 : 4)))
tdi_kernel(const __grid_constant__ FastParams p)
{
    extern __shared__ double smem[];
    constexpr int FAST_TC = tdi_tc(WHICH), FAST_TC_G = tdi_g(WHICH), FAST_TC_THREADS = tdi_threads(WHICH);
    constexpr int FAST_TCA_TILES = FAST_TCA / FAST_TC;
    constexpr int H = M / 2;
    constexpr int ANC = FAST_ANC_DOUBLES(M);
    constexpr bool has_full = WHICH != LTDI_RESPONSE_LFA, has_lfa = WHICH != LTDI_RESPONSE_FULL;
    constexpr int NLR = has_full ? 6 : 3;   /* light-time rows the tile needs (LFA: the positive links) */
    int64_t b, tile;
    work_item(p, blockIdx.x, b, tile);
    const int64_t n0 = tile * FAST_TC;
    const int64_t n1 = min(n0 + (int64_t)FAST_TC, p.n);
    const int tid = threadIdx.x;
    const int w = (int)p.w;

    /* The hybrid response (p.which == HYBRID) runs as three launches over compact tile lists (hybrid_plan_kernel): the
     * LFA instance takes the 448-sample blocks that lie entirely before the window (w_Full = 0; it applies w_LFA in
     * its epilogue), the HYBRID instance the blocks the window touches (both responses, blended by (4.6)), and the
     * FULL instance -- no LFA shared memory, four CTAs per SM -- the 224-sample tiles entirely after the window
     * (w_LFA = 0; it applies w_Full in its epilogue). */
    constexpr bool need_full = WHICH != LTDI_RESPONSE_LFA, need_lfa = WHICH != LTDI_RESPONSE_FULL;
    const bool hybrid_mode = p.which == LTDI_RESPONSE_HYBRID;
    const double *hy = nullptr;
    if (hybrid_mode) hy = p.use_small ? p.small + 96 + 4 * (p.n_hyb == 1 ? 0 : p.b0 + b) : p.hyb + 4 * (p.n_hyb == 1 ? 0 : b);

    /* shared memory (host: tdi_smem_bytes):
     *   sa   anchors [na][ANC]            (39 full, then 6 LFA; only the kinds this response has)
     *   yF   [6][yr] full links           dL  [3][yr] time derivative of the LFA links, as the link kernel stored it
     *                                          (element 0 = sample y0, even)
     *   Lr   [NLR][FAST_TC] light times L_l(n0 + i) of the tile; after the term loop: X, Y, Z of the tile
     *        (full response with second-order weights: [6][yr], element 0 = sample y0 -- nested delays look back)
     *   Xs   [3][FAST_TC] exchange        sa2  [na][M] second derivative of the weights (ORD2) */
    const int yr = tdi_yr<M>(FAST_TC, p.m2);
    const int64_t y0 = n0 - tdi_back(p.m2);
    constexpr int na_full = has_full ? FAST_NA_FULL : 0;
    double *sa = smem;
    double *yF = sa + (size_t)(na_full + (has_lfa ? FAST_NA_LFA_GEN : 0)) * ANC;
    double *dL = yF + (has_full ? 6 * yr : 0);
    constexpr bool LR_EXT = ORD2 && WHICH == LTDI_RESPONSE_FULL;
    const int LRW = LR_EXT ? yr : FAST_TC;                       /* elements per light-time row */
    const int lroff = LR_EXT ? tdi_back(p.m2) : 0;               /* element of sample n0 */
    double *Lr = dL + (has_lfa ? 3 * yr : 0);
    double *Xs0 = Lr + NLR * LRW;
    /* X, Y, Z exchange: its own region (full, LFA: no barrier between the term loop and the exchange), or on top of
     * the light times (hybrid: six rows, and the shared memory of two responses) */
    constexpr bool xs_alias = WHICH == LTDI_RESPONSE_HYBRID;
    double *Xs = xs_alias ? Lr : Xs0;
    double *sa2 = Xs0 + (xs_alias ? 0 : 3 * FAST_TC);   /* behind everything else */
    const double *sa_lfa = sa + (size_t)na_full * ANC;
    const double *sa2_lfa = sa2 + (size_t)na_full * M;
    const int lfa_a0 = p.gen == LTDI_GEN_15 ? 0 : FAST_NA_LFA_GEN;   /* first LFA anchor of this generation */
    const double *tabL = p.tab + (int64_t)ROW_L * p.stride;
    __shared__ __align__(16) double s_hdr[FAST_NA * 4];
    __shared__ uint64_t s_bar;

    /* phase 0: thread 0 issues one TMA bulk copy per staged row (clipped to the rows' allocations), everybody waits
     * on the mbarrier.  What lies before the series is zero-filled; what lies behind it (scratch never written) only
     * reaches margin outputs, which are overwritten with 0. */
    if (tid == 0) {
        mbar_init(&s_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const int64_t g0 = max(y0, (int64_t)0), g1 = min(y0 + yr, p.lds);                  /* full links, even bounds */
    const int nyF = (int)max(g1 - g0, (int64_t)0), nyL = nyF;                             /* the LFA rows cover the same samples */
    const int64_t lr0 = n0 - lroff;                                                      /* first sample of a light-time row */
    const int64_t l0 = max(lr0, (int64_t)0), l1 = min(lr0 + LRW, p.stride);
    const int nl = (int)max(l1 - l0, (int64_t)0);
    if (LR_EXT && (lr0 < 0 || nl < LRW))
        for (int k = tid; k < 6 * LRW; k += FAST_TC_THREADS) {
            const int c = k % LRW;
            if (c < l0 - lr0 || c >= l0 - lr0 + nl) Lr[k] = 0.0;
        }
    if (has_full && (y0 < 0 || nyF < yr))
        for (int k = tid; k < 6 * yr; k += FAST_TC_THREADS) {
            const int c = k % yr;
            if (c < g0 - y0 || c >= g0 - y0 + nyF) yF[k] = 0.0;
        }
    if (has_lfa && (y0 < 0 || nyL < yr))
        for (int k = tid; k < 3 * yr; k += FAST_TC_THREADS) {
            const int c = k % yr;
            if (c < g0 - y0 || c >= g0 - y0 + nyL) dL[k] = 0.0;
        }
    __syncthreads();   /* the barrier is initialised, the zero fill is visible */
    if (tid == 0) {
        const int64_t ystride = p.batch * p.lds;
        const int64_t atile = tile / FAST_TCA_TILES;
        const double *ga = p.anc + atile * (int64_t)(FAST_NA * ANC);
        const double *ga2 = ORD2 ? p.anc2 + atile * (int64_t)(FAST_NA * M) : nullptr;
        mbar_expect_tx(&s_bar, (unsigned)(((has_full ? 6 * nyF + FAST_NA_FULL * (ANC + (ORD2 ? M : 0)) : 0) +
                                           (has_lfa ? 3 * nyL + FAST_NA_LFA_GEN * (ANC + (ORD2 ? M : 0)) : 0) +
                                           NLR * nl + FAST_NA * 4) * sizeof(double)));
#pragma unroll 1
        for (int l = 0; l < NLR; ++l)
            if (nl > 0) bulk_g2s(Lr + l * LRW + (l0 - lr0), tabL + l * p.stride + l0, nl * 8u, &s_bar);
        if (ORD2 && has_full) bulk_g2s(sa2, ga2, FAST_NA_FULL * M * 8u, &s_bar);
        if (ORD2 && has_lfa) bulk_g2s(sa2 + (size_t)na_full * M, ga2 + (FAST_NA_FULL + lfa_a0) * M, FAST_NA_LFA_GEN * M * 8u, &s_bar);
        if (has_full) {
#pragma unroll 1
            for (int l = 0; l < 6; ++l)
                if (nyF > 0) bulk_g2s(yF + l * yr + (g0 - y0), p.yF + b * p.lds + l * ystride + g0, nyF * 8u, &s_bar);
            bulk_g2s(sa, ga, FAST_NA_FULL * ANC * 8u, &s_bar);
        }
        if (has_lfa) {
#pragma unroll 1
            for (int l = 0; l < 3; ++l)
                if (nyL > 0) bulk_g2s(dL + l * yr + (g0 - y0), p.yL + b * p.lds + l * ystride + g0, nyL * 8u, &s_bar);
            bulk_g2s(sa + (size_t)na_full * ANC, ga + (FAST_NA_FULL + lfa_a0) * ANC, FAST_NA_LFA_GEN * ANC * 8u, &s_bar);   /* this generation's six */
        }
        bulk_g2s(s_hdr, p.anc_hdr + atile * (FAST_NA * 4), FAST_NA * 4 * 8u, &s_bar);
    }
    mbar_wait(&s_bar, 0);

    const int ch = tid / FAST_TC_G, g = tid % FAST_TC_G;
    const int i2 = (1 + ch) % 3, i3 = (2 + ch) % 3;
    const int r0 = FAST_TC_R * g;                       /* first of my samples, relative to n0 */
    const int64_t nf = n0 + r0;
    double Xf[FAST_TC_R], Xl[FAST_TC_R];
#pragma unroll
    for (int r = 0; r < FAST_TC_R; ++r) { Xf[r] = 0.0; Xl[r] = 0.0; }

    /* every anchor this channel uses must be valid for the tile (the decision is per channel: no barrier needed) */
    bool ok = true;
    if (has_full && need_full) {
        const int nd = p.gen == LTDI_GEN_20 ? 13 : 6;
        for (int id = 0; id < nd; ++id) ok = ok && anchor_ok<ORD2>(s_hdr[4 * (13 * ch + id) + 3]);
    }
    if (has_lfa && need_lfa)
        ok = ok && anchor_ok<ORD2>(s_hdr[4 * (FAST_NA_FULL + lfa_a0 + 2 * ch) + 3]) &&
             anchor_ok<ORD2>(s_hdr[4 * (FAST_NA_FULL + lfa_a0 + 2 * ch + 1) + 3]);
    const bool nested = LR_EXT && p.nested;

    if (ok) {
        /* one loop over the interpolated terms of this channel: 6 / 14 of Eq. (2.7) / (2.8) on the full links, then
         * the two of (B25) / (B33) on the differentiated LFA links.  Per term: anchor, series offset, and the
         * coefficients of the delay d_n = cP L_-p2 + c2 L_p2 + cU L_p3 + c3 L_-p3 in the light times of the channel's
         * links (a = L_-p2 + L_p2, b = L_p3 + L_-p3, dP = L_-p2, dU = L_p3; LFA: L_p2 and L_p3 only);
         * D = eps_n - eps_c = (d_c - d_n) / dt */
        const double *LP = Lr + (has_full ? (i2 + 3) * LRW : 0) + lroff + r0, *L2p = Lr + i2 * LRW + lroff + r0;
        const double *LU = Lr + i3 * LRW + lroff + r0, *L3m = Lr + (has_full ? (i3 + 3) * LRW : 0) + lroff + r0;
        const bool g20 = p.gen == LTDI_GEN_20;
        const int tm_first = (has_full && need_full) ? 0 : 14;
        const int i0 = (int)(nf - y0);
        const double lfa_hi = p.gen == LTDI_GEN_15 ? 1.0 : 2.0, lfa_lo = p.gen == LTDI_GEN_15 ? 0.5 : 1.5;
        double dn[FAST_TC_R];   /* nested delays: the chain so far (oracle O12) */
#pragma unroll 1
        for (int tm = tm_first; tm < ((has_lfa && need_lfa) ? 16 : 14); ++tm) {
            const bool lt = has_lfa && (!has_full || tm >= 14);
            if (!lt && !g20 && (tm % 7) >= 3) continue;    /* TDI 1.5: the first three terms of either chain */
            const double *anc_t, *anc2_t = nullptr, *xs;
            double cP, c2, cU, c3, dc, sgn = 0.0;
            const double *Lk = nullptr;                     /* nested: the row of the link this term adds to the chain */
            if (!lt) {
                const TermDef td = c_term_def[tm];
                const DelayDef df = c_delay_def[td.delay];
                const int series = td.series == 0 ? i2 : td.series == 1 ? i2 + 3 : td.series == 2 ? i3 + 3 : i3; /* P Q U W */
                const double *hd = s_hdr + 4 * (13 * ch + td.delay);
                dc = hd[0];
                xs = yF + series * yr + i0 - (int)hd[1] - (H - 1);
                anc_t = sa + (13 * ch + td.delay) * ANC;
                if (ORD2) anc2_t = sa2 + (13 * ch + td.delay) * M;
                if (LR_EXT) Lk = Lr + (td.link == 0 ? i3 : td.link == 1 ? i3 + 3 : td.link == 2 ? i2 + 3 : i2) * LRW;
                cP = (double)((df.base == 1) + df.i); c2 = (double)df.i;
                cU = (double)((df.base == 2) + df.j); c3 = (double)df.j;
                sgn = (double)td.sign;
            } else {
                const int id = tm - 14;   /* 0: d/dt y_{p2} at L_p3 + L_p2 / 2 (gen 1.5);  1: d/dt y_{p3} at L_p2 + L_p3 / 2 */
                const double *hd = s_hdr + 4 * (FAST_NA_FULL + lfa_a0 + 2 * ch + id);
                dc = hd[0];
                xs = dL + (id == 0 ? i2 : i3) * yr + i0 - (int)hd[1] - (H - 1);
                anc_t = sa_lfa + (2 * ch + id) * ANC;
                if (ORD2) anc2_t = sa2_lfa + (2 * ch + id) * M;
                cP = 0.0; c3 = 0.0;
                c2 = id == 0 ? lfa_lo : lfa_hi;
                cU = id == 0 ? lfa_hi : lfa_lo;
            }
            double D[FAST_TC_R], Dt = 0.0;   /* second order: D = eps_n - eps_c before the filters, Dt = the thread's own expansion point */
            if (ORD2) {
                if (LR_EXT && nested && !lt) {
                    /* d_j = d_{j-1} + L_cj(t - d_{j-1}); a chain starts at terms 0 and 7 */
                    const bool first = tm == 0 || tm == 7;
#pragma unroll
                    for (int r = 0; r < FAST_TC_R; ++r) {
                        const double prev = first ? 0.0 : dn[r];
                        dn[r] = prev + light_time_at(Lk, lroff + r0 + r, prev, p.dt, p.inv_dt);
                        D[r] = (dc - dn[r]) * p.inv_dt;
                    }
                } else {
#pragma unroll
                    for (int r = 0; r < FAST_TC_R; ++r)   /* the LFA delays have no L_-p2, L_-p3 part (cP = c3 = 0: the same bits) */
                        D[r] = (WHICH == LTDI_RESPONSE_LFA ? fma(-cU, LU[r], fma(-c2, L2p[r], dc))
                                                           : fma(-c3, L3m[r], fma(-cU, LU[r], fma(-c2, L2p[r], fma(-cP, LP[r], dc))))) * p.inv_dt;
                }
                Dt = D[FAST_TC_R / 2];
            }
            double s0[FAST_TC_R], s1[FAST_TC_R];
            term7<M, ORD2>(anc_t, anc2_t, Dt, xs, s0, s1);
#pragma unroll
            for (int r = 0; r < FAST_TC_R; ++r) {
                const double Dr = ORD2 ? D[r] - Dt
                                  : (WHICH == LTDI_RESPONSE_LFA ? fma(-cU, LU[r], fma(-c2, L2p[r], dc))
                                                                : fma(-c3, L3m[r], fma(-cU, LU[r], fma(-c2, L2p[r], fma(-cP, LP[r], dc))))) * p.inv_dt;
                const double v = fma(Dr, s1[r], s0[r]);
                if (!lt) Xf[r] = fma(sgn, v, Xf[r]);
                else {
                    const double L2 = L2p[r], L3 = LU[r];
                    const double pre = p.gen == LTDI_GEN_15 ? 4.0 : 8.0 * (L2 + L3);   /* (B25) / (B33) */
                    if (WHICH == LTDI_RESPONSE_LFA) {
                        /* the LFA instance keeps the running sum in its slot of the exchange region (the thread's own until
                         * the barrier): in registers it was spilled across term7 under the 80-register cap of four CTAs per SM */
                        double *xo = Xs + ch * FAST_TC + r0 + r;
                        *xo = tm == 14 ? (pre * L3) * v : fma(-(pre * L2), v, *xo);
                    } else
                        Xl[r] = fma(tm == 14 ? pre * L3 : -(pre * L2), v, Xl[r]);
                }
            }
        }
        if (has_full && need_full) { /* the two undelayed terms: + Q(t) - W(t) */
            const double *Q = yF + (i2 + 3) * yr + i0, *W = yF + i3 * yr + i0;
#pragma unroll
            for (int r = 0; r < FAST_TC_R; ++r) Xf[r] += Q[r] - W[r];
        }
    } else {
        /* exact per-sample weights */
        if (g == 0) atomicAdd(&d_slow_tiles, 1ULL);
        for (int r = 0; r < FAST_TC_R; ++r) {
            const int64_t n = nf + r;
            if (n >= n1) break;
            double L[6];
            for (int l = 0; l < 6; ++l) L[l] = tabL[l * p.stride + n];
            const int idx = (int)(n - y0);
            if (has_full && need_full) {
                const double *ser[4] = {yF + i2 * yr, yF + (i2 + 3) * yr, yF + (i3 + 3) * yr, yF + i3 * yr};
                const double dP = L[i2 + 3], dU = L[i3], a = L[i2 + 3] + L[i2], bb = L[i3] + L[i3 + 3];
                double x = ser[1][idx] - ser[3][idx];
                double chain = 0.0;
                for (int tm = 0; tm < 14; ++tm) {
                    if (p.gen != LTDI_GEN_20 && (tm % 7) >= 3) continue;
                    const TermDef td = c_term_def[tm];
                    double delay = tdi_delay(td.delay, dP, dU, a, bb);
                    if (LR_EXT && nested) {
                        const double *Lk = Lr + (td.link == 0 ? i3 : td.link == 1 ? i3 + 3 : td.link == 2 ? i2 + 3 : i2) * LRW;
                        const double prev = (tm == 0 || tm == 7) ? 0.0 : chain;
                        chain = prev + light_time_at(Lk, idx, prev, p.dt, p.inv_dt);
                        delay = chain;
                    }
                    x += (double)td.sign * slow_delayed<M>(ser[td.series], yr, idx, delay, p.dt, p.inv_dt);
                }
                Xf[r] = x;
            }
            if (has_lfa && need_lfa) {
                const double L2 = L[i2], L3 = L[i3];
                const double v2 = slow_delayed<M>(dL + i2 * yr, yr, idx, lfa_delay(p.gen, 0, L2, L3), p.dt, p.inv_dt);
                const double v3 = slow_delayed<M>(dL + i3 * yr, yr, idx, lfa_delay(p.gen, 1, L2, L3), p.dt, p.inv_dt);
                Xl[r] = (p.gen == LTDI_GEN_15 ? 4.0 : 8.0 * (L2 + L3)) * (L3 * v2 - L2 * v3);
            }
        }
    }
    if (xs_alias) __syncthreads();   /* every thread is done with the light times: Lr becomes X, Y, Z */

    /* exchange through shared memory: rows 0..2 = X, Y, Z (hybrid: of the full response, rows 3..5 = of the LFA) */
#pragma unroll
    for (int r = 0; r < FAST_TC_R; ++r) {
        if (WHICH == LTDI_RESPONSE_LFA) {
            if (!ok) Xs[ch * FAST_TC + r0 + r] = Xl[r];   /* fast path: already there */
        } else Xs[ch * FAST_TC + r0 + r] = Xf[r];
        if (WHICH == LTDI_RESPONSE_HYBRID) Xs[(3 + ch) * FAST_TC + r0 + r] = Xl[r];
    }
    __syncthreads();

    /* blend (4.6), margins, A, E, T (2.9): one sample per thread and pass, the taper evaluated once per sample */
    const double is2 = 0.70710678118654752440, is6 = 0.40824829046386301637, is3 = 0.57735026918962576451;
    const int64_t src_off = b * p.ld;
    const int64_t ystride = p.batch * p.lds;
#pragma unroll 1
    for (int i = tid; i < FAST_TC; i += FAST_TC_THREADS) {
        const int64_t n = n0 + i;
        if (n >= n1) break;
        double X = Xs[i], Y = Xs[FAST_TC + i], Z = Xs[2 * FAST_TC + i];
        double wa = 1.0, wb = 1.0;
        if (WHICH == LTDI_RESPONSE_HYBRID) {
            hybrid_weights_fast(hy, p.t0 + (double)n * p.dt, wa, wb);
            const bool use_l = need_lfa && wa != 0.0, use_f = need_full && wb != 0.0;
            const double xl = Xs[3 * FAST_TC + i], yl = Xs[4 * FAST_TC + i], zl = Xs[5 * FAST_TC + i];
            const double x0 = use_l ? wa * xl : 0.0, y0b = use_l ? wa * yl : 0.0, z0 = use_l ? wa * zl : 0.0;
            X = use_f ? fma(wb, X, x0) : x0;
            Y = use_f ? fma(wb, Y, y0b) : y0b;
            Z = use_f ? fma(wb, Z, z0) : z0;
        } else if (WHICH == LTDI_RESPONSE_LFA && hybrid_mode) {    /* a block before the window: w_Full = 0 */
            hybrid_weights_fast(hy, p.t0 + (double)n * p.dt, wa, wb);
            X = wa != 0.0 ? wa * X : 0.0;
            Y = wa != 0.0 ? wa * Y : 0.0;
            Z = wa != 0.0 ? wa * Z : 0.0;
        } else if (WHICH == LTDI_RESPONSE_FULL && hybrid_mode) {   /* a tile after the window: w_LFA = 0 */
            hybrid_weights_fast(hy, p.t0 + (double)n * p.dt, wa, wb);
            X = wb != 0.0 ? wb * X : 0.0;
            Y = wb != 0.0 ? wb * Y : 0.0;
            Z = wb != 0.0 ? wb * Z : 0.0;
        }
        if (!(n >= p.lo && n < p.n - p.hi)) { X = 0.0; Y = 0.0; Z = 0.0; }
        p.A[src_off + n] = (Z - X) * is2;                 /* (2.9a) */
        p.E[src_off + n] = (X - 2.0 * Y + Z) * is6;       /* (2.9b) */
        p.T[src_off + n] = (X + Y + Z) * is3;             /* (2.9c) */
        if (p.XYZ) {
            p.XYZ[((int64_t)0 * p.batch_all + p.b0 + b) * p.ld + n] = X;
            p.XYZ[((int64_t)1 * p.batch_all + p.b0 + b) * p.ld + n] = Y;
            p.XYZ[((int64_t)2 * p.batch_all + p.b0 + b) * p.ld + n] = Z;
        }
        if (p.Y) {
            /* optional link output: the LFA links come back from the scratch series (their shared copy is gone) */
            const int iy = (int)(n - y0);
            const double *gl = p.yLraw + b * p.lds + n;   /* the LFA links themselves (written because d_y was asked for) */
#pragma unroll 1
            for (int l = 0; l < 6; ++l) {
                double v = 0.0;
                if (WHICH == LTDI_RESPONSE_FULL) {
                    if (!hybrid_mode) v = yF[l * yr + iy];
                    else if (wb != 0.0 && n >= p.m1 + w && n < p.n - p.m1 - w) v = wb * yF[l * yr + iy];          /* (4.5) */
                }
                else if (WHICH == LTDI_RESPONSE_LFA) {
                    if (!hybrid_mode) v = l < 3 ? gl[l * ystride] : 0.0;
                    else if (l < 3 && wa != 0.0 && n >= p.m1 + w && n < p.n - p.m1 - w) v = wa * gl[l * ystride]; /* (4.5) */
                }
                else if (n >= p.m1 + w && n < p.n - p.m1 - w) { /* (4.5) */
                    if (need_lfa && l < 3 && wa != 0.0) v = wa * gl[l * ystride];
                    if (need_full && wb != 0.0) v = fma(wb, yF[l * yr + iy], v);
                }
                p.Y[((int64_t)l * p.batch_all + p.b0 + b) * p.ld + n] = v;
            }
        }
    }
}

/* dynamic shared memory of tdi_kernel<M> in bytes (mirrors the carve-up above) */
template <int M>
static inline size_t tdi_smem_bytes(int which, int64_t m2, int64_t w, bool ord2)
{
    const bool has_full = which != LTDI_RESPONSE_LFA, has_lfa = which != LTDI_RESPONSE_FULL;
    const size_t yr = (size_t)tdi_yr<M>(tdi_tc(which), m2);
    const size_t na = (size_t)((has_full ? FAST_NA_FULL : 0) + (has_lfa ? FAST_NA_LFA : 0));
    size_t dbl = na * FAST_ANC_DOUBLES(M);
    dbl += (has_full ? 6 * yr : 0) + (has_lfa ? 3 * yr : 0);
    dbl += (size_t)(has_full ? 6 : 3) * ((ord2 && which == LTDI_RESPONSE_FULL) ? yr : (size_t)tdi_tc(which));
    dbl += which == LTDI_RESPONSE_HYBRID ? 0 : (size_t)3 * tdi_tc(which);   /* X, Y, Z exchange */
    dbl += ord2 ? na * M : 0;                                                /* second derivative of the weights */
    return dbl * sizeof(double);
}
