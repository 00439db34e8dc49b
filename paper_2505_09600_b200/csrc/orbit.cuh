// orbit.cuh -- S0: orbit / delay kernel (first-order Keplerian orbits, G5-G7).
//
// One thread per time sample writes the 24 table rows: spacecraft positions R_i(t_n) [m],
// link unit vectors n_l(t_n) for l = +1,+2,+3 (sender -> receiver; n_-l = -n_l) and the
// six light travel times L_l(t_n) [s].  HBM-bound: 192 B written per sample, nothing read
// (analytic modes) or 120 B read (tables mode).
#pragma once
#include "common.cuh"

struct OrbitKernelParams {
    double t0, dt;
    int64_t n, stride;
    double arm_m, R_m, omega, alpha0, rot0;
    double sb[3], cb[3]; /* sin, cos of beta_i */
    int mode;
    const double *R_in; /* tables mode: [3][3][n] */
    const double *L_in; /* tables mode: [6][n] */
    double *tab;
};

__global__ void __launch_bounds__(256) orbit_delay_kernel(OrbitKernelParams p)
{
    const int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= p.n) return;
    double R[3][3], V[3][3];
    if (p.mode == LTDI_ORBIT_TABLES) {
#pragma unroll
        for (int i = 0; i < 9; ++i) {
            R[i / 3][i % 3] = p.R_in[(int64_t)i * p.n + n];
            V[i / 3][i % 3] = 0.0;
        }
    } else {
        // alpha(t) = Omega t + alpha0; spacecraft i: beta_i = 2 pi (i-1)/3 + rot0.  Positions to first
        // order in the eccentricity e = L / (2 sqrt(3) R): a rigid triangle of side L, cartwheeling at 1 AU.
        const double t = p.t0 + (double)n * p.dt;
        const double alpha = p.omega * t + p.alpha0;
        const double ecc = p.arm_m / (2.0 * sqrt(3.0) * p.R_m);
        const double eR = ecc * p.R_m;
        double sa, ca;
        sincos(alpha, &sa, &ca);
        /* one sincos per sample: the angles 2 alpha - beta_i and alpha - beta_i by the addition theorems
         * (a few ulp of 1 on terms that are e R = 7e8 m: 1e-6 m, far inside the table tolerance) */
        const double s2a = 2.0 * sa * ca, c2a = (ca - sa) * (ca + sa);
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            const double sb = p.sb[i], cb = p.cb[i];
            const double s2 = s2a * cb - c2a * sb, c2 = c2a * cb + s2a * sb;
            const double s1 = sa * cb - ca * sb, c1 = ca * cb + sa * sb;
            R[i][0] = p.R_m * ca + 0.5 * eR * (c2 - 3.0 * cb);
            R[i][1] = p.R_m * sa + 0.5 * eR * (s2 - 3.0 * sb);
            R[i][2] = -sqrt(3.0) * eR * c1;
            V[i][0] = -p.R_m * p.omega * sa - eR * p.omega * s2;
            V[i][1] = p.R_m * p.omega * ca + eR * p.omega * c2;
            V[i][2] = sqrt(3.0) * eR * p.omega * s1;
        }
    }
    double *out = p.tab + n;
#pragma unroll
    for (int i = 0; i < 9; ++i) out[(int64_t)(ROW_R + i) * p.stride] = R[i / 3][i % 3];
    const double inv_c = 1.0 / LTDI_C_LIGHT;
#pragma unroll
    for (int l = 0; l < 3; ++l) {
        const int s = link_sender(l), r = link_receiver(l);
        const double dx = R[r][0] - R[s][0], dy = R[r][1] - R[s][1], dz = R[r][2] - R[s][2];
        const double len = sqrt(dx * dx + dy * dy + dz * dz);
        const double nx = dx / len, ny = dy / len, nz = dz / len;
        out[(int64_t)(ROW_N + 3 * l + 0) * p.stride] = nx;
        out[(int64_t)(ROW_N + 3 * l + 1) * p.stride] = ny;
        out[(int64_t)(ROW_N + 3 * l + 2) * p.stride] = nz;
        double Lp, Lm; /* link +l (s -> r) and -l (r -> s) */
        if (p.mode == LTDI_ORBIT_STATIC_EQUALARM) {
            Lp = Lm = p.arm_m / LTDI_C_LIGHT;
        } else if (p.mode == LTDI_ORBIT_KEPLERIAN) {
            // first-order light time |d|/c (1 + n.V_sender / c): L_l != L_-l (Eq. B22)
            const double nvs = nx * V[s][0] + ny * V[s][1] + nz * V[s][2];
            const double nvr = -(nx * V[r][0] + ny * V[r][1] + nz * V[r][2]);
            Lp = (len / LTDI_C_LIGHT) * (1.0 + nvs / LTDI_C_LIGHT);
            Lm = (len / LTDI_C_LIGHT) * (1.0 + nvr / LTDI_C_LIGHT);
        } else {
            Lp = p.L_in[(int64_t)l * p.n + n];
            Lm = p.L_in[(int64_t)(l + 3) * p.n + n];
        }
        out[(int64_t)(ROW_L + l) * p.stride] = Lp;
        out[(int64_t)(ROW_L + 3 + l) * p.stride] = Lm;
    }
    (void)inv_c;
}
