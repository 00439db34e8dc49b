"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Every test here checks oracle/ against something OTHER than itself: a closed form, an
invariant, a library routine (numpy / scipy) on a special case, a value printed in the
paper (tests/golden/paper_constants.txt) or brute force on tiny inputs.
"""
import math
import os

import numpy as np
import pytest
from scipy.interpolate import BarycentricInterpolator

import workloads as W

C = 299792458.0
HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    out = {}
    with open(os.path.join(HERE, "golden", "paper_constants.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            name, val, tol = line.split()[:3]
            out[name] = (float(val), float(tol))
    return out


# ------------------------------------------------------------------ O4 Lagrange
@pytest.mark.parametrize("order", [1, 3, 9, 31])
def test_lagrange_exact_on_polynomials(orc80, order):
    """north-star check 1: a degree <= p polynomial is reproduced at any fractional delay"""
    rng = np.random.default_rng(10 + order)
    n, dt = 200, 2.5
    x = np.arange(n, dtype=np.float64)
    for deg in {0, 1, order // 2, order}:
        coef = rng.normal(size=deg + 1)
        # polynomial in the centred, scaled variable so that values stay O(1)
        poly = np.polynomial.Polynomial(coef, domain=[80, 120])
        series = poly(x)
        for d in rng.uniform(-10.0, 10.0, size=6) * dt:
            n0 = 100
            got = orc80.interp(series, n0, d, dt, order)
            want = poly(n0 - d / dt)
            assert abs(got - want) <= 2e-13 * max(1.0, np.abs(series[80:120]).max()), (order, deg, d)


@pytest.mark.parametrize("order", [1, 9, 31])
def test_lagrange_weights_sum_and_library(orc80, order):
    """weights sum to 1 and equal scipy's barycentric Lagrange basis on the same nodes"""
    M = order + 1
    nodes = np.arange(-(M // 2 - 1), M // 2 + 1, dtype=np.float64)
    for eps in [0.0, 0.125, 0.5, 0.73, 0.999]:
        w = orc80.lagrange_weights(eps, order)
        assert abs(w.sum() - 1.0) < 1e-13
        basis = np.array([BarycentricInterpolator(nodes, np.eye(M)[k])(eps) for k in range(M)])
        assert np.allclose(w, basis, rtol=0, atol=1e-12)
    w0 = orc80.lagrange_weights(0.0, order)
    assert w0[M // 2 - 1] == 1.0 and np.count_nonzero(w0) == 1


def test_integer_delay_is_pure_shift(orc80):
    rng = np.random.default_rng(3)
    x = rng.normal(size=300)
    dt = 5.0
    for q in (-7, 0, 1, 12):
        assert orc80.interp(x, 150, q * dt, dt, 31) == x[150 - q]  # bitwise


def test_order1_is_linear_interpolation(orc80):
    rng = np.random.default_rng(4)
    x = rng.normal(size=100)
    dt = 10.0
    for d in (3.3, 17.0, -4.2, 0.4):
        want = np.interp(50 - d / dt, np.arange(100.0), x)
        assert abs(orc80.interp(x, 50, d, dt, 1) - want) < 1e-14


def test_interp_matches_library_interpolant_on_random_data(orc80):
    """brute force: the value equals the unique degree-p polynomial through the p+1 centred taps"""
    rng = np.random.default_rng(5)
    x = rng.normal(size=120)
    dt, order, n0 = 5.0, 9, 60
    for d in (12.3, -8.7, 0.1):
        s = d / dt
        q = math.ceil(s)
        j = n0 - q
        taps = np.arange(j - 4, j + 6)
        want = BarycentricInterpolator(taps.astype(float), x[taps])(n0 - s)
        assert abs(orc80.interp(x, n0, d, dt, order) - want) < 1e-12


# ------------------------------------------------------------------ O8 stencils
@pytest.mark.parametrize("fd_order,which,deg", [(2, 1, 2), (2, 2, 3), (4, 1, 4), (4, 2, 5)])
def test_stencils_exact_on_polynomials(orc80, fd_order, which, deg):
    dt = 0.5
    i = np.arange(41, dtype=np.float64)
    tt = (i - 20) * dt
    rng = np.random.default_rng(6)
    p = np.polynomial.Polynomial(rng.normal(size=deg + 1))
    got = orc80.stencil(p(tt), dt, fd_order, which)
    want = p.deriv(which)(tt)
    w = fd_order // 2
    assert np.allclose(got[w:-w], want[w:-w], rtol=0, atol=1e-9 * np.abs(p(tt)).max())
    # and NOT exact one degree higher (the stencil has the stated order, not more)
    p2 = np.polynomial.Polynomial(np.r_[np.zeros(deg + 1 + (deg + which) % 2), 1.0])
    got2 = orc80.stencil(p2(tt), dt, fd_order, which)
    assert np.abs(got2[w:-w] - p2.deriv(which)(tt)[w:-w]).max() > 1e-6


# ------------------------------------------------------------------ O2 source frame
def test_source_frame_is_right_handed_orthonormal_triad(orc80):
    """P:79 'orthonormal triad'; k = -e_r, u = -e_phi, v = -e_theta from the spherical basis"""
    rng = np.random.default_rng(7)
    for _ in range(10):
        beta, lam, psi = math.asin(rng.uniform(-1, 1)), rng.uniform(0, 2 * math.pi), rng.uniform(0, math.pi)
        f = orc80.source_frame(beta, lam, psi)
        k, u, v = f["k"], f["u"], f["v"]
        G = np.array([k, u, v]) @ np.array([k, u, v]).T
        assert np.allclose(G, np.eye(3), atol=1e-15)
        assert np.allclose(np.cross(u, v), k, atol=1e-15)
        theta, phi = math.pi / 2 - beta, lam
        e_r = np.array([math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), math.cos(theta)])
        e_th = np.array([math.cos(theta) * math.cos(phi), math.cos(theta) * math.sin(phi), -math.sin(theta)])
        e_ph = np.array([-math.sin(phi), math.cos(phi), 0.0])
        assert np.allclose(k, -e_r, atol=1e-15) and np.allclose(u, -e_ph, atol=1e-15)
        assert np.allclose(v, -e_th, atol=1e-15)
        assert abs(f["c2"] - math.cos(2 * psi)) < 1e-15 and abs(f["s2"] - math.sin(2 * psi)) < 1e-15


# ------------------------------------------------------------------ O1 orbits
def test_orbit_rigid_triangle_and_printed_constants(orc80):
    g = golden()
    n = 2000
    orbit = W.orbit_desc(n, W.YEAR_S / n, W.ORBIT_KEPLERIAN, alpha0=0.3, rot0=0.7)
    R, nh, L = orc80.orbit_tables(orbit)
    Rm, arm = orbit["R_m"], orbit["arm_m"]
    assert abs(arm - g["arm_length_m"][0]) == 0
    assert abs(Rm / g["R_m"][0] - 1) < g["R_m"][1]
    assert abs(2 * math.pi / orbit["period_s"] / g["Omega_rad_s"][0] - 1) < g["Omega_rad_s"][1]
    assert abs(arm / C / g["light_time_s"][0] - 1) < g["light_time_s"][1]
    assert abs(C / (2 * math.pi * arm) / g["f_c_over_2piL_hz"][0] - 1) < g["f_c_over_2piL_hz"][1]
    assert abs(C / arm / g["f_c_over_L_hz"][0] - 1) < g["f_c_over_L_hz"][1]
    assert abs(C / (2 * math.pi * Rm) / g["f_c_over_2piR_hz"][0] - 1) < g["f_c_over_2piR_hz"][1]
    assert abs(Rm * 2 * math.pi / orbit["period_s"] / C / g["R_Omega_over_c"][0] - 1) < g["R_Omega_over_c"][1]
    e = arm / (2 * math.sqrt(3) * Rm)
    # rigid equilateral triangle of side L (config 1's "rigid rotating triangle")
    for (a, b) in ((0, 1), (1, 2), (2, 0)):
        side = np.linalg.norm(R[a] - R[b], axis=0)
        assert np.abs(side / arm - 1).max() < 5e-14
    # heliocentric distance R (1 +- e) to first order in e
    for i in range(3):
        r = np.linalg.norm(R[i], axis=0)
        assert abs(r.max() / Rm - 1 - e) < 3 * e * e and abs(r.min() / Rm - 1 + e) < 3 * e * e
    # the centre moves on the circle of radius R in the ecliptic with phase alpha
    R0 = R.mean(axis=0)
    t = orbit["t0"] + orbit["dt"] * np.arange(n)
    alpha = 2 * math.pi * t / orbit["period_s"] + orbit["alpha0"]
    assert np.abs(R0 - Rm * np.array([np.cos(alpha), np.sin(alpha), 0 * alpha])).max() < 1e-3  # metres
    # triangle plane inclined by 60 degrees to the ecliptic
    normal = np.cross((R[1] - R[0]).T, (R[2] - R[0]).T)
    normal /= np.linalg.norm(normal, axis=1)[:, None]
    assert np.abs(np.abs(normal[:, 2]) - 0.5).max() < 2 * e
    # unit vectors: sender -> receiver, n_-l = -n_l ; link +1 is 3->2
    assert np.allclose(nh[0], (R[1] - R[2]) / arm, atol=1e-13)
    assert np.allclose(nh[1], (R[2] - R[0]) / arm, atol=1e-13)
    assert np.allclose(nh[2], (R[0] - R[1]) / arm, atol=1e-13)
    assert np.allclose(nh[3:], -nh[:3], atol=1e-15)
    # Eq. (B22): L_l - L_-l = 2 (R Omega L / c) sin(Omega t - delta_|l|) / c  -> amplitude and period
    Om = 2 * math.pi / orbit["period_s"]
    amp = 2 * (Rm * Om / C) * (arm / C)
    for l in range(3):
        diff = L[l] - L[l + 3]
        assert abs(np.abs(diff).max() / amp - 1) < 0.01
        # pure sinusoid at the orbital frequency: projects entirely on cos/sin(Omega t)
        cs = np.array([np.cos(Om * t), np.sin(Om * t)])
        coef = 2 * cs @ diff / n
        assert abs(np.hypot(*coef) / amp - 1) < 0.01
        assert np.abs(diff - coef @ cs).max() < 0.01 * amp
        # mean light time is L/c (no O(e L) flexing in the first-order model)
        assert abs((L[l] + L[l + 3]).mean() / 2 / (arm / C) - 1) < 1e-6
    # the three |l| are 120 degrees apart in phase
    ph = [np.angle(np.exp(-1j * Om * t) @ (L[l] - L[l + 3])) for l in range(3)]
    d01 = (ph[1] - ph[0]) % (2 * math.pi)
    d12 = (ph[2] - ph[1]) % (2 * math.pi)
    assert abs(d01 - d12) < 1e-3 and abs(abs(d01 if d01 < math.pi else d01 - 2 * math.pi) - 2 * math.pi / 3) < 1e-3


def test_static_mode_has_constant_equal_delays(orc80):
    orbit = W.orbit_desc(50, 1000.0, W.ORBIT_STATIC_EQUALARM)
    _, _, L = orc80.orbit_tables(orbit)
    assert np.all(L == orbit["arm_m"] / C)


def test_light_time_is_first_order_retarded_distance(orc80):
    """L_l solves c T = |R_r(t) - R_s(t - T)| to first order in v/c (reading G6): residual O((v/c)^2)"""
    n = 64
    orbit = W.orbit_desc(n, 1.0e5, W.ORBIT_KEPLERIAN)
    R, _, L = orc80.orbit_tables(orbit)
    # sender position a light time earlier, from a fine table around each sample
    for l, (s, r) in enumerate([(2, 1), (0, 2), (1, 0), (1, 2), (2, 0), (0, 1)]):
        for n0 in (5, 30, 60):
            T = L[l, n0]
            fine = W.orbit_desc(3, T, W.ORBIT_KEPLERIAN, t0=orbit["t0"] + n0 * orbit["dt"] - T)
            Rf, _, _ = orc80.orbit_tables(fine)
            dist = np.linalg.norm(R[r][:, n0] - Rf[s][:, 0])
            assert abs(dist / C - T) < 5e-8 * T  # (v/c)^2 ~ 1e-8


# ------------------------------------------------------------------ helpers for closed forms
def tensor_H(beta, lam, psi, nvec, a_plus, a_cross):
    """n^T h n for h = a+ e+' + ax ex' with the polarisation basis rotated by psi (definition of
    Eqs. 2.2-2.4 in tensor form, independent of the oracle's xi / F algebra)."""
    theta, phi = math.pi / 2 - beta, lam
    e_th = np.array([math.cos(theta) * math.cos(phi), math.cos(theta) * math.sin(phi), -math.sin(theta)])
    e_ph = np.array([-math.sin(phi), math.cos(phi), 0.0])
    u, v = -e_ph, -e_th
    p = u * math.cos(psi) + v * math.sin(psi)
    q = -u * math.sin(psi) + v * math.cos(psi)
    eplus = np.outer(p, p) - np.outer(q, q)
    ecross = np.outer(p, q) + np.outer(q, p)
    return nvec @ (a_plus * eplus + a_cross * ecross) @ nvec


LINKS = [(2, 1), (0, 2), (1, 0), (1, 2), (2, 0), (0, 1)]  # (sender, receiver) for +1,+2,+3,-1,-2,-3


def closed_form(orbit_snapshot_R, Lsec, src, w, ap, ac):
    """complex amplitudes of y_l (6) and X,Y,Z for gen 1.5 and 2.0 on a frozen constellation for
    h+ = Re[ap e^{iwt}], hx = Re[ac e^{iwt}]  (delay D_x -> factor e^{-iwx})"""
    beta, lam, psi = src
    k = -np.array([math.cos(beta) * math.cos(lam), math.cos(beta) * math.sin(lam), math.sin(beta)])
    R = orbit_snapshot_R
    Y = np.zeros(6, dtype=complex)
    for l, (s, r) in enumerate(LINKS):
        d = R[r] - R[s]
        nv = d / np.linalg.norm(d)
        Hc = tensor_H(beta, lam, psi, nv, ap, ac)
        ds = Lsec[l] + k @ R[s] / C
        dr = k @ R[r] / C
        Y[l] = Hc * (np.exp(-1j * w * ds) - np.exp(-1j * w * dr)) / (2 * (1 - k @ nv))
    out = {"y": Y}
    idx = lambda lab: lab - 1 if lab > 0 else 2 - lab
    D = lambda x: np.exp(-1j * w * x)
    X15, X20 = [], []
    for ch in range(3):
        p2 = (2 + ch - 1) % 3 + 1
        p3 = (3 + ch - 1) % 3 + 1
        Lp2, Lm2, Lp3, Lm3 = Lsec[idx(p2)], Lsec[idx(-p2)], Lsec[idx(p3)], Lsec[idx(-p3)]
        a, b = Lm2 + Lp2, Lp3 + Lm3
        P, Q, U, Wl = Y[idx(p2)], Y[idx(-p2)], Y[idx(-p3)], Y[idx(p3)]
        x15 = (1 - D(b)) * (D(Lm2) * P + Q) - (1 - D(a)) * (D(Lp3) * U + Wl)
        X15.append(x15)
        X20.append((1 - D(a + b)) * x15)
    out["X15"], out["X20"] = np.array(X15), np.array(X20)
    return out


def fit_complex_amplitude(series, t, w, lo, hi):
    """least-squares complex amplitude Z of series ~ Re[Z e^{iwt}] on [lo, hi)"""
    tt = t[lo:hi]
    Amat = np.stack([np.cos(w * tt), -np.sin(w * tt)], axis=1)
    sol, *_ = np.linalg.lstsq(Amat, series[lo:hi], rcond=None)
    resid = series[lo:hi] - Amat @ sol
    return sol[0] + 1j * sol[1], np.linalg.norm(resid) / max(np.linalg.norm(series[lo:hi]), 1e-300)


def frozen_orbit(orc, n, dt, distinct_L=True):
    snap = W.orbit_desc(1, 1.0, W.ORBIT_KEPLERIAN, t0=0.37 * W.YEAR_S, rot0=0.4)
    R, _, L = orc.orbit_tables(snap)
    R0, L0 = R[:, :, 0], L[:, 0].copy()
    if distinct_L:  # six different light times exercise the link bookkeeping of Eqs. (2.7), (2.8)
        L0 = L0 + np.array([0.00, 0.11, -0.07, 0.05, -0.13, 0.09])
    return W.frozen_tables(W.orbit_desc(n, dt), R0, L0), R0, L0


# ------------------------------------------------------------------ O5-O7 full response
def test_constant_strain_gives_zero_response(orc80):
    """north-star check 2"""
    n, dt = 1500, 5.0
    orbit = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN)
    hp, hc = np.full((1, n), 1.0), np.full((1, n), -0.3)
    src = [[0.4, 1.3, 0.9]]
    for gen in (15, 20):
        r = orc80.response_full(orbit, hp, hc, src, gen, 31)
        assert np.abs(r["y"]).max() < 5e-18 and np.abs(r["XYZ"]).max() < 2e-17


@pytest.mark.parametrize("f_hz", [1.0e-3, 5.0e-3])
def test_full_response_matches_plane_wave_closed_form(orc80, f_hz):
    """north-star check 4: frozen constellation + monochromatic wave -> closed-form transfer
    (the Fourier-domain form of Eqs. 2.5-2.8; |Y_l| is Eq. C3)."""
    n, dt, order = 1400, 5.0, 31
    orbit, R0, L0 = frozen_orbit(orc80, n, dt)
    w = 2 * math.pi * f_hz
    ap, ac = 1.0 * np.exp(0.3j), 0.7 * np.exp(1.1j)
    hp, hc = W.monochromatic(n, dt, f_hz, 1.0, 0.7, 0.3, 1.1)
    src = (0.45, 2.1, 0.8)
    cf = closed_form(R0, L0, src, w, ap, ac)
    t = dt * np.arange(n)
    for gen, key in ((15, "X15"), (20, "X20")):
        r = orc80.response_full(orbit, hp[None], hc[None], [src], gen, order)
        lo, hi = orc80.margins(orbit, gen, order)
        for l in range(6):
            z, res = fit_complex_amplitude(r["y"][l, 0], t, w, lo, n - hi)
            assert res < 1e-10 and abs(z - cf["y"][l]) < 2e-11 * abs(cf["y"][l]), (l, z, cf["y"][l])
        for ch in range(3):
            z, res = fit_complex_amplitude(r["XYZ"][ch, 0], t, w, lo, n - hi)
            assert res < 1e-9 and abs(z - cf[key][ch]) < 5e-10 * abs(cf[key][ch]), (gen, ch)
        X, Y, Z = r["XYZ"][:, 0]
        assert np.allclose(r["A"][0], (Z - X) / math.sqrt(2), rtol=0, atol=1e-15 * np.abs(X).max())
        assert np.allclose(r["E"][0], (X - 2 * Y + Z) / math.sqrt(6), rtol=0, atol=1e-15 * np.abs(X).max())
        assert np.allclose(r["T"][0], (X + Y + Z) / math.sqrt(3), rtol=0, atol=1e-15 * np.abs(X).max())


def test_link_transfer_modulus_is_sinc_of_eq_C3(orc80):
    """|Y_l| = |H_l| (w L / 2c) |sinc[(w L / 2c)(1 - k.n)]| when L_l n_l = R_r - R_s  (Eq. C3)"""
    n, dt, order, f_hz = 1200, 5.0, 31, 3.0e-3
    snap = W.orbit_desc(1, 1.0, W.ORBIT_KEPLERIAN, t0=0.1 * W.YEAR_S)
    R, _, _ = orc80.orbit_tables(snap)
    R0 = R[:, :, 0]
    L0 = np.array([np.linalg.norm(R0[r] - R0[s]) / C for s, r in LINKS])
    orbit = W.frozen_tables(W.orbit_desc(n, dt), R0, L0)
    hp, hc = W.monochromatic(n, dt, f_hz, 1.0, 0.0, 0.0, 0.0)
    src = (-0.3, 4.0, 0.2)
    r = orc80.response_full(orbit, hp[None], hc[None], [src], 15, order)
    lo, hi = orc80.margins(orbit, 15, order)
    w = 2 * math.pi * f_hz
    t = dt * np.arange(n)
    k = -np.array([math.cos(src[0]) * math.cos(src[1]), math.cos(src[0]) * math.sin(src[1]), math.sin(src[0])])
    for l, (s, rr) in enumerate(LINKS):
        nv = (R0[rr] - R0[s]) / np.linalg.norm(R0[rr] - R0[s])
        x = 0.5 * w * L0[l] * (1 - k @ nv)
        want = abs(tensor_H(*src, nv, 1.0, 0.0)) * 0.5 * w * L0[l] * abs(math.sin(x) / x)
        z, _ = fit_complex_amplitude(r["y"][l, 0], t, w, lo, n - hi)
        assert abs(abs(z) - want) < 1e-10 * want


def test_tdi20_is_tdi15_minus_shifted_tdi15_for_static_equal_arms(orc80):
    """north-star check 3 (operator form): with dt = L/c all delays are integer shifts and
    X_2.0[n] = X_1.5[n] - X_1.5[n - 4]"""
    n = 1200
    dt = W.ARM_M / C
    orbit = W.orbit_desc(n, dt, W.ORBIT_STATIC_EQUALARM)
    rng = np.random.default_rng(11)
    t = dt * np.arange(n)
    hp = np.cos(2 * math.pi * 2e-3 * t) + 0.1 * rng.normal(size=n)
    hc = np.sin(2 * math.pi * 3e-3 * t)
    src = [(0.2, 0.5, 1.0)]
    r15 = orc80.response_full(orbit, hp[None], hc[None], src, 15, 31)
    r20 = orc80.response_full(orbit, hp[None], hc[None], src, 20, 31)
    lo, hi = orc80.margins(orbit, 20, 31)
    for ch in range(3):
        x15, x20 = r15["XYZ"][ch, 0], r20["XYZ"][ch, 0]
        lhs = x20[lo + 4:n - hi]
        rhs = x15[lo + 4:n - hi] - x15[lo:n - hi - 4]
        assert np.abs(lhs - rhs).max() < 1e-15 * np.abs(x15).max()


def test_low_frequency_relation_between_generations(orc80):
    """Eq. (3.7): X_2.0(t) -> (4L/c) dX_1.5/dt (t - 2L/c), relative error ~ (w 4L/c)^2 / 24"""
    n, dt = 4000, 5.0
    Ls = W.ARM_M / C
    _, R0, _ = frozen_orbit(orc80, 1, dt)
    orbit = W.frozen_tables(W.orbit_desc(n, dt), R0, np.full(6, Ls))  # frozen, equal constant arms
    errs = []
    for f_hz in (4e-4, 2e-4):
        hp, hc = W.monochromatic(n, dt, f_hz)
        src = [(0.2, 0.5, 1.0)]
        r15 = orc80.response_full(orbit, hp[None], hc[None], src, 15, 31)
        r20 = orc80.response_full(orbit, hp[None], hc[None], src, 20, 31)
        lo, hi = orc80.margins(orbit, 20, 31)
        w = 2 * math.pi * f_hz
        t = dt * np.arange(n)
        z15, _ = fit_complex_amplitude(r15["XYZ"][0, 0], t, w, lo, n - hi)
        z20, _ = fit_complex_amplitude(r20["XYZ"][0, 0], t, w, lo, n - hi)
        pred = 4 * Ls * (1j * w) * np.exp(-1j * w * 2 * Ls) * z15
        errs.append(abs(z20 - pred) / abs(z20))
        assert errs[-1] < 1.5 * (w * 4 * Ls) ** 2 / 24
    assert 3.0 < errs[0] / errs[1] < 5.0  # falls as f^2


def test_linearity_and_polarisation_invariances(orc80):
    """linear in h; psi -> psi + pi leaves the response unchanged, psi -> psi + pi/2 flips it"""
    n, dt = 1300, 5.0
    orbit = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN, alpha0=1.0)
    rng = np.random.default_rng(12)
    t = dt * np.arange(n)
    h1 = np.cos(2 * math.pi * 3e-3 * t) * (1 + 1e-4 * t)
    h2 = np.sin(2 * math.pi * 5e-3 * t)
    g1, g2 = rng.normal(size=n), rng.normal(size=n)
    src = (0.7, 3.3, 0.4)
    run = lambda hp, hc, s: orc80.response_full(orbit, hp[None], hc[None], [s], 20, 31)["XYZ"][:, 0]
    a = run(h1, h2, src)
    b = run(g1, g2, src)
    c = run(2 * h1 - 3 * g1, 2 * h2 - 3 * g2, src)
    assert np.abs(c - (2 * a - 3 * b)).max() < 1e-13 * np.abs(c).max()
    a_pi = run(h1, h2, (src[0], src[1], src[2] + math.pi))
    a_half = run(h1, h2, (src[0], src[1], src[2] + math.pi / 2))
    assert np.abs(a_pi - a).max() < 1e-13 * np.abs(a).max()
    assert np.abs(a_half + a).max() < 1e-13 * np.abs(a).max()


def test_full_response_brute_force_single_sample(orc80):
    """tiny brute force: one X sample rebuilt from Eqs. (2.5)-(2.7) with scipy's Lagrange
    interpolant doing every interpolation and the (separately pinned) orbit tables"""
    n, dt, order = 700, 10.0, 9
    orbit = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN, alpha0=2.0, rot0=0.3)
    rng = np.random.default_rng(13)
    t = dt * np.arange(n)
    hp = np.cos(2 * math.pi * 2e-3 * t + 0.2) + 0.3 * np.cos(2 * math.pi * 7e-3 * t)
    hc = np.sin(2 * math.pi * 2e-3 * t)
    src = (0.3, 1.2, 0.5)
    r = orc80.response_full(orbit, hp[None], hc[None], [src], 15, order)
    R, nh, L = orc80.orbit_tables(orbit)
    beta, lam, psi = src
    k = -np.array([math.cos(beta) * math.cos(lam), math.cos(beta) * math.sin(lam), math.sin(beta)])
    M = order + 1

    def interp(series, n0, d):
        s = d / dt
        q = math.ceil(s)
        taps = np.arange(n0 - q - (M // 2 - 1), n0 - q + M // 2 + 1)
        return float(BarycentricInterpolator(taps.astype(float), series[taps])(n0 - s))

    def y_at(l, m):
        s_, r_ = LINKS[l]
        nv = nh[l][:, m]
        Hs = tensor_H(beta, lam, psi, nv, interp(hp, m, L[l, m] + k @ R[s_][:, m] / C),
                      interp(hc, m, L[l, m] + k @ R[s_][:, m] / C))
        Hr = tensor_H(beta, lam, psi, nv, interp(hp, m, k @ R[r_][:, m] / C), interp(hc, m, k @ R[r_][:, m] / C))
        return (Hs - Hr) / (2 * (1 - k @ nv))

    n0 = 350
    assert abs(y_at(1, n0) - r["y"][1, 0, n0]) < 1e-12 * np.abs(r["y"][1, 0]).max()
    # X_1.5 at n0, Eq. (2.7), with y series from the brute force on the needed window
    win = np.arange(n0 - 12, n0 + 8)
    ys = {l: np.zeros(n) for l in (1, 2, 4, 5)}
    for l in ys:
        for m in win:
            ys[l][m] = y_at(l, m)
    Lp2, Lp3, Lm2, Lm3 = L[1, n0], L[2, n0], L[4, n0], L[5, n0]
    X = (interp(ys[5], n0, Lm2 + Lp2 + Lp3) - interp(ys[5], n0, Lp3)
         + interp(ys[2], n0, Lp2 + Lm2) - ys[2][n0]
         + interp(ys[1], n0, Lm2) - interp(ys[1], n0, Lm2 + Lm3 + Lp3)
         + ys[4][n0] - interp(ys[4], n0, Lm3 + Lp3))
    assert abs(X - r["XYZ"][0, 0, n0]) < 1e-11 * np.abs(r["XYZ"][0, 0]).max()


def test_margins_are_zero_and_interior_is_not(orc80):
    n, dt = 900, 10.0
    orbit = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN)
    hp, hc = W.monochromatic(n, dt, 3e-3)
    r = orc80.response_full(orbit, hp[None], hc[None], [(0.1, 0.2, 0.3)], 20, 9)
    lo, hi = orc80.margins(orbit, 20, 9)
    for key in ("A", "E", "T"):
        assert np.all(r[key][0, :lo] == 0) and np.all(r[key][0, n - hi:] == 0)
    assert np.all(r["A"][0, lo:n - hi] != 0)
    ylo, yhi = orc80.link_margins(orbit, 9)
    assert np.all(r["y"][:, 0, :ylo] == 0) and np.all(r["y"][:, 0, n - yhi:] == 0)
    assert np.all(r["y"][:, 0, ylo:n - yhi] != 0)


def test_range_evaluation_equals_full_evaluation(orc80):
    """the sampled-output mode used at full sizes returns exactly the whole-grid values"""
    n, dt = 1500, 5.0
    orbit = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN)
    hp, hc = W.monochromatic(n, dt, 2e-3)
    src = [(0.1, 0.2, 0.3)]
    hyb = {"t_hyb": 4000.0, "window_s": 1000.0, "sigma_s": 25.0, "taper": W.TAPER_COSINE}
    whole = {"full": orc80.response_full(orbit, hp[None], hc[None], src, 20, 31),
             "lfa": orc80.response_lfa(orbit, hp[None], hc[None], src, 20, 31, 4),
             "hyb": orc80.response_hybrid(orbit, hp[None], hc[None], src, 20, 31, 2, hyb)}
    part = {"full": orc80.response_full(orbit, hp[None], hc[None], src, 20, 31, nb=700, ne=760),
            "lfa": orc80.response_lfa(orbit, hp[None], hc[None], src, 20, 31, 4, nb=700, ne=760),
            "hyb": orc80.response_hybrid(orbit, hp[None], hc[None], src, 20, 31, 2, hyb, nb=700, ne=760)}
    for k in whole:
        for key in ("A", "E", "T"):
            assert np.array_equal(whole[k][key][:, 700:760], part[k][key])
        assert np.array_equal(whole[k]["y"][:, :, 700:760], part[k]["y"])


# ---------------------------------------------------------------------------------------------
# O10 margins (G11): no valid output reads a margin sample
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gen", [15, 20])
@pytest.mark.parametrize("order,dt", [(31, 5.0), (9, 10.0), (31, 1.7)])
def test_valid_michelson_samples_never_read_the_link_margins(orc80, gen, order, dt):
    """Plant a sentinel in every margin sample of the link series (n < m1 or n >= N - m1, orc_link_margins): X, Y, Z
    on the valid range [lo, N - hi) of orc_margins must not change by a bit.  Fails if the TDI reach of O10 is too
    short for the largest delay of Eq. (2.7) / (2.8) (3 resp. 7 light times plus half a stencil) or if the forward
    stencil half overruns hi."""
    lo, hi = orc80.margins(W.orbit_desc(10, dt), gen, order, 0)
    n = lo + hi + 700
    orbit = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN, t0=4.0e6)
    ylo, yhi = orc80.link_margins(orbit, order, 0)
    rng = np.random.default_rng(5)
    y = rng.standard_normal((6, n))
    ref = orc80.michelson_from_links(orbit, y, gen, order)
    y2 = y.copy()
    y2[:, :ylo] = 1.0e30
    y2[:, n - yhi:] = -1.0e30
    got = orc80.michelson_from_links(orbit, y2, gen, order)
    assert np.array_equal(got[:, lo:n - hi], ref[:, lo:n - hi])
    assert np.all(got[:, :lo] == 0.0) and np.all(got[:, n - hi:] == 0.0)
    # and the bound is not vacuous: one more valid sample at the front would read the sentinel for gen 2.0 ...
    # (the reach 7.2 L / c + M / 2 exceeds the largest delay by < 0.3 L / c + stencil slack), checked loosely:
    assert lo - ylo < (7.2 if gen == 20 else 3.1) * (orbit["arm_m"] / W.C_LIGHT) / dt + order + 3


def test_link_quantities_split_as_hi_plus_lo(orc80):
    """orc_orbit_tables_split: hi is the fp64 rounding of the long-double n_l, L_l; |lo| <= ulp(hi) / 2; the plain
    tables are the hi parts"""
    orbit = W.orbit_desc(2001, 5.0, W.ORBIT_KEPLERIAN, t0=1.0e7)
    nh, nl, Lh, Ll = orc80.orbit_tables_split(orbit)
    _, n_plain, L_plain = orc80.orbit_tables(orbit)
    assert np.array_equal(nh, n_plain) and np.array_equal(Lh, L_plain)
    assert np.all(np.abs(nl) <= 0.5 * np.spacing(np.abs(nh)) + 1e-300) and np.all(np.abs(Ll) <= 0.5 * np.spacing(Lh))
    assert np.abs(nl).max() > 1e-18          # the long double build really carries more digits
    # unit vectors to beyond fp64: |n|^2 - 1 from the split pieces (exact products via math.fsum)
    import math
    for l in range(3):
        for i in (0, 1000, 2000):
            h, lw = nh[l, :, i], nl[l, :, i]
            s = math.fsum([h[0] * h[0], h[1] * h[1], h[2] * h[2], 2 * h[0] * lw[0], 2 * h[1] * lw[1], 2 * h[2] * lw[2], -1.0])
            assert abs(s) < 2e-16            # products rounded to fp64 in this check; the split itself is at 1e-19
