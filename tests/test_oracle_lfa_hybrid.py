"""Pins of the oracle's LFA (Sec. III, App. B) and hybrid (Sec. IV) parts (no GPU)."""
import math

import numpy as np
import pytest

import workloads as W
from test_oracle_pins import (C, LINKS, closed_form, fit_complex_amplitude, frozen_orbit, golden,
                              tensor_H)


def stencil_transfer(which, fd_order, w, dt):
    """Fourier symbol of the central stencils (textbook): FD1 -> i w S1, FD2 -> -w^2 S2"""
    x = w * dt
    if which == 1:
        return 1j * (math.sin(x) if fd_order == 2 else (8 * math.sin(x) - math.sin(2 * x)) / 6) / dt
    if fd_order == 2:
        return (2 * math.cos(x) - 2) / dt ** 2
    return (-30 + 32 * math.cos(x) - 2 * math.cos(2 * x)) / (12 * dt ** 2)


def triangle_tables(orc, n, dt):
    """frozen constellation with L_l = |R_r - R_s| / c, so that L_l = L_-l and L n = R_r - R_s"""
    snap = W.orbit_desc(1, 1.0, W.ORBIT_KEPLERIAN, t0=0.21 * W.YEAR_S, rot0=1.1)
    R, _, _ = orc.orbit_tables(snap)
    R0 = R[:, :, 0]
    L0 = np.array([np.linalg.norm(R0[r] - R0[s]) / C for s, r in LINKS])
    return W.frozen_tables(W.orbit_desc(n, dt), R0, L0), R0, L0


@pytest.mark.parametrize("gen,fd_order", [(15, 2), (15, 4), (20, 2), (20, 4)])
def test_lfa_closed_form_on_frozen_constellation(orc80, gen, fd_order):
    """Eqs. (B1), (B10), (B25), (B33) in the Fourier domain, with distinct light times per link"""
    n, dt, order, f_hz = 1400, 5.0, 31, 1.5e-3
    orbit, R0, L0 = frozen_orbit(orc80, n, dt)
    w = 2 * math.pi * f_hz
    ap, ac = 1.0 * np.exp(0.3j), 0.7 * np.exp(1.1j)
    hp, hc = W.monochromatic(n, dt, f_hz, 1.0, 0.7, 0.3, 1.1)
    src = (0.45, 2.1, 0.8)
    beta, lam, psi = src
    k = -np.array([math.cos(beta) * math.cos(lam), math.cos(beta) * math.sin(lam), math.sin(beta)])
    r = orc80.response_lfa(orbit, hp[None], hc[None], [src], gen, order, fd_order)
    lo, hi = orc80.margins(orbit, gen, order, fd_order)
    t = dt * np.arange(n)
    D1 = stencil_transfer(1, fd_order, w, dt)
    Dk = stencil_transfer(1 if gen == 15 else 2, fd_order, w, dt)
    Yl = np.zeros(3, dtype=complex)
    for l in range(3):
        s, rr = LINKS[l]
        nv = (R0[rr] - R0[s]) / np.linalg.norm(R0[rr] - R0[s])
        tau = L0[l] / 2 + k @ (R0[s] + R0[rr]) / (2 * C)
        Yl[l] = -(L0[l] / 2) * tensor_H(beta, lam, psi, nv, ap, ac) * D1 * np.exp(-1j * w * tau)
        z, res = fit_complex_amplitude(r["y"][l, 0], t, w, lo, n - hi)
        assert res < 1e-10 and abs(z - Yl[l]) < 1e-11 * abs(Yl[l])
    assert np.all(r["y"][3:] == 0)  # "the rest are set to zero"
    for ch in range(3):
        p2 = (2 + ch - 1) % 3 + 1
        p3 = (3 + ch - 1) % 3 + 1
        L2, L3 = L0[p2 - 1], L0[p3 - 1]
        y123, y231 = Yl[p2 - 1], Yl[p3 - 1]
        D = lambda x: np.exp(-1j * w * x)
        if gen == 15:
            want = 4 * Dk * (L3 * D(L3 + L2 / 2) * y123 - L2 * D(L2 + L3 / 2) * y231)
        else:
            want = 8 * (L2 + L3) * Dk * (L3 * D(2 * L3 + 1.5 * L2) * y123 - L2 * D(2 * L2 + 1.5 * L3) * y231)
        z, res = fit_complex_amplitude(r["XYZ"][ch, 0], t, w, lo, n - hi)
        assert res < 1e-9 and abs(z - want) < 1e-10 * abs(want), (gen, ch)


def test_lfa_link_converges_to_full_with_x_over_sinx_law(orc80):
    """north-star check 5 / Eq. (B4): y_LFA / y_Full = (x / sin x) * S(w), x = (w L / 2)(1 - k.n), on a
    frozen triangle; S(w) = FD1 symbol / (i w) is the textbook transfer of the order-4 stencil
    (1 - (w dt)^4 / 30 + ...), 3.4e-6 away from 1 at the highest frequency used here"""
    n, dt, order = 2600, 2.0, 31
    orbit, R0, L0 = triangle_tables(orc80, n, dt)
    src = (0.3, 5.0, 0.4)
    beta, lam, _ = src
    k = -np.array([math.cos(beta) * math.cos(lam), math.cos(beta) * math.sin(lam), math.sin(beta)])
    t = dt * np.arange(n)
    prev = None
    for f_hz in (8e-3, 4e-3, 2e-3):
        w = 2 * math.pi * f_hz
        hp, hc = W.monochromatic(n, dt, f_hz)
        rf = orc80.response_full(orbit, hp[None], hc[None], [src], 15, order)
        rl = orc80.response_lfa(orbit, hp[None], hc[None], [src], 15, order, 4)
        lo, hi = orc80.margins(orbit, 15, order, 4)
        errs = []
        for l in range(3):
            s, rr = LINKS[l]
            nv = (R0[rr] - R0[s]) / np.linalg.norm(R0[rr] - R0[s])
            x = 0.5 * w * L0[l] * (1 - k @ nv)
            zf, _ = fit_complex_amplitude(rf["y"][l, 0], t, w, lo, n - hi)
            zl, _ = fit_complex_amplitude(rl["y"][l, 0], t, w, lo, n - hi)
            ratio = zl / zf
            S = (stencil_transfer(1, 4, w, dt) / (1j * w)).real
            assert abs(ratio - S * x / math.sin(x)) < 2e-8, (f_hz, l, ratio, x / math.sin(x))
            assert abs(ratio - x / math.sin(x)) < 5e-6
            errs.append(abs(ratio - 1))
        if prev is not None:  # relative error falls as f^2
            for a, b in zip(prev, errs):
                assert 3.5 < a / b < 4.5
        prev = errs


@pytest.mark.parametrize("gen", [15, 20])
def test_lfa_michelson_converges_to_full_as_f_squared(orc80, gen):
    """(B25)/(B33) and their cyclic permutations against the (closed-form-pinned) full response:
    the difference falls as f^2 for X, Y and Z -> every sign, prefactor and retarded time is right"""
    n, dt, order = 3000, 5.0, 31
    orbit, R0, L0 = triangle_tables(orc80, n, dt)
    src = (-0.5, 1.0, 1.3)
    t = dt * np.arange(n)
    errs = []
    for f_hz in (1.0e-3, 0.5e-3, 0.25e-3):
        w = 2 * math.pi * f_hz
        hp, hc = W.monochromatic(n, dt, f_hz)
        rf = orc80.response_full(orbit, hp[None], hc[None], [src], gen, order)
        rl = orc80.response_lfa(orbit, hp[None], hc[None], [src], gen, order, 4)
        lo, hi = orc80.margins(orbit, gen, order, 4)
        e = []
        for ch in range(3):
            zf, _ = fit_complex_amplitude(rf["XYZ"][ch, 0], t, w, lo, n - hi)
            zl, _ = fit_complex_amplitude(rl["XYZ"][ch, 0], t, w, lo, n - hi)
            e.append(abs(zl - zf) / abs(zf))
        errs.append(e)
    errs = np.array(errs)
    assert errs[0].max() < 2e-2 and errs[2].max() < 1.5e-3
    assert np.all(errs[0] / errs[1] > 3.5) and np.all(errs[0] / errs[1] < 4.5)
    assert np.all(errs[1] / errs[2] > 3.5) and np.all(errs[1] / errs[2] < 4.5)


def test_lfa_on_moving_constellation_is_at_the_1e4_level(orc80):
    """with L_l != L_-l and a moving constellation the LFA-full residual in the early
    inspiral is O(R Omega / c) ~ 1e-4 (order-of-magnitude pin, not a parity target)"""
    n, dt, order = 6000, 10.0, 31
    orbit = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN)
    hp, hc = W.monochromatic(n, dt, 1.0e-4)
    src = [(0.3, 1.0, 0.7)]
    rf = orc80.response_full(orbit, hp[None], hc[None], src, 15, order)
    rl = orc80.response_lfa(orbit, hp[None], hc[None], src, 15, order, 4)
    lo, hi = orc80.margins(orbit, 15, order, 4)
    x, y = rf["XYZ"][0, 0, lo:n - hi], rl["XYZ"][0, 0, lo:n - hi]
    rel = np.linalg.norm(x - y) / np.linalg.norm(x)
    assert 2e-5 < rel < 1.5e-3


@pytest.mark.parametrize("gen", [15, 20])
def test_T_channel_of_lfa_vanishes_for_equal_constant_arms(orc80, gen):
    """(B27)/(B35): X + Y + Z = 0 identically when all L_l are equal ("T ~ 0")"""
    n, dt = 2000, 5.0
    orbit = W.orbit_desc(n, dt, W.ORBIT_STATIC_EQUALARM)
    hp, hc = W.monochromatic(n, dt, 1.0e-3)
    r = orc80.response_lfa(orbit, hp[None], hc[None], [(0.3, 1.0, 0.7)], gen, 31, 2)
    assert np.abs(r["T"]).max() < 1e-16 * np.abs(r["A"]).max()


def test_lfa_generation_relation_B34(orc80):
    """Eq. (B34)/(B36): X_2.0^LFA = 2 (L2 + L3) d/dt X_1.5^LFA (t - L2 - L3) up to O((w dt)^2, (w L)^2)"""
    n, dt, f_hz = 3000, 2.0, 2.0e-4
    orbit, R0, L0 = triangle_tables(orc80, n, dt)
    hp, hc = W.monochromatic(n, dt, f_hz)
    src = [(0.2, 0.5, 1.0)]
    w = 2 * math.pi * f_hz
    t = dt * np.arange(n)
    r15 = orc80.response_lfa(orbit, hp[None], hc[None], src, 15, 31, 4)
    r20 = orc80.response_lfa(orbit, hp[None], hc[None], src, 20, 31, 4)
    lo, hi = orc80.margins(orbit, 20, 31, 4)
    for ch in range(3):
        p2 = (2 + ch - 1) % 3 + 1
        p3 = (3 + ch - 1) % 3 + 1
        L2, L3 = L0[p2 - 1], L0[p3 - 1]
        z15, _ = fit_complex_amplitude(r15["XYZ"][ch, 0], t, w, lo, n - hi)
        z20, _ = fit_complex_amplitude(r20["XYZ"][ch, 0], t, w, lo, n - hi)
        pred = 2 * (L2 + L3) * 1j * w * np.exp(-1j * w * (L2 + L3)) * z15
        assert abs(z20 - pred) < 2e-4 * abs(z20)


def test_lfa_margins_are_zero(orc80):
    n, dt = 900, 10.0
    orbit = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN)
    hp, hc = W.monochromatic(n, dt, 3e-3)
    r = orc80.response_lfa(orbit, hp[None], hc[None], [(0.1, 0.2, 0.3)], 20, 9, 4)
    lo, hi = orc80.margins(orbit, 20, 9, 4)
    lo0, hi0 = orc80.margins(orbit, 20, 9, 0)
    assert lo == lo0 + 4 and hi == hi0 + 4
    for key in ("A", "E", "T"):
        assert np.all(r[key][0, :lo] == 0) and np.all(r[key][0, n - hi:] == 0)
    assert np.all(r["A"][0, lo:n - hi] != 0)


# ------------------------------------------------------------------ hybrid
def test_printed_lfa_fractions_and_hybridisation_time(orc80):
    g = golden()
    v, tol = g["lfa_fraction_3e-4"]
    assert abs(orc80.lfa_fraction(3e-4, 1e-4, 1.0) / v - 1) < tol            # 0.95
    v, tol = g["lfa_fraction_3e-4_fmin08"]
    assert abs(orc80.lfa_fraction(3e-4, 0.8e-4, 1.0) / v - 1) < tol          # 0.97
    v, tol = g["lfa_fraction_8e-4_fmin08"]
    assert abs(orc80.lfa_fraction(8e-4, 0.8e-4, 1.0) / v - 1) < tol          # 0.99
    v, tol = g["full_fraction_percent"]
    assert abs(100 * (1 - orc80.lfa_fraction(3e-4, 0.8e-4, 1.0)) / v - 1) < tol  # 3 %
    # Eq. (4.2) is the inverse of the leading-order f(tau) relation (textbook, Maggiore [69])
    for M, q, f in ((1e6, 1.0, 3e-4), (1e5, 4.0, 2e-3), (5e6, 8.0, 1e-4)):
        mc = W.chirp_mass_s(M, q)
        t_c = 1.0e6
        th = orc80.hyb_time(f, mc, t_c)
        assert abs(W.f_of_tau(t_c - th, mc) / f - 1) < 1e-12
        assert abs((t_c - th) / W.tau_of_f(f, mc) - 1) < 1e-12


@pytest.mark.parametrize("taper", [W.TAPER_SIGMOID, W.TAPER_COSINE])
def test_hybrid_weights(orc80, taper):
    T = 4000.0
    hyb = {"t_hyb": 50000.0, "window_s": T, "sigma_s": T / 40, "taper": taper}
    t = np.linspace(40000.0, 60000.0, 4001)
    a, b = orc80.hybrid_weights(hyb, t)
    inside = np.abs(t - 50000.0) <= T / 2
    assert np.abs(a[inside] + b[inside] - 1).max() < 1e-15      # partition of unity in the window
    assert np.all(b[t < 50000.0 - T / 2] == 0) and np.all(a[t > 50000.0 + T / 2] == 0)
    mid = np.argmin(np.abs(t - 50000.0))
    assert abs(a[mid] - 0.5) < 1e-12 and abs(b[mid] - 0.5) < 1e-12
    assert np.all(np.diff(b[inside]) >= 0) and np.all(np.diff(a[inside]) <= 0)
    if taper == W.TAPER_SIGMOID:
        # Eq. (4.1) literally, also outside the window on each response's own domain (G18)
        assert np.allclose(a[t <= 52000.0], 1 / (1 + np.exp((t[t <= 52000.0] - 50000.0) / (T / 40))), atol=1e-15)
        assert np.allclose(b[t >= 48000.0], 1 / (1 + np.exp(-(t[t >= 48000.0] - 50000.0) / (T / 40))), atol=1e-15)
        assert abs(a[inside][0] - 1) < 3e-9 and abs(b[inside][-1] - 1) < 3e-9   # 1 - 2e-9 at the edge
    else:
        assert np.all(a[t < 50000.0 - T / 2] == 1) and np.all(b[t > 50000.0 + T / 2] == 1)
        x = (t[inside] - 50000.0 + T / 2) / T
        assert np.allclose(b[inside], 0.5 * (1 - np.cos(math.pi * x)), atol=1e-15)
        # C^1 at the window ends: one-sided slope -> 0
        assert abs(b[inside][1] - b[inside][0]) < 1e-5 and abs(b[inside][-1] - b[inside][-2]) < 1e-5


@pytest.mark.parametrize("taper", [W.TAPER_SIGMOID, W.TAPER_COSINE])
def test_hybrid_is_separate_blend_of_links_and_michelson(orc80, taper):
    """Eqs. (4.5) and (4.6): y and X, Y, Z are blended separately (G19); far before the window the
    hybrid is the LFA, far after it is the full response"""
    n, dt, order, fd = 3000, 5.0, 31, 2
    orbit = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN)
    t = dt * np.arange(n)
    hp = np.cos(2 * math.pi * (5e-4 * t + 1.5e-7 * t ** 2))
    hc = np.sin(2 * math.pi * (5e-4 * t + 1.5e-7 * t ** 2))
    src = [(0.3, 1.0, 0.7)]
    T = 800 * dt if taper == W.TAPER_SIGMOID else 3600.0
    hyb = {"t_hyb": 7000.0, "window_s": T, "sigma_s": T / 40, "taper": taper}
    rh = orc80.response_hybrid(orbit, hp[None], hc[None], src, 20, order, fd, hyb)
    rf = orc80.response_full(orbit, hp[None], hc[None], src, 20, order)
    rl = orc80.response_lfa(orbit, hp[None], hc[None], src, 20, order, fd)
    lo, hi = orc80.margins(orbit, 20, order, fd)
    a, b = orc80.hybrid_weights(hyb, t)
    sl = slice(lo, n - hi)
    scale = np.abs(rf["XYZ"]).max()
    assert np.abs(rh["XYZ"][:, 0, sl] - (a[sl] * rl["XYZ"][:, 0, sl] + b[sl] * rf["XYZ"][:, 0, sl])).max() < 1e-15 * scale
    ylo, yhi = orc80.link_margins(orbit, order, fd)
    ys = slice(ylo, n - yhi)
    assert np.abs(rh["y"][:, 0, ys] - (a[ys] * rl["y"][:, 0, ys] + b[ys] * rf["y"][:, 0, ys])).max() < 1e-15 * np.abs(rf["y"]).max()
    assert np.all(rh["A"][0, :lo] == 0) and np.all(rh["A"][0, n - hi:] == 0)
    if taper == W.TAPER_COSINE:
        late = t > hyb["t_hyb"] + T / 2
        late[n - hi:] = False
        early = t < hyb["t_hyb"] - T / 2
        early[:lo] = False
        assert np.array_equal(rh["A"][0, late], rf["A"][0, late])
        assert np.array_equal(rh["A"][0, early], rl["A"][0, early])
        # NOT the same as recomputing X from the blended links: check (4.6) differs from that inside the window
        mid = np.abs(t - hyb["t_hyb"]) < T / 4
        assert np.abs(rh["XYZ"][0, 0, mid] - rf["XYZ"][0, 0, mid]).max() > 1e-6 * scale


# ---------------------------------------------------------------------------------------------
# higher-order single-link series (B4) and the other expansion points (B12)-(B14)
# ---------------------------------------------------------------------------------------------
def stencil3_transfer(fd_order, w, dt):
    """Fourier symbol of the central third-derivative stencils (textbook): FD3 -> (i w)^3 S3"""
    x = w * dt
    if fd_order == 2:
        return 1j * (math.sin(2 * x) - 2 * math.sin(x)) / dt ** 3
    return 1j * (-math.sin(3 * x) + 8 * math.sin(2 * x) - 13 * math.sin(x)) / (4 * dt ** 3)


@pytest.mark.parametrize("fd_order,exact_deg", [(2, 4), (4, 6)])
def test_third_derivative_stencil_is_exact_on_polynomials(orc80, fd_order, exact_deg):
    dt = 0.7
    x = np.arange(-12, 13) * dt
    for deg in range(exact_deg + 2):
        c = np.random.default_rng(deg).standard_normal(deg + 1)
        p = np.polynomial.Polynomial(c)
        got = orc80.stencil3(p(x), dt, fd_order)
        want = p.deriv(3)(x)
        w = fd_order // 2 + 1
        err = np.abs(got[w:-w] - want[w:-w]).max() / max(1.0, np.abs(want).max())
        if deg <= exact_deg:
            assert err < 1e-10, (deg, err)
        else:
            assert err > 1e-6, (deg, err)          # one degree higher: the truncation error shows
    assert np.all(orc80.stencil3(p(x), dt, fd_order)[:w] == 0)
    # and the symbol on a complex exponential
    wv = 0.31
    zs = orc80.stencil3(np.sin(wv * x), dt, fd_order)[12]       # d^3/dt^3 sin(w t) at t = 0 is -w^3: symbol / i
    assert abs(zs - (stencil3_transfer(fd_order, wv, dt) / 1j).real) < 1e-12


def test_lfa_ext_with_one_central_term_is_the_lfa(orc80):
    cfg = W.config(2, n=3000)
    hp, hc, ang, _ = W.sources(cfg, [0])
    a = orc80.response_lfa(cfg["orbit"], hp, hc, ang, 20, 31, 4)
    b = orc80.response_lfa_ext(cfg["orbit"], hp, hc, ang, 20, 31, 4, terms=1, point=0)
    for k in ("A", "E", "T", "XYZ", "y"):
        assert np.array_equal(a[k], b[k]), k
    assert orc80.margins_lfa_ext(cfg["orbit"], 20, 31, 4, 1) == orc80.margins(cfg["orbit"], 20, 31, 4)
    lo, hi = orc80.margins(cfg["orbit"], 20, 31, 4)
    assert orc80.margins_lfa_ext(cfg["orbit"], 20, 31, 4, 2) == (lo + 1, hi + 1)
    with pytest.raises(ValueError):
        orc80.response_lfa_ext(cfg["orbit"], hp, hc, ang, 20, 31, 4, terms=2, point=1)   # (B13), (B14): leading order only


def test_second_term_of_B4_turns_the_f2_law_into_f4(orc80):
    """Eq. (B4) on a frozen triangle: with m = 0, 1 the ratio to the full link is (x - x^3 / 6) / sin x up to the
    stencil symbols, x = (w L / 2)(1 - k.n): the residual falls as f^4 (factor 16 per octave) instead of f^2, and
    matches the closed form with the textbook symbols of the two stencils"""
    n, dt, order = 2600, 2.0, 31
    orbit, R0, L0 = triangle_tables(orc80, n, dt)
    src = (0.3, 5.0, 0.4)
    beta, lam, _ = src
    k = -np.array([math.cos(beta) * math.cos(lam), math.cos(beta) * math.sin(lam), math.sin(beta)])
    t = dt * np.arange(n)
    prev = None
    for f_hz in (8e-3, 4e-3, 2e-3):
        w = 2 * math.pi * f_hz
        hp, hc = W.monochromatic(n, dt, f_hz)
        rf = orc80.response_full(orbit, hp[None], hc[None], [src], 15, order)
        r2 = orc80.response_lfa_ext(orbit, hp[None], hc[None], [src], 15, order, 4, terms=2, point=0)
        lo, hi = orc80.margins_lfa_ext(orbit, 15, order, 4, 2)
        errs = []
        for l in range(3):
            s, rr = LINKS[l]
            nv = (R0[rr] - R0[s]) / np.linalg.norm(R0[rr] - R0[s])
            x = 0.5 * w * L0[l] * (1 - k @ nv)
            zf, _ = fit_complex_amplitude(rf["y"][l, 0], t, w, lo, n - hi)
            z2, _ = fit_complex_amplitude(r2["y"][l, 0], t, w, lo, n - hi)
            S1 = (stencil_transfer(1, 4, w, dt) / (1j * w)).real
            S3 = (stencil3_transfer(4, w, dt) / (1j * w) ** 3).real
            # (i w)^3 = -i w w^2: the series is i w (1 - x^2 / 6) against i w sin(x) / x of the full link
            want = (x * S1 - x ** 3 / 6 * S3) / math.sin(x)
            assert abs(z2 / zf - want) < 2e-8, (f_hz, l)
            errs.append(abs(z2 / zf - 1))
        if prev is not None:
            for a, b in zip(prev, errs):
                assert 12.0 < a / b < 20.0, (a, b)        # f^4 (the one-term series gives 4: test above)
        prev = errs


def test_forward_and_backward_points_are_first_order(orc80):
    """(B13), (B14) on a frozen triangle: y = -(L/2) dH/dt at t - delta_s resp. t - delta_r, so
    y_bwd / y_full = x e^{-i x} / sin x and y_fwd / y_full = x e^{+i x} / sin x: the error is O(x) -- the first-order
    error the paper attributes to the forward form of Ref. [46] -- against O(x^2) for the central point"""
    n, dt, order = 2600, 2.0, 31
    orbit, R0, L0 = triangle_tables(orc80, n, dt)
    src = (0.3, 5.0, 0.4)
    beta, lam, _ = src
    k = -np.array([math.cos(beta) * math.cos(lam), math.cos(beta) * math.sin(lam), math.sin(beta)])
    t = dt * np.arange(n)
    lo, hi = orc80.margins(orbit, 15, order, 4)
    prev = None
    for f_hz in (4e-3, 2e-3, 1e-3):
        w = 2 * math.pi * f_hz
        hp, hc = W.monochromatic(n, dt, f_hz)
        rf = orc80.response_full(orbit, hp[None], hc[None], [src], 15, order)
        errs = []
        for point, sign in ((1, -1.0), (2, +1.0)):
            r = orc80.response_lfa_ext(orbit, hp[None], hc[None], [src], 15, order, 4, terms=1, point=point)
            for l in range(3):
                s, rr = LINKS[l]
                nv = (R0[rr] - R0[s]) / np.linalg.norm(R0[rr] - R0[s])
                x = 0.5 * w * L0[l] * (1 - k @ nv)
                zf, _ = fit_complex_amplitude(rf["y"][l, 0], t, w, lo, n - hi)
                z, _ = fit_complex_amplitude(r["y"][l, 0], t, w, lo, n - hi)
                S1 = (stencil_transfer(1, 4, w, dt) / (1j * w)).real
                assert abs(z / zf - S1 * x * np.exp(sign * 1j * x) / math.sin(x)) < 2e-8, (f_hz, point, l)
                errs.append(abs(z / zf - 1))
        if prev is not None:
            for a, b in zip(prev, errs):
                assert 1.9 < a / b < 2.1, (a, b)          # first order in f
        prev = errs
