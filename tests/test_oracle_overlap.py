"""Pins of the overlap oracle (oracle/overlap_oracle.py): the noise model of Sec. II C and the inner product,
overlap, mismatch and SNR of Eqs. (5.1), (5.2), (6.1) against what the paper and the mathematics fix."""
import numpy as np
import pytest

from oracle import overlap_oracle as oo

L = 2.5e9
C = 299792458.0


def test_printed_noise_constants_and_reference_frequencies():
    # P:175, P:180-186 (typed from the paper a second time, independently of the oracle's table)
    assert oo.SQRT_S_ACC == 2.4e-15 and oo.SQRT_S_OMS == 7.9e-12
    assert (oo.GAL_A, oo.GAL_ALPHA, oo.GAL_F2) == (1.28265531e-44, 1.62966700, 4.81078093e-4)
    assert (oo.GAL_A1, oo.GAL_B1, oo.GAL_AK, oo.GAL_BK) == (-0.223499956, -2.70408439, -0.360976122, -2.37822436)
    # Fig. 2 caption: c / (2 pi L) = 0.019 Hz is where x = 1
    assert abs(C / (2 * np.pi * L) - 0.019) < 1e-3


def test_component_noises_follow_their_formulas_at_hand_computed_points():
    # Eq. (2.10a) at f = 0.0004 Hz: [1 + 1] [1 + (0.05)^4]; Eq. (2.10b) at f = 0.002 Hz: [1 + 1]
    f = 0.0004
    want = (2.4e-15) ** 2 / (2 * np.pi * f * C) ** 2 * 2.0 * (1.0 + 0.05 ** 4)
    assert oo.s_pm(f) == pytest.approx(want, rel=1e-14)
    f = 0.002
    want = (7.9e-12) ** 2 * (2 * np.pi * f / C) ** 2 * 2.0
    assert oo.s_op(f) == pytest.approx(want, rel=1e-14)
    # acceleration noise dominates below, optical-path noise above the crossing between 1 and 3 mHz
    assert oo.s_pm(1e-3) > oo.s_op(1e-3) and oo.s_pm(3e-3) < oo.s_op(3e-3)
    # asymptotic slopes: S_pm ~ f^-4 at low f, f^+2 at high f; S_op ~ f^-2 at low f, f^+2 at high f
    for fn, f, want in ((oo.s_pm, 1e-6, -4.0), (oo.s_pm, 10.0, 2.0), (oo.s_op, 1e-6, -2.0), (oo.s_op, 10.0, 2.0)):
        slope = np.log(fn(2 * f) / fn(f)) / np.log(2.0)
        assert abs(slope - want) < 1e-2


def test_galactic_foreground_shape():
    # Eq. (2.12) with T_obs = 1 yr: f1 = 10^b1, f_knee = 10^bk; the tanh factor switches the foreground off above f_knee
    f1, fk = 10 ** -2.70408439, 10 ** -2.37822436
    assert 1.9e-3 < f1 < 2.0e-3 and 4.1e-3 < fk < 4.3e-3
    f = np.array([1e-4, 1e-3, 3e-2])
    g = oo.s_gal(f, L, 1.0)
    x = 2 * np.pi * f * L / C
    want = 2 * x ** 2 * np.sin(x) ** 2 * 1.28265531e-44 * f ** (-7 / 3) * np.exp(-(f / f1) ** 1.629667) * (1 + np.tanh((fk - f) / 4.81078093e-4))
    assert np.allclose(g, want, rtol=1e-13)
    assert g[2] < 1e-20 * g[1]            # gone at 30 mHz
    # longer observation -> lower knee (a_k < 0): less foreground at 3 mHz
    assert oo.s_gal(3e-3, L, 4.0) < oo.s_gal(3e-3, L, 1.0)


@pytest.mark.parametrize("galactic", [False, True])
def test_generation_relation_and_low_frequency_power_laws(galactic):
    f = np.logspace(-5, -1, 300)
    x = 2 * np.pi * f * L / C
    a15, t15 = oo.psd_aet(f, 15, L, 1.0, galactic)
    a20, t20 = oo.psd_aet(f, 20, L, 1.0, galactic)
    lam = 4 * np.sin(2 * x) ** 2
    assert np.allclose(a20, lam * a15, rtol=1e-13) and np.allclose(t20, lam * t15, rtol=1e-13)
    assert np.all(a15 > 0) and np.all(t15 > 0)
    if not galactic:
        # S^{A 2.0} ~ c1 f^0 + c2 f^2 and S^{A 1.5} ~ c3 f^-2 + c4 f^0 at low frequency: slopes at 1e-5 Hz
        lo = slice(0, 20)
        s20 = np.polyfit(np.log(f[lo]), np.log(a20[lo]), 1)[0]
        s15 = np.polyfit(np.log(f[lo]), np.log(a15[lo]), 1)[0]
        assert abs((s20 - s15) - 2.0) < 0.01        # the two generations differ by f^2
        assert abs(s15 - (-2.0)) < 0.01 and abs(s20) < 0.01


def test_psd_has_the_zeros_of_the_tdi_transfer_function():
    # sin^2 x = 0 at f = n c / (2 L): the response and the noise vanish together ("0/0")
    f0 = C / (2 * L)
    a, t = oo.psd_aet(np.array([f0]), 15, L, 1.0, False)
    a_near, _ = oo.psd_aet(np.array([0.9 * f0]), 15, L, 1.0, False)
    assert a[0] < 1e-25 * a_near[0] and t[0] < 1e-25 * a_near[0]
    # TDI 2.0 adds the zeros of sin 2x: f = c / (4 L)
    a20, _ = oo.psd_aet(np.array([0.5 * f0]), 20, L, 1.0, False)
    a15, _ = oo.psd_aet(np.array([0.5 * f0]), 15, L, 1.0, False)
    assert a20[0] < 1e-25 * a15[0]


def test_parseval_with_white_noise():
    """S_n = 1: <x|y> = 4 Re int_0^inf x~* y~ df = 2 int x y dt (one-sided); the oracle's band excludes f = 0 and the
    sum is a rectangle rule, so the identity is exact for zero-mean series once the Nyquist bin is halved"""
    rng = np.random.default_rng(3)
    n, dt = 4096, 5.0
    x, y = rng.standard_normal(n), rng.standard_normal(n)
    x -= x.mean(); y -= y.mean()
    s = np.ones(n // 2 + 1)
    got = oo.inner(x, y, dt, s, 0.0, 1.0)
    # remove the double counting of the Nyquist bin (it appears once in the two-sided sum)
    nyq = (oo.spectrum(x, dt)[-1].conjugate() * oo.spectrum(y, dt)[-1]).real / (n * dt)
    assert got - 2.0 * nyq == pytest.approx(2.0 * np.sum(x * y) * dt, rel=1e-12)


def test_bin_centred_sinusoid_closed_form_and_band_limits():
    n, dt, k0, amp = 8000, 5.0, 37, 3.0e-21
    T = n * dt
    f0 = k0 / T
    t = dt * np.arange(n)
    x = amp * np.cos(2 * np.pi * f0 * t + 0.4)
    f = np.arange(n // 2 + 1) / T
    s = np.full_like(f, np.inf); s[1:], _ = oo.psd_aet(f[1:], 20)
    assert oo.inner(x, x, dt, s, 1e-5, 0.05) == pytest.approx(amp ** 2 * T / s[k0], rel=1e-10)
    # band limits are inclusive bins f_min <= f_k <= f_max (G25)
    assert oo.inner(x, x, dt, s, f0, f0) == pytest.approx(amp ** 2 * T / s[k0], rel=1e-10)
    assert abs(oo.inner(x, x, dt, s, f0 * 1.01, 0.05)) < 1e-20 * amp ** 2 * T / s[k0]
    # quadrature: cos against sin at the same bin is orthogonal, cos against itself shifted by phi gives cos(phi)
    y = amp * np.cos(2 * np.pi * f0 * t + 0.4 + 0.3)
    assert oo.inner(x, y, dt, s, 1e-5, 0.05) / oo.inner(x, x, dt, s, 1e-5, 0.05) == pytest.approx(np.cos(0.3), rel=1e-10)


def test_overlap_mismatch_and_snr_properties():
    rng = np.random.default_rng(5)
    n, dt = 6000, 10.0
    t = dt * np.arange(n)
    base = {c: 1e-21 * (np.sin(2 * np.pi * 2e-3 * t + i) * np.hanning(n) + 0.01 * rng.standard_normal(n))[None]
            for i, c in enumerate("AET")}
    same = oo.products(base, base, dt, 20, 1e-4, 2e-2)
    assert np.allclose(same[:, :, 3], 1.0, atol=1e-15) and np.allclose(same[:, :, 4], 0.0, atol=1e-15)
    neg = oo.products(base, {c: -2.5 * v for c, v in base.items()}, dt, 20, 1e-4, 2e-2)
    assert np.allclose(neg[:, :, 3], -1.0, atol=1e-15)                   # (5.2): scale-free, sign-aware
    assert np.allclose(neg[:, :, 4], 0.0, atol=1e-15)                    # M = 1 - |O|
    assert np.allclose(neg[:, :, 1], 6.25 * neg[:, :, 0], rtol=1e-14)
    other = {c: v + 3e-22 * rng.standard_normal(v.shape) for c, v in base.items()}
    ab = oo.products(base, other, dt, 20, 1e-4, 2e-2)
    ba = oo.products(other, base, dt, 20, 1e-4, 2e-2)
    assert np.allclose(ab[:, :, 2], ba[:, :, 2], rtol=1e-13)             # <a|b> = <b|a> (real series)
    assert np.all(np.abs(ab[:, :, 3]) <= 1.0 + 1e-15)                    # Cauchy-Schwarz
    assert np.all((ab[:, :, 4] >= 0.0) & (ab[:, :, 4] <= 1.0))
    # (6.1): rho^2 adds over the channels
    assert oo.snr(same[:, :, 0])[0] == pytest.approx(np.sqrt(same[0, :, 0].sum()), rel=1e-15)
    # T uses S_n^T, A and E share S_n^{A,E}: swapping the A and E series swaps their products
    swapped = oo.products({"A": base["E"], "E": base["A"], "T": base["T"]}, base, dt, 20, 1e-4, 2e-2)
    assert swapped[0, 0, 0] == pytest.approx(same[0, 1, 0], rel=1e-14)
    assert swapped[0, 2, 0] == pytest.approx(same[0, 2, 0], rel=1e-14)


def test_paper_accuracy_statements_hold_on_a_synthetic_merger(orc64):
    """hybrid mismatch below 1e-5 for A and E with both generations; LFA below 0.1 % (TDI 1.5) and below
    10 % (TDI 2.0) for A and E, 10-100 % for T -- reproduced by the two oracles on config 2's chirp + ringdown
    (last 200 000 samples; f_Hyb = 2 mHz as BASELINE.json asks; f_max = 0.02 Hz as P:502)."""
    import workloads as W
    from parity_util import hybrid_params
    cfg = W.config(2, n=200000)
    hp, hc, ang, metas = W.sources(cfg, [0])
    orbit, dt = cfg["orbit"], cfg["dt"]
    for gen, lfa_bar in ((15, 1e-3), (20, 1e-1)):
        full = orc64.response_full(orbit, hp, hc, ang, gen, 31, want=())
        lfa = orc64.response_lfa(orbit, hp, hc, ang, gen, 31, 2, want=())
        for taper in (W.TAPER_COSINE, W.TAPER_SIGMOID):
            hyb = orc64.response_hybrid(orbit, hp, hc, ang, gen, 31, 2, hybrid_params(metas, orc64.hyb_time, taper, dt),
                                        want=())
            m = oo.products(full, hyb, dt, gen, 1e-4, 2e-2)[0, :, 4]
            assert m[0] < 1e-5 and m[1] < 1e-5, (gen, taper, m)
        m = oo.products(full, lfa, dt, gen, 1e-4, 2e-2)[0, :, 4]
        assert m[0] < lfa_bar and m[1] < lfa_bar and 0.1 < m[2] <= 1.0, (gen, m)
    rho = oo.snr(oo.products(full, full, dt, 20, 1e-4, 2e-2)[:, :, 0])[0]
    assert 100.0 < rho < 1e4        # an MBHB at 5 Gpc: SNR in the hundreds to thousands (P:502 quotes 1876)


def test_log_likelihood_of_eq_D4():
    rng = np.random.default_rng(9)
    n, dt = 5000, 10.0
    t = dt * np.arange(n)
    d = {c: 1e-21 * (np.sin(2 * np.pi * 3e-3 * t + i) * np.hanning(n))[None] for i, c in enumerate("AET")}
    same = oo.products(d, d, dt, 20, 1e-4, 2e-2)
    assert abs(oo.log_likelihood(same)[0]) < 1e-12 * oo.snr(same[:, :, 0])[0] ** 2        # h = d: ln L = 0
    zero = {c: np.zeros_like(v) for c, v in d.items()}
    pz = oo.products(d, zero, dt, 20, 1e-4, 2e-2)
    assert oo.log_likelihood(pz)[0] == pytest.approx(-0.5 * oo.snr(pz[:, :, 0])[0] ** 2, rel=1e-14)   # h = 0: -rho^2 / 2
    eps = 1e-3
    ps = oo.products(d, {c: (1 + eps) * v for c, v in d.items()}, dt, 20, 1e-4, 2e-2)
    assert oo.log_likelihood(ps)[0] == pytest.approx(-0.5 * eps ** 2 * oo.snr(ps[:, :, 0])[0] ** 2, rel=1e-6)
    # direct definition: inner product of the residual with itself
    h = {c: v + 1e-23 * rng.standard_normal(v.shape) for c, v in d.items()}
    pr = oo.products(d, h, dt, 20, 1e-4, 2e-2)
    res = {c: d[c] - h[c] for c in "AET"}
    direct = -0.5 * oo.products(res, res, dt, 20, 1e-4, 2e-2)[0, :, 0].sum()
    assert oo.log_likelihood(pr)[0] == pytest.approx(direct, rel=1e-9)
