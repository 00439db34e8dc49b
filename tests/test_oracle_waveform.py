"""Pins of O13 (no GPU): the chirp + ringdown waveform MODEL of the oracle and the projection that
evaluates it at the retarded times.  Checked against: the numpy input generator (an independent implementation of the
same recipe), Eq. (4.2) of the paper (the instantaneous frequency at t_hyb is f_hyb), the closed-form behaviour at the
join, and the already pinned interpolating response on the sampled model."""
import math

import numpy as np
import pytest

import workloads as W


@pytest.mark.parametrize("k,n,tol", [(1, None, 1e-12), (2, 30000, 1e-12), (4, 30000, 1e-12), (3, 30000, 2e-10)])
def test_model_equals_the_input_generator(orc80, k, n, tol):
    """C long double against numpy double, source by source (config 3: the generator's own fp64 phase of 1.5e5 rad)"""
    cfg = W.config(k, n=n) if n else W.config(k)
    for idx in (0, 1, 2):
        hp, hc, _, _ = W.source(cfg, idx)
        a, c = orc80.waveform_chirp([W.chirp_params(cfg, idx)], cfg["orbit"]["t0"], cfg["dt"], cfg["n"])
        assert np.abs(a[0] - hp).max() <= tol * np.abs(hp).max()
        assert np.abs(c[0] - hc).max() <= tol * np.abs(hc).max()


def test_frequency_at_t_hyb_is_f_hyb(orc80):
    """Eq. (4.2): t_hyb is where the model's instantaneous GW frequency reaches f_hyb"""
    mc, t_c = W.chirp_mass_s(1.0e6, 3.0), 5.0e5
    par = {"t_c": t_c, "mc_s": mc, "dist_m": 5 * W.GPC_M, "cos_iota": 0.3, "phi_c": 0.7, "tau_cut": 1e-3,
           "f_rd": 1.0, "tau_rd": 1.0}
    for f_hyb in (3e-4, 1e-3, 2e-3):
        th = orc80.hyb_time(f_hyb, mc, t_c)
        dt = 0.5
        hp, hc = orc80.waveform_chirp([par], th - 200 * dt, dt, 401)
        phase = np.unwrap(np.arctan2(hc[0] / par["cos_iota"], hp[0] / (0.5 * (1 + par["cos_iota"] ** 2))))
        f_inst = (phase[202] - phase[198]) / (4 * dt) / (2 * math.pi)
        assert abs(f_inst / f_hyb - 1.0) < 1e-6, (f_hyb, f_inst)


def test_join_and_ringdown(orc80):
    cfg = W.config(2, n=20000)
    par = W.chirp_params(cfg, 0)
    t_m = par["t_c"] - par["tau_cut"]
    eps = 1e-4
    (a0, a1), _ = orc80.waveform_chirp([par], t_m - eps, 2 * eps, 2)[0][0], None
    scale = np.abs(orc80.waveform_chirp([par], t_m - 100.0, 1.0, 200)[0]).max()
    assert abs(a1 - a0) < 1e-5 * scale                      # continuous across the join
    # one damping time after the join the envelope has fallen by e, and the frequency has relaxed towards f_rd
    dt = 0.25
    hp, hc = orc80.waveform_chirp([par], t_m, dt, int(8 * par["tau_rd"] / dt))
    env = np.hypot(hp[0] / (0.5 * (1 + par["cos_iota"] ** 2)), hc[0] / par["cos_iota"])
    k1 = int(round(par["tau_rd"] / dt))
    assert abs(env[k1] / env[0] - math.exp(-k1 * dt / par["tau_rd"])) < 1e-9
    phase = np.unwrap(np.arctan2(hc[0] / par["cos_iota"], hp[0] / (0.5 * (1 + par["cos_iota"] ** 2))))
    f_late = (phase[-1] - phase[-9]) / (8 * dt) / (2 * math.pi)
    f_cut = W.f_of_tau(par["tau_cut"], par["mc_s"])
    assert abs(f_late - par["f_rd"]) < 1e-3 * (par["f_rd"] - f_cut) + 1e-9 and f_cut < par["f_rd"]
    # 1 / d_L
    far = dict(par, dist_m=2 * par["dist_m"])
    h2 = orc80.waveform_chirp([far], t_m - 50.0, 1.0, 100)[0]
    h1 = orc80.waveform_chirp([par], t_m - 50.0, 1.0, 100)[0]
    assert np.abs(2 * h2 - h1).max() <= 1e-15 * np.abs(h1).max()


@pytest.mark.parametrize("k,gen", [(2, 20), (2, 15), (1, 15), (4, 20)])
def test_projection_at_retarded_times_equals_the_interpolated_one(orc80, k, gen):
    """the fused path against the pinned sampled path: the same model sampled on the grid, Lagrange order 31 (9 for config
    1), whose interpolation error is far below 1e-10 for these signals"""
    cfg = W.config(k, n=None if k == 1 else 12000, batch=1)
    par = [W.chirp_params(cfg, 0)]
    hp, hc, ang, _ = W.sources(cfg, [0])
    orbit, order = cfg["orbit"], 31
    fused = orc80.response_full_chirp(orbit, par, ang, gen, order)
    hs, cs = orc80.waveform_chirp(par, orbit["t0"], cfg["dt"], cfg["n"])
    sampled = orc80.response_full(orbit, hs, cs, ang, gen, order)
    lo, hi = orc80.margins(orbit, gen, order, 0)
    # the envelope of the model has a kink at the join (growing chirp -> decaying ringdown); a sampled series interpolates
    # through it with a first-order error, the fused path does not: compare where no stencil reaches the join
    n_join = int((par[0]["t_c"] - par[0]["tau_cut"] - orbit["t0"]) / cfg["dt"])
    end = min(cfg["n"] - hi, n_join - lo - 64)
    assert end - lo > 2000
    sl = slice(lo, end)
    top = max(np.linalg.norm(sampled[c][0, sl]) for c in "AET")
    for c in "AET":
        assert np.linalg.norm((fused[c] - sampled[c])[0, sl]) <= 1e-10 * top, c
    ytop = np.abs(sampled["y"][..., sl]).max()
    assert np.abs(fused["y"] - sampled["y"])[..., sl].max() <= 1e-10 * ytop
    if n_join < cfg["n"]:   # and near the join the two differ by the interpolation error of the kink: the reason O13 is its own oracle
        near = slice(n_join - 110, n_join + 110)   # k.R / c shifts the join by up to 100 samples either way
        assert np.abs(fused["y"] - sampled["y"])[..., near].max() > 1e-6 * np.abs(sampled["y"][..., near]).max()


# ---- O13b: the harmonic-sum waveform of an eccentric inspiral (config 5's recipe as a model) ---------------------------

def test_eccentric_model_equals_the_input_generator(orc80):
    cfg = W.config(5, n=30000, batch=2)
    for idx in (0, 1):
        hp, hc, _, _ = W.source(cfg, idx)
        tab, par = W.ecc_params(cfg, idx)
        a, c = orc80.waveform_ecc(tab[None], par[None], 10, cfg["orbit"]["t0"], cfg["dt"], cfg["n"])
        assert np.abs(a[0] - hp).max() <= 2e-12 * np.abs(hp).max()
        assert np.abs(c[0] - hc).max() <= 2e-12 * np.abs(hc).max()


def _table(tk, F, dF, e, de, ell, dell):
    return np.array([tk, F, e, ell, dF, de, dell])


def test_circular_limit_and_hermite_exactness(orc80):
    """e = 0: only n = 2 survives, h+ = 2 A (1 + cos^2 iota) cos(2 l + 2 gamma), hx = -4 A cos iota sin(2 l + 2 gamma); F and l
    cubic in time: the Hermite interpolation between the knots is exact"""
    tk = np.linspace(0.0, 4.0e4, 9)                      # 5000 s between knots
    s = tk / 4.0e4
    F = 1.0e-3 * (1 + 0.3 * s + 0.2 * s ** 2 + 0.1 * s ** 3)
    dF = 1.0e-3 * (0.3 + 0.4 * s + 0.3 * s ** 2) / 4.0e4
    ell = 2 * math.pi * 1.0e-3 * 4.0e4 * (s + 0.15 * s ** 2 + 0.2 / 3 * s ** 3)
    dell = 2 * math.pi * 1.0e-3 * (1 + 0.3 * s + 0.2 * s ** 2)
    M, eta, dist, ci, gam, l0 = 5.0, 0.2, 1.0e25, 0.37, 0.9, 0.4
    tab = _table(tk, F, dF, 0 * tk, 0 * tk, ell, dell)
    n, dt, t0 = 3000, 11.0, 777.0
    hp, hc = orc80.waveform_ecc(tab[None], np.array([[M, eta, dist, ci, gam, l0]]), 10, t0, dt, n)
    t = t0 + dt * np.arange(n)
    st = t / 4.0e4
    Ft = 1.0e-3 * (1 + 0.3 * st + 0.2 * st ** 2 + 0.1 * st ** 3)
    lt = 2 * math.pi * 1.0e-3 * 4.0e4 * (st + 0.15 * st ** 2 + 0.2 / 3 * st ** 3) + l0
    A = (2 * math.pi * Ft * M) ** (2.0 / 3.0) * eta * M * 299792458.0 / dist
    want_p = 2 * A * (1 + ci * ci) * np.cos(2 * lt + 2 * gam)
    want_c = -4 * A * ci * np.sin(2 * lt + 2 * gam)
    assert np.abs(hp[0] - want_p).max() <= 1e-12 * np.abs(want_p).max()
    assert np.abs(hc[0] - want_c).max() <= 1e-12 * np.abs(want_p).max()


@pytest.mark.parametrize("e", [0.1, 0.3, 0.5])
def test_peters_mathews_power_sum(orc80, e):
    """the harmonic amplitudes, read off the model's own output by a Fourier analysis over one orbit, satisfy the classic sum
    sum_n g(n, e) = (1 + 73/24 e^2 + 37/96 e^4) / (1 - e^2)^(7/2), g = n^2 / 32 [a_n^2 + b_n^2 + c_n^2 / 3] in units of A"""
    nh, F0, N = 40, 1.0e-3, 512
    P = 1.0 / F0
    tk = np.array([-P, 0.0, P, 2 * P, 3 * P])
    one = np.ones_like(tk)
    tab = _table(tk, F0 * one, 0 * one, e * one, 0 * one, 2 * math.pi * F0 * tk, 2 * math.pi * F0 * one)
    M, eta, dist = 5.0, 0.2, 1.0e25
    A = (2 * math.pi * F0 * M) ** (2.0 / 3.0) * eta * M * 299792458.0 / dist
    dt = P / N

    def harmonics(ci):
        hp, hc = orc80.waveform_ecc(tab[None], np.array([[M, eta, dist, ci, 0.0, 0.0]]), nh, 0.0, dt, N)
        return 2 * np.fft.rfft(hp[0]).real[1:nh + 1] / N / A, -2 * np.fft.rfft(hc[0]).imag[1:nh + 1] / N / A

    p1, q1 = harmonics(1.0)          # h+ = -2 a_n cos(n l),  hx = 2 b_n sin(n l)
    p0, _ = harmonics(0.0)           # h+ = (-a_n + c_n) cos(n l)
    a, b = -p1 / 2, q1 / 2
    c = p0 + a
    n = np.arange(1, nh + 1)
    g = n ** 2 / 32.0 * (a ** 2 + b ** 2 + c ** 2 / 3.0)
    want = (1 + 73.0 / 24 * e ** 2 + 37.0 / 96 * e ** 4) / (1 - e ** 2) ** 3.5
    assert abs(g.sum() / want - 1.0) < 1e-9, (e, g.sum(), want)
