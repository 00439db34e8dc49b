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
