"""GPU parity of SURVEY 8(f)-3: the chirp + ringdown model generated on the device (ltdi_waveform_chirp) and the
projection that evaluates it at the retarded times (ltdi_response_full_chirp), against the long-double oracle O13."""
import numpy as np
import pytest
import torch

import workloads as W
from parity_util import hybrid_params, record, strict_check, to_numpy

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ltdi():
    import paper_2505_09600_b200 as m
    assert torch.cuda.is_available(), "GPU parity tests need a CUDA device"
    return m


@pytest.mark.parametrize("k,n", [(1, None), (2, 60001), (3, 200003), (4, 50001)])
def test_model_on_the_grid(ltdi, orc80, k, n):
    """element by element: a few fp64 roundings of the envelope, also where the phase is 1.5e5 rad (config 3): the phase is
    carried in double-double"""
    cfg = W.config(k, n=n, batch=3) if n else W.config(k)
    idx = list(range(cfg["batch"]))
    par = [W.chirp_params(cfg, i) for i in idx]
    hp, hc = ltdi.waveform_chirp(par, cfg["orbit"]["t0"], cfg["dt"], cfg["n"])
    torch.cuda.synchronize()
    rp, rc = orc80.waveform_chirp(par, cfg["orbit"]["t0"], cfg["dt"], cfg["n"])
    for b in idx:
        env = np.maximum.accumulate(np.abs(rp[b]) + np.abs(rc[b]))   # running envelope (the amplitude grows towards the merger)
        env = np.maximum(env, env[-1] * 1e-300)
        ep = np.abs(hp[b].cpu().numpy() - rp[b]) / env
        ec = np.abs(hc[b].cpu().numpy() - rc[b]) / env
        # the long-double oracle itself rounds the phase to 2^-64 relative: 8e-15 rad at the 1.5e5 rad of config 3
        phase_max = 2.0 * ((par[b]["t_c"] - cfg["orbit"]["t0"]) / (5.0 * par[b]["mc_s"])) ** 0.625
        bar = 4e-15 + 2.0 ** -62 * phase_max
        record(series="h", label=["cfg%d" % k, "source", str(b)], err=float(max(ep.max(), ec.max())), bar=bar)
        assert max(ep.max(), ec.max()) <= bar, (k, b, ep.max(), ec.max(), bar)


@pytest.mark.parametrize("k,n,gen", [(2, 40007, 20), (2, 40007, 15), (1, None, 15), (4, 20001, 20)])
def test_projection_at_retarded_times(ltdi, orc80, k, n, gen):
    cfg = W.config(k, n=n, batch=3 if k == 4 else 1) if n else W.config(k)
    idx = list(range(cfg["batch"]))
    par = [W.chirp_params(cfg, i) for i in idx]
    ang = np.array([W.source(dict(cfg, n=16), i)[2] for i in idx])
    orbit, order = cfg["orbit"], cfg["order"]
    ref = orc80.response_full_chirp(orbit, par, ang, gen, order)
    orb = ltdi.Orbits(orbit)
    out = to_numpy(ltdi.response_full_chirp(orb, par, ang, gen, order, True, True))
    lo, hi = orc80.margins(orbit, gen, order, 0)
    strict_check(out, ref, lo, hi, cfg["n"])


def test_hybrid_without_host_strain(ltdi, orc80):
    """the strain generated on the device feeds the hybrid response (no host -> device copy of h); reference: the oracle's
    hybrid on the oracle's own samples of the model"""
    cfg = W.config(2, n=40007)
    par = [W.chirp_params(cfg, 0)]
    _, _, ang, metas = W.sources(cfg, [0])
    orbit, order = cfg["orbit"], cfg["order"]
    rp, rc = orc80.waveform_chirp(par, orbit["t0"], cfg["dt"], cfg["n"])
    ref = orc80.response_hybrid(orbit, rp, rc, ang, 20, order, 2, hybrid_params(metas, orc80.hyb_time, W.TAPER_COSINE, cfg["dt"]))
    hp, hc = ltdi.waveform_chirp(par, orbit["t0"], cfg["dt"], cfg["n"])
    orb = ltdi.Orbits(orbit)
    out = to_numpy(ltdi.response_hybrid(orb, hp, hc, ang, 20, order, 2, hybrid_params(metas, ltdi.hyb_time, W.TAPER_COSINE, cfg["dt"]), True, True))
    lo, hi = orc80.margins(orbit, 20, order, 2)
    strict_check(out, ref, lo, hi, cfg["n"])


def test_chirp_argument_errors(ltdi):
    cfg = W.config(2, n=5003)
    par = [W.chirp_params(cfg, 0)]
    ang = np.array([[0.1, 0.2, 0.3]])
    orb = ltdi.Orbits(cfg["orbit"])
    with pytest.raises(ltdi.LtdiError):
        ltdi.response_full_chirp(orb, [dict(par[0], mc_s=0.0)], ang, 20, 31)
    with pytest.raises(ltdi.LtdiError):
        ltdi.response_full_chirp(orb, par, ang, 20, 7)      # tuned orders only
    with pytest.raises(ltdi.LtdiError):
        ltdi.waveform_chirp([dict(par[0], tau_rd=-1.0)], 0.0, 5.0, 100)


@pytest.mark.parametrize("n,nharm", [(40001, 10), (262147, 6)])
def test_eccentric_model_on_the_grid(ltdi, orc80, n, nharm):
    """the harmonic-sum model (orbital evolution table + cubic Hermite + Bessel coefficients, ltdi_waveform_ecc) against O13b,
    element by element: roundings of the sum of nharm harmonics, plus the oracle's own 2^-64 rounding of the mean anomaly
    times the harmonic number"""
    cfg = W.config(5, n=n, batch=3)
    idx = list(range(cfg["batch"]))
    tabs, pars = zip(*[W.ecc_params(cfg, i) for i in idx])
    tab, par = np.stack(tabs), np.stack(pars)
    hp, hc = ltdi.waveform_ecc(torch.as_tensor(tab, device="cuda"), par, nharm, cfg["orbit"]["t0"], cfg["dt"], cfg["n"])
    torch.cuda.synchronize()
    rp, rc = orc80.waveform_ecc(tab, par, nharm, cfg["orbit"]["t0"], cfg["dt"], cfg["n"])
    for b in idx:
        env = np.maximum.accumulate(np.abs(rp[b]) + np.abs(rc[b]))
        env = np.maximum(env, env[-1] * 1e-300)
        ep = np.abs(hp[b].cpu().numpy() - rp[b]) / env
        ec = np.abs(hc[b].cpu().numpy() - rc[b]) / env
        l_max = np.abs(tab[b, 3]).max() + abs(par[b, 5])
        bar = 8e-15 + nharm * 2.0 ** -62 * l_max
        record(series="h_ecc", label=["cfg5", "nharm%d" % nharm, "source", str(b)], err=float(max(ep.max(), ec.max())), bar=bar)
        assert max(ep.max(), ec.max()) <= bar, (b, ep.max(), ec.max(), bar, l_max)


def test_eccentric_model_outside_the_table_and_errors(ltdi, orc80):
    """sample times before the first and after the last knot use the end intervals, as O13b does; bad arguments are refused"""
    cfg = W.config(5, n=20001, batch=1)
    tab, par = W.ecc_params(cfg, 0)
    t0 = tab[0, 0] - 12 * cfg["dt"]                # under one knot interval out: the cubic is still well conditioned
    n = 1200
    hp, hc = ltdi.waveform_ecc(torch.as_tensor(tab[None], device="cuda"), par[None], 8, t0, cfg["dt"], n)
    rp, rc = orc80.waveform_ecc(tab[None], par[None], 8, t0, cfg["dt"], n)
    scale = np.abs(rp).max() + np.abs(rc).max()
    assert np.abs(hp.cpu().numpy() - rp).max() <= 1e-13 * scale and np.abs(hc.cpu().numpy() - rc).max() <= 1e-13 * scale
    t_last = tab[0, -1] - 388 * cfg["dt"]
    hp, hc = ltdi.waveform_ecc(torch.as_tensor(tab[None], device="cuda"), par[None], 8, t_last, cfg["dt"], 400)
    rp, rc = orc80.waveform_ecc(tab[None], par[None], 8, t_last, cfg["dt"], 400)
    assert np.abs(hp.cpu().numpy() - rp).max() <= 1e-13 * scale and np.abs(hc.cpu().numpy() - rc).max() <= 1e-13 * scale
    dtab = torch.as_tensor(tab[None], device="cuda")
    with pytest.raises(ltdi.LtdiError):
        ltdi.waveform_ecc(dtab, par[None], 0, t0, cfg["dt"], n)
    with pytest.raises(ltdi.LtdiError):
        ltdi.waveform_ecc(dtab, par[None], 65, t0, cfg["dt"], n)
    with pytest.raises(ltdi.LtdiError):
        ltdi.waveform_ecc(dtab, np.array([[0.0, 0.2, 1e25, 0.3, 0.1, 0.2]]), 8, t0, cfg["dt"], n)
    with pytest.raises(ltdi.LtdiError):
        ltdi.waveform_ecc(dtab[:, :, :1].contiguous(), par[None], 8, t0, cfg["dt"], n)


def test_eccentric_model_feeds_the_response(ltdi, orc80):
    """the strain generated on the device goes straight into the full response (no host copy): A, E, T against the oracle's
    response of the oracle's own strain, at the bar of the hot path"""
    cfg = W.config(5, n=30001, batch=2)
    tabs, pars = zip(*[W.ecc_params(cfg, i) for i in range(2)])
    tab, par = np.stack(tabs), np.stack(pars)
    ang = np.array([W.source(dict(cfg, n=16), i)[2] for i in range(2)])
    hp, hc = ltdi.waveform_ecc(torch.as_tensor(tab, device="cuda"), par, 10, cfg["orbit"]["t0"], cfg["dt"], cfg["n"])
    orb = ltdi.Orbits(cfg["orbit"])
    out = to_numpy(ltdi.response_full(orb, hp, hc, ang, 20, 31, True, True))
    rp, rc = orc80.waveform_ecc(tab, par, 10, cfg["orbit"]["t0"], cfg["dt"], cfg["n"])
    ref = orc80.response_full(cfg["orbit"], rp, rc, ang, 20, 31)
    lo, hi = orc80.margins(cfg["orbit"], 20, 31, 0)
    strict_check(out, ref, lo, hi, cfg["n"])
