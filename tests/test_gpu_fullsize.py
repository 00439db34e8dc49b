"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (reused Workspace,
A / E / T outputs only, same tile plan and source chunking), on sampled windows of the output that the
long-double oracle evaluates one by one through its range arguments (nb, ne), plus properties that hold at
any size (margins exactly zero, replicated sources bitwise equal across chunks of the batch).

Bar: the north-star metric over the sampled outputs -- per channel, relative L2 pooled over the windows of a run
<= 1e-11 (T against the largest channel) -- and every single window within 1e-8 of the oracle against its own
norm (parity_util.Pooled); achieved errors and the fp64 floors go to gpurun_out/parity_report.jsonl."""
import numpy as np
import pytest
import torch

import workloads as W
from parity_util import Pooled, hybrid_params

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ltdi():
    import paper_2505_09600_b200 as m
    assert torch.cuda.is_available(), "GPU parity tests need a CUDA device"
    return m


def windows_of(n, lo, hi, extra=(), width=1500):
    """sample windows [nb, ne): both ends of the valid range (with a piece of margin), the middle, and any
    extra centres (the hybrid window, the merger, the loudest sample of the input strain -- the part of the series
    that carries its norm, so that the pooled metric weighs the windows as the whole-series norm would)"""
    centres = [lo + width // 2 - 40, n // 3, n // 2, n - hi - width // 2 + 40, *extra]
    out = []
    for c in centres:
        nb = int(min(max(c - width // 2, 0), n - width))
        out.append((nb, nb + width))
    return out


def run_gpu(ltdi, which, orb, dhp, dhc, ang, gen, order, fd, hyb, ws):
    if which == "full":
        out = ltdi.response_full(orb, dhp, dhc, ang, gen, order, workspace=ws)
    elif which == "lfa":
        out = ltdi.response_lfa(orb, dhp, dhc, ang, gen, order, fd, workspace=ws)
    else:
        out = ltdi.response_hybrid(orb, dhp, dhc, ang, gen, order, fd, hyb, workspace=ws)
    torch.cuda.synchronize()
    return out


def run_orc(o, which, orbit, hp, hc, ang, gen, order, fd, hyb, nb, ne):
    if which == "full":
        return o.response_full(orbit, hp, hc, ang, gen, order, nb=nb, ne=ne, want=())
    if which == "lfa":
        return o.response_lfa(orbit, hp, hc, ang, gen, order, fd, nb=nb, ne=ne, want=())
    return o.response_hybrid(orbit, hp, hc, ang, gen, order, fd, hyb, nb=nb, ne=ne, want=())


def single_source_case(ltdi, orc80, orc64, k, runs, extra_centres=lambda n, metas, cfg: ()):
    """configs 1-3: one source at full length; runs = [(which, gen, fd, taper)]"""
    cfg = W.config(k)
    n, order, orbit = cfg["n"], cfg["order"], cfg["orbit"]
    hp, hc, ang, metas = W.sources(cfg, [0])
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(orbit, device=dev)
    dhp, dhc = torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev)
    ws = ltdi.Workspace(1, n, dev)
    for which, gen, fd, taper in runs:
        fd_eff = 0 if which == "full" else fd
        lo, hi = orc80.margins(orbit, gen, order, fd_eff)
        hyb_g = hybrid_params(metas, ltdi.hyb_time, taper, cfg["dt"]) if which == "hybrid" else None
        hyb_o = hybrid_params(metas, orc80.hyb_time, taper, cfg["dt"]) if which == "hybrid" else None
        got = {c: v.cpu().numpy() for c, v in run_gpu(ltdi, which, orb, dhp, dhc, ang, gen, order, fd, hyb_g, ws).items()
               if c in "AET"}
        pool = Pooled((cfg["name"], which, gen, fd, taper))
        loud = [int(np.argmax(np.abs(hp[0])))]      # the loudest part of the input carries the norm of the whole series
        for nb, ne in windows_of(n, lo, hi, [*extra_centres(n, metas, cfg), *loud]):
            r80 = run_orc(orc80, which, orbit, hp, hc, ang, gen, order, fd, hyb_o, nb, ne)
            r64 = run_orc(orc64, which, orbit, hp, hc, ang, gen, order, fd, hyb_o, nb, ne)
            pool.add(got, r80, r64, nb, ne, lo, n, hi)
        pool.check()


def _hyb_centres(n, metas, cfg):
    """sample indices of the hybrid window centre and of the merger"""
    t0, dt = cfg["orbit"]["t0"], cfg["dt"]
    from oracle import Oracle
    th = Oracle("f64").hyb_time(metas[0]["f_hyb_hz"], metas[0]["mchirp_s"], metas[0]["t_c"])
    return [int(np.clip((th - t0) / dt, 0, n - 1)), int(np.clip((metas[0]["t_c"] - t0) / dt, 0, n - 1))]


def test_config2_full_size(ltdi, orc80, orc64):
    """the default bench workload: N = 518 400, TDI 2.0, order 31: full, LFA, hybrid (cosine and sigmoid)"""
    single_source_case(ltdi, orc80, orc64, 2,
                       [("full", 20, 0, 0), ("lfa", 20, 2, 0), ("hybrid", 20, 2, W.TAPER_COSINE),
                        ("hybrid", 20, 2, W.TAPER_SIGMOID)], _hyb_centres)


def test_config3_full_size(ltdi, orc80, orc64):
    """N = 6 307 200 LFA, both generations, both stencil orders"""
    single_source_case(ltdi, orc80, orc64, 3, [("lfa", g, fd, 0) for g in (15, 20) for fd in (2, 4)])


def batched_case(ltdi, orc80, orc64, k, batch, subset, runs):
    """configs 1, 4, 5 at full batch.  `subset` = indices (into the config's population of `batch` seeded sources) of
    the parity subset of SURVEY.md 8(d); those sources are generated and tiled over the `batch` rows (host
    generation of thousands of series would dominate the test), so that every chunk of the batch the library forms
    is exercised: replicas must be bitwise equal to the first copy, and EVERY source of the subset is compared with
    the oracle on its sampled windows."""
    cfg = W.config(k, batch=batch)
    n, order, orbit = cfg["n"], cfg["order"], cfg["orbit"]
    hp, hc, ang, metas = W.sources(cfg, subset)
    unique = len(subset)
    row_src = np.arange(batch) % unique                      # row -> position in the subset
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(orbit, device=dev)
    sel = torch.from_numpy(row_src).to(dev)
    dhp = torch.from_numpy(hp).to(dev)[sel].contiguous()
    dhc = torch.from_numpy(hc).to(dev)[sel].contiguous()
    ang_all = ang[row_src]
    ws = ltdi.Workspace(batch, n, dev)
    for which, gen, fd in runs:
        fd_eff = 0 if which == "full" else fd
        lo, hi = orc80.margins(orbit, gen, order, fd_eff)
        hyb_all = hybrid_params(metas, ltdi.hyb_time, W.TAPER_COSINE, cfg["dt"]) if which == "hybrid" else None
        hyb_g = [hyb_all[i] for i in row_src] if which == "hybrid" else None
        out = run_gpu(ltdi, which, orb, dhp, dhc, ang_all, gen, order, fd, hyb_g, ws)
        full = (batch // unique) * unique
        for c in "AET":
            v = out[c][:full].view(batch // unique, unique, n)
            assert bool((v == v[0:1]).all()), (cfg["name"], which, c, "replicated sources differ across the batch")
            assert bool((out[c][full:] == out[c][:batch - full]).all()), (cfg["name"], which, c, "ragged tail")
            assert bool((out[c][..., :lo] == 0).all()) and bool((out[c][..., n - hi:] == 0).all())
        for s in range(unique):
            got = {c: out[c][s:s + 1].cpu().numpy() for c in "AET"}
            hyb_o = hybrid_params(metas[s:s + 1], orc80.hyb_time, W.TAPER_COSINE, cfg["dt"]) if which == "hybrid" else None
            extra = [*(_hyb_centres(n, metas[s:s + 1], cfg) if which == "hybrid" else ()), int(np.argmax(np.abs(hp[s])))]
            pool = Pooled((cfg["name"], which, gen, fd, "source", subset[s]))
            for nb, ne in windows_of(n, lo, hi, extra, width=1000):
                a = (orbit, hp[s:s + 1], hc[s:s + 1], ang[s:s + 1], gen, order, fd, hyb_o, nb, ne)
                pool.add(got, run_orc(orc80, which, *a), run_orc(orc64, which, *a), nb, ne, lo, n, hi)
            pool.check()


def stratified_sources(orc, k, batch, strata, random=3):
    """the parity subset of a batched config, chosen from the drawn PARAMETERS of all `batch` sources
    (workloads.draw: no series is generated): `strata` sources spread evenly over the chirp-mass order of the whole
    population, both extremes included; the source whose Eq. (2.5) is worst conditioned (smallest min_l (1 - k.n_l));
    plus `random` further ones drawn with a fixed seed."""
    cfg = W.config(k, batch=batch)
    pars = [W.draw(cfg, i) for i in range(batch)]
    order = np.argsort([p["mchirp_s"] for p in pars])
    picks = [int(order[j]) for j in np.unique(np.round(np.linspace(0, batch - 1, strata)).astype(int))]
    cond = [float(np.min(1.0 - orc.antenna(cfg["orbit"], (p["beta"], p["lam"], p["psi"]), cfg["n"] // 2)[:, 2]))
            for p in pars]
    worst = int(np.argmin(cond))
    if worst not in picks:
        picks[len(picks) // 2] = worst
    rng = np.random.default_rng(20250509 + k)
    rest = [i for i in range(batch) if i not in picks]
    picks += [int(i) for i in rng.choice(rest, size=random, replace=False)]
    return picks


def test_config4_full_batch(ltdi, orc80, orc64):
    """B = 4096 x N = 131 072 hybrid TDI 2.0 (8.6 GB in, 12.9 GB out); parity subset: 64 stratified + 3 random"""
    batched_case(ltdi, orc80, orc64, 4, 4096, stratified_sources(orc80, 4, 4096, 64), [("hybrid", 20, 2)])


def test_config5_full_batch(ltdi, orc80, orc64):
    """B = 256 x N = 1 048 576 eccentric, full and LFA TDI 2.0; parity subset: 8 stratified + 3 random"""
    batched_case(ltdi, orc80, orc64, 5, 256, stratified_sources(orc80, 5, 256, 8), [("full", 20, 0), ("lfa", 20, 2)])


def test_config1_full_size_filled(ltdi, orc80, orc64):
    """config 1 (N = 8640, order 9, static arms, TDI 1.5) with the device filled: 4096 sources"""
    batched_case(ltdi, orc80, orc64, 1, 4096, stratified_sources(orc80, 1, 4096, 29), [("full", 15, 0)])
