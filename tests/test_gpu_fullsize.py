"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (reused Workspace,
A / E / T outputs only, same tile plan and source chunking), on sampled windows of the output that the
long-double oracle evaluates one by one through its range arguments (nb, ne), plus properties that hold at
any size (margins exactly zero, replicated sources bitwise equal across chunks of the batch).

Bar per window and channel: relative L2 <= max(1e-11, 3 x the fp64 floor of the oracle's double build on
that window); a near-null channel is measured against the largest channel."""
import numpy as np
import pytest
import torch

import workloads as W
from parity_util import FLOOR_FACTOR, NEAR_NULL, TOL, hybrid_params, record

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ltdi():
    import paper_2505_09600_b200 as m
    assert torch.cuda.is_available(), "GPU parity tests need a CUDA device"
    return m


def windows_of(n, lo, hi, extra=(), width=1500):
    """sample windows [nb, ne): both ends of the valid range (with a piece of margin), the middle, and any
    extra centres (the hybrid window, the merger)"""
    centres = [lo + width // 2 - 40, n // 3, n // 2, n - hi - width // 2 + 40, *extra]
    out = []
    for c in centres:
        nb = int(min(max(c - width // 2, 0), n - width))
        out.append((nb, nb + width))
    return out


def compare_window(got, ref80, ref64, nb, ne, lo, n, hi, label):
    a, b = max(nb, lo), min(ne, n - hi)     # valid part of the window
    norms = {c: np.linalg.norm(ref80[c][:, a - nb:b - nb]) for c in "AET"}
    top = max(norms.values())
    for c in "AET":
        g = got[c][:, nb:ne]
        assert np.all(g[:, :max(0, lo - nb)] == 0.0) and np.all(g[:, max(0, n - hi - nb):] == 0.0), (label, c, "margin")
        if b <= a or top == 0.0:
            continue
        w80, w64 = ref80[c][:, a - nb:b - nb], ref64[c][:, a - nb:b - nb]
        near_null = norms[c] < NEAR_NULL * top
        den = top if near_null else norms[c]
        err = np.linalg.norm(g[:, a - nb:b - nb] - w80) / den
        floor = np.linalg.norm(w64 - w80) / den
        bar = max(TOL, FLOOR_FACTOR * floor)
        record(label=[str(x) for x in label], series=c, window=[int(nb), int(ne)], err=float(err),
               err_vs_top=float(np.linalg.norm(g[:, a - nb:b - nb] - w80) / top), floor=float(floor), bar=float(bar),
               near_null=bool(near_null))
        assert err <= bar, (label, c, (nb, ne), err, bar)


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
        for nb, ne in windows_of(n, lo, hi, extra_centres(n, metas, cfg)):
            r80 = run_orc(orc80, which, orbit, hp, hc, ang, gen, order, fd, hyb_o, nb, ne)
            r64 = run_orc(orc64, which, orbit, hp, hc, ang, gen, order, fd, hyb_o, nb, ne)
            compare_window(got, r80, r64, nb, ne, lo, n, hi, (cfg["name"], which, gen, fd))


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


def batched_case(ltdi, orc80, orc64, k, batch, unique, runs, check_sources):
    """configs 4, 5 at full batch: `unique` distinct seeded sources tiled to `batch` rows (host generation
    of thousands of sources would dominate the test), so that every chunk of the batch the library forms
    is exercised; replicas must be bitwise equal to the first copy, and the first copy matches the oracle."""
    cfg = W.config(k, batch=batch)
    n, order, orbit = cfg["n"], cfg["order"], cfg["orbit"]
    hp, hc, ang, metas = W.sources(cfg, list(range(unique)))
    reps = batch // unique
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(orbit, device=dev)
    dhp = torch.from_numpy(hp).to(dev).repeat(reps, 1)
    dhc = torch.from_numpy(hc).to(dev).repeat(reps, 1)
    ang_all = np.tile(ang, (reps, 1))
    ws = ltdi.Workspace(batch, n, dev)
    for which, gen, fd in runs:
        fd_eff = 0 if which == "full" else fd
        lo, hi = orc80.margins(orbit, gen, order, fd_eff)
        hyb_g = hybrid_params(metas, ltdi.hyb_time, W.TAPER_COSINE, cfg["dt"]) * reps if which == "hybrid" else None
        out = run_gpu(ltdi, which, orb, dhp, dhc, ang_all, gen, order, fd, hyb_g, ws)
        for c in "AET":
            v = out[c].view(reps, unique, n)
            assert bool((v == v[0:1]).all()), (cfg["name"], which, c, "replicated sources differ across the batch")
            assert bool((v[..., :lo] == 0).all()) and bool((v[..., n - hi:] == 0).all())
        for s in check_sources:
            got = {c: out[c][s:s + 1].cpu().numpy() for c in "AET"}
            hyb_o = hybrid_params(metas[s:s + 1], orc80.hyb_time, W.TAPER_COSINE, cfg["dt"]) if which == "hybrid" else None
            extra = _hyb_centres(n, metas[s:s + 1], cfg) if which == "hybrid" else ()
            for nb, ne in windows_of(n, lo, hi, extra, width=1000):
                a = (orbit, hp[s:s + 1], hc[s:s + 1], ang[s:s + 1], gen, order, fd, hyb_o, nb, ne)
                compare_window(got, run_orc(orc80, which, *a), run_orc(orc64, which, *a), nb, ne, lo, n, hi,
                               (cfg["name"], which, "source", s))


def stratified_sources(orc, k, unique):
    """the parity subset holds the chirp-mass extremes and the source whose Eq. (2.5) is worst
    conditioned (smallest min_l (1 - k.n_l)), plus two fixed ones"""
    cfg = W.config(k, batch=unique)
    mc, cond = [], []
    for i in range(unique):
        _, _, ang, meta = W.source(W.config(k, n=16, batch=1), i)     # parameters only: a 16-sample series is cheap
        mc.append(meta["mchirp_s"])
        kn = orc.antenna(cfg["orbit"], ang, cfg["n"] // 2)[:, 2]
        cond.append(float(np.min(1.0 - kn)))
    picks = {int(np.argmin(mc)), int(np.argmax(mc)), int(np.argmin(cond)), 0, unique - 1}
    return sorted(picks)


def test_config4_full_batch(ltdi, orc80, orc64):
    """B = 4096 x N = 131 072 hybrid TDI 2.0 (8.6 GB in, 12.9 GB out)"""
    batched_case(ltdi, orc80, orc64, 4, 4096, 64, [("hybrid", 20, 2)], stratified_sources(orc80, 4, 64))


def test_config5_full_batch(ltdi, orc80, orc64):
    """B = 256 x N = 1 048 576 eccentric, full and LFA TDI 2.0"""
    batched_case(ltdi, orc80, orc64, 5, 256, 2, [("full", 20, 0), ("lfa", 20, 2)], [0, 1])


def test_config1_full_size_filled(ltdi, orc80, orc64):
    """config 1 (N = 8640, order 9, static arms, TDI 1.5) with the device filled: 4096 sources"""
    batched_case(ltdi, orc80, orc64, 1, 4096, 32, [("full", 15, 0)], [0, 31])
