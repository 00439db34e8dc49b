"""GPU parity of the first "next" row: noise PSD kernel, the hand-written FFT (Stockham / Bluestein) + inner-product kernels against
the numpy oracle (oracle/overlap_oracle.py) on the same inputs.

Tolerances: PSD 1e-12 relative away from its zeros (libm differences of a few ulp, amplified by
1 / tan x within 0.05 of a zero of sin x); inner products 1e-11 relative (the two
FFTs differ by O(log N) ulp per bin, the sums run over up to 5e5 bins in different orders); overlap and mismatch
1e-12 absolute."""
import numpy as np
import pytest
import torch

import workloads as W
from oracle import overlap_oracle as oo
from parity_util import hybrid_params

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(scope="module")
def ltdi():
    import paper_2505_09600_b200 as m
    assert torch.cuda.is_available(), "GPU parity tests need a CUDA device"
    return m


@pytest.mark.parametrize("gen", [15, 20])
@pytest.mark.parametrize("galactic", [False, True])
def test_noise_psd_kernel(ltdi, gen, galactic):
    n, dt = 100001, 5.0
    ov = ltdi.Overlap(n, n, 1, DEV)
    got = ov.psd(dt, gen, galactic=galactic, t_obs_yr=2.5).cpu().numpy()
    f = np.arange(n // 2 + 1) / (n * dt)
    want = np.stack(oo.psd_aet(f[1:], gen, 2.5e9, 2.5, galactic))
    assert np.all(np.isinf(got[:, 0]))
    rel = np.abs(got[:, 1:] / want - 1.0)
    # the PSD vanishes with sin x (and sin 2x for TDI 2.0): next to those zeros one rounding of x moves it by
    # eps x / tan x, so the relative bar applies away from them and a looser one everywhere
    x = 2 * np.pi * f[1:] * 2.5e9 / 299792458.0
    away = (np.abs(np.sin(x)) > 0.05) & (np.abs(np.sin(2 * x)) > 0.05)
    assert np.max(rel[:, away]) < 1e-12
    assert np.max(rel) < 1e-8


def compare(got, snr, want):
    got, snr = got.cpu().numpy(), snr.cpu().numpy()
    assert np.max(np.abs(got[:, :, :3] / want[:, :, :3] - 1.0)) < 1e-11
    assert np.max(np.abs(got[:, :, 3:] - want[:, :, 3:])) < 1e-12
    assert np.max(np.abs(snr[:, 0] / oo.snr(want[:, :, 0]) - 1.0)) < 1e-11
    assert np.max(np.abs(snr[:, 1] / oo.snr(want[:, :, 1]) - 1.0)) < 1e-11
    # ln L of (D4) is a difference of the products: judged against their size
    scale = np.sum(want[:, :, 0] + want[:, :, 1], axis=-1)
    assert np.max(np.abs(snr[:, 2] - oo.log_likelihood(want)) / scale) < 1e-11


@pytest.mark.parametrize("gen", [15, 20])
def test_products_of_full_and_hybrid_small(ltdi, gen):
    """three sources of config 2 (40 007 samples, not a power of two), padded rows (ld > n)"""
    cfg = W.config(2, n=40007, batch=3)
    hp, hc, ang, metas = W.sources(cfg, [0, 1, 2])
    n, dt, ld = cfg["n"], cfg["dt"], cfg["n"] + 9
    pad = np.zeros((3, 9))
    dhp = torch.from_numpy(np.concatenate([hp, pad], 1)).to(DEV)
    dhc = torch.from_numpy(np.concatenate([hc, pad], 1)).to(DEV)
    orb = ltdi.Orbits(cfg["orbit"], device=DEV)
    full = {k: v.clone() for k, v in ltdi.response_full(orb, dhp, dhc, ang, gen, 31).items() if k in "AET"}
    hyb = {k: v.clone() for k, v in ltdi.response_hybrid(orb, dhp, dhc, ang, gen, 31, 2,
                                                        hybrid_params(metas, ltdi.hyb_time, W.TAPER_COSINE, dt)).items()
           if k in "AET"}
    for d in (full, hyb):          # the columns beyond n are not part of the series
        for k in d:
            d[k][:, n:] = 7.0
    ov = ltdi.Overlap(n, ld, 3, DEV)
    out, snr = ov.products(full, hyb, dt, ov.psd(dt, gen), 1e-4, 2e-2)
    torch.cuda.synchronize()
    a = {k: v[:, :n].cpu().numpy() for k, v in full.items()}
    b = {k: v[:, :n].cpu().numpy() for k, v in hyb.items()}
    compare(out, snr, oo.products(a, b, dt, gen, 1e-4, 2e-2))


def test_config2_full_size_reproduces_the_paper_accuracy_statements(ltdi):
    """N = 518 400: GPU responses -> GPU overlap; parity with the oracle's overlap of the same series, and the paper's
    statements: hybrid mismatch < 1e-5 (A, E), LFA < 10 % (TDI 2.0, A, E)"""
    cfg = W.config(2)
    hp, hc, ang, metas = W.sources(cfg, [0])
    n, dt = cfg["n"], cfg["dt"]
    dhp, dhc = torch.from_numpy(hp).to(DEV), torch.from_numpy(hc).to(DEV)
    orb = ltdi.Orbits(cfg["orbit"], device=DEV).prepare(20, 31)
    keep = lambda d: {k: v.clone() for k, v in d.items() if k in "AET"}
    full = keep(ltdi.response_full(orb, dhp, dhc, ang, 20, 31))
    lfa = keep(ltdi.response_lfa(orb, dhp, dhc, ang, 20, 31, 2))
    hyb = keep(ltdi.response_hybrid(orb, dhp, dhc, ang, 20, 31, 2, hybrid_params(metas, ltdi.hyb_time, W.TAPER_COSINE, dt)))
    ov = ltdi.Overlap(n, n, 1, DEV)
    psd = ov.psd(dt, 20)
    cpu = lambda d: {k: v.cpu().numpy() for k, v in d.items()}
    out, snr = ov.products(full, hyb, dt, psd, 1e-4, 2e-2)
    got_h = out.clone()
    compare(out, snr, oo.products(cpu(full), cpu(hyb), dt, 20, 1e-4, 2e-2))
    out, snr = ov.products(full, lfa, dt, psd, 1e-4, 2e-2)
    compare(out, snr, oo.products(cpu(full), cpu(lfa), dt, 20, 1e-4, 2e-2))
    assert float(got_h[0, 0, 4]) < 1e-5 and float(got_h[0, 1, 4]) < 1e-5
    assert float(out[0, 0, 4]) < 1e-1 and float(out[0, 1, 4]) < 1e-1
    assert 100.0 < float(snr[0, 0]) < 1e4


def test_batch_in_several_passes_with_a_tail(ltdi):
    """23 series of 2^20 + 2 samples: the spectra of a pass are capped at 1 GiB, so the batch runs as 21 + 2"""
    n, dt, batch = (1 << 20) + 2, 5.0, 23
    rng = np.random.default_rng(8)
    t = dt * np.arange(n)
    a, b = {}, {}
    for i, c in enumerate("AET"):
        f0 = 1e-3 * (1 + i) * (1.0 + 0.1 * np.arange(batch))[:, None]
        x = 1e-21 * np.sin(2 * np.pi * f0 * t[None] * (1 + 2e-8 * t[None])) * np.hanning(n)[None]
        a[c] = x
        b[c] = x * (1.0 + 1e-3 * i) + 1e-24 * rng.standard_normal((batch, n))
    ov = ltdi.Overlap(n, n, batch, DEV)
    da = {c: torch.from_numpy(v).to(DEV) for c, v in a.items()}
    db = {c: torch.from_numpy(v).to(DEV) for c, v in b.items()}
    out, snr = ov.products(da, db, dt, ov.psd(dt, 15, galactic=False), 2e-4, 1.5e-2)
    torch.cuda.synchronize()
    compare(out, snr, oo.products(a, b, dt, 15, 2e-4, 1.5e-2, galactic=False))


def test_overlap_argument_errors(ltdi):
    ov = ltdi.Overlap(1000, 1000, 1, DEV)
    x = {c: torch.zeros(1, 1000, dtype=torch.float64, device=DEV) for c in "AET"}
    psd = ov.psd(5.0, 20)
    with pytest.raises(ltdi.LtdiError):
        ov.products(x, x, -1.0, psd, 1e-4, 1e-2)
    with pytest.raises(ltdi.LtdiError):
        ov.products(x, x, 5.0, psd, 1e-2, 1e-4)
    with pytest.raises(ltdi.LtdiError):
        ltdi.Overlap(1000, 999, 1, DEV)
    with pytest.raises(ltdi.LtdiError):
        ov.psd(5.0, 17)
