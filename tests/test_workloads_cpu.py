"""Host logic of the seeded input generators (workloads/): the recipe DESIGN.md section 4 states -- sizes of
BASELINE.json's configs, determinism per (seed, source index), frequency content."""
import json
import os

import numpy as np

import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def inst_freq(hp, hc, dt):
    """GW frequency from the phase of h+ - i hx (circular chirps: quadrature pair up to the inclination factors)"""
    ph = np.unwrap(np.arctan2(hc / np.max(np.abs(hc)), hp / np.max(np.abs(hp))))
    return np.abs(np.gradient(ph, dt)) / (2 * np.pi)


def test_config_sizes_are_those_of_baseline_json():
    txt = " ".join(json.load(open(os.path.join(ROOT, "BASELINE.json")))["configs"])
    want = {1: (8640, 10.0, 1, 9), 2: (518400, 5.0, 1, 31), 3: (6307200, 5.0, 1, 31), 4: (131072, 10.0, 4096, 31),
            5: (1048576, 5.0, 256, 31)}
    for k, (n, dt, batch, order) in want.items():
        c = W.config(k)
        assert (c["n"], c["dt"], c["batch"], c["order"]) == (n, dt, batch, order)
        assert f"{n:,}" in txt or str(n) in txt          # the sample counts are the ones BASELINE.json prints
    assert W.config(1)["mode"] == W.ORBIT_STATIC_EQUALARM and W.config(2)["mode"] == W.ORBIT_KEPLERIAN


def test_sources_are_deterministic_and_independent_of_the_batch_they_are_drawn_in():
    cfg = W.config(4, n=4096, batch=8)
    a = W.sources(cfg, [5, 2, 7])
    b = W.sources(cfg, [2])
    c = W.sources(cfg, [5, 2, 7])
    assert np.array_equal(a[0], c[0]) and np.array_equal(a[1], c[1]) and np.array_equal(a[2], c[2])
    assert np.array_equal(a[0][1], b[0][0]) and np.array_equal(a[2][1], b[2][0])
    assert not np.array_equal(a[0][0], a[0][1])
    for arr in a[:3]:
        assert np.all(np.isfinite(arr))


def test_config1_and_config3_chirps_sweep_the_stated_bands():
    # DESIGN.md section 4 / SURVEY 8(d): cfg1 f_gw 2.8e-4 -> 3.2e-4 Hz; cfg3 2.35e-4 -> 3.05e-4 Hz
    cfg = W.config(1)
    hp, hc, _, _ = W.source(cfg, 0)
    f = inst_freq(hp, hc, cfg["dt"])
    assert 2.6e-4 < np.median(f[:200]) < 3.0e-4 and 3.0e-4 < np.median(f[-200:]) < 3.4e-4
    cfg = W.config(3, n=6307200)
    hp, hc, _, _ = W.source(cfg, 0)
    f0 = inst_freq(hp[:4000], hc[:4000], cfg["dt"])
    f1 = inst_freq(hp[-4000:], hc[-4000:], cfg["dt"])
    assert 2.2e-4 < np.median(f0) < 2.5e-4 and 2.9e-4 < np.median(f1) < 3.2e-4


def test_config2_and_config4_mergers_lie_where_the_recipe_puts_them():
    cfg = W.config(2)
    hp, hc, _, meta = W.source(cfg, 0)
    t_end = cfg["orbit"]["t0"] + cfg["n"] * cfg["dt"]
    peak = np.argmax(hp ** 2 + hc ** 2) * cfg["dt"]
    assert 0.4 * 3600 < t_end - peak < 2.2 * 3600            # merger 0.5-2 h before the end, ringdown after it
    assert abs(hp[-1]) < 1e-3 * np.max(np.abs(hp))           # the ringdown has died out
    cfg = W.config(4)
    for i in range(6):
        hp, hc, _, meta = W.source(cfg, i)
        frac = np.argmax(hp ** 2 + hc ** 2) / cfg["n"]
        assert 0.88 < frac <= 1.0                            # merger in the last 10 % of the segment
        assert meta["f_hyb_hz"] == 2.0e-3 and meta["window_s"] == 3600.0 and meta["taper"] == W.TAPER_COSINE


def test_config5_eccentric_sources_reach_the_millihertz_band():
    cfg = W.config(5, n=32768)          # the last 32 768 samples carry the loudest, fastest part
    full = W.config(5)
    for i in range(2):
        rng_cfg = dict(cfg)
        hp, hc, _, _ = W.source(rng_cfg, i)
        assert np.all(np.isfinite(hp)) and np.all(np.isfinite(hc)) and np.max(np.abs(hp)) > 0
        spec = np.abs(np.fft.rfft(hp * np.hanning(len(hp))))
        fpk = np.argmax(spec[1:]) / (len(hp) * cfg["dt"])
        assert 2e-4 < fpk < 5e-2                             # harmonics between 0.2 and 50 mHz, below Nyquist (0.1 Hz)
    assert full["n"] == 1048576
