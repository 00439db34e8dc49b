"""Pins of O14 (no GPU): the six-link LFA and the Michelson variables Taylor-expanded without the
link-reversal symmetry, Eq. (B20) P:832 (TDI 1.5) and Eq. (B30) P:894 (TDI 2.0) at the mid-points (B18) / (B31).

Checked against the exact Michelson combination of the SAME link series (already pinned, O6): for six unrelated
smooth link series and six unequal delays the expansion must agree with Eq. (2.7) / (2.8) up to its next order,
a residual that falls as f^2 -- a wrong sign, prefactor or mid-point leaves a first-order residual instead; and
against Eq. (B25) / (B33) where the symmetry holds exactly (constant equal arms)."""
import numpy as np
import pytest

import workloads as W


def unequal_tables(n, dt, t0=1.0e6):
    base = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN, t0=t0)
    from oracle import Oracle
    R, _, _ = Oracle("f64").orbit_tables(base)
    L0 = np.array([8.3, 9.3, 7.2, 7.5, 9.9, 6.9])   # grossly unequal, so that a wrong light time anywhere shows at first order
    L = np.repeat(L0[:, None], n, axis=1)
    return dict(base, mode=W.ORBIT_TABLES, R_table=np.ascontiguousarray(R), L_table=np.ascontiguousarray(L))


def six_links(t, f0):
    fl = f0 * np.array([1.00, 0.83, 1.21, 0.92, 1.13, 0.77])
    return np.array([(1.0 + 0.2 * l) * np.sin(2 * np.pi * fl[l] * t + 0.9 * l) for l in range(6)])


@pytest.mark.parametrize("gen", [15, 20])
def test_expansion_agrees_with_the_exact_combination_to_second_order(orc80, gen):
    n, dt = 6000, 5.0
    orbit = unequal_tables(n, dt)
    t = orbit["t0"] + dt * np.arange(n)
    lo, hi = orc80.margins(orbit, gen, 31, 4)
    sl = slice(lo + 2, n - hi - 2)
    res = []
    for f0 in (4e-4, 2e-4):
        y = six_links(t, f0)
        exact = orc80.michelson_from_links(orbit, y, gen, 31)[:, sl]
        b20 = orc80.michelson_b20_from_links(orbit, y, gen, 31, 4)[:, sl]
        res.append(np.linalg.norm(b20 - exact) / np.linalg.norm(exact))
    omega_L = 2 * np.pi * 4e-4 * 8.3
    assert res[0] < 3.0 * omega_L ** 2, res              # next order of the Taylor series, not first order (omega L = 0.02)
    assert 3.2 < res[0] / res[1] < 4.8, res              # ... and it falls as f^2


@pytest.mark.parametrize("gen,fd", [(15, 2), (20, 2), (20, 4)])
def test_equal_constant_arms_reduce_to_the_symmetric_lfa(orc80, gen, fd):
    """y_slr = y_r-ls and L_l = L_-l exactly: the second- (third-) derivative terms cancel pairwise and (B20) / (B30)
    become (B25) / (B33) -- prefactors and the retarded times of (B18) / (B31) against (B25) / (B33)"""
    cfg = W.config(1)
    hp, hc, ang, _ = W.sources(cfg, [0])
    orbit = cfg["orbit"]
    a = orc80.response_lfa6(orbit, hp, hc, ang, gen, 9, fd)
    b = orc80.response_lfa(orbit, hp, hc, ang, gen, 9, fd)
    lo, hi = orc80.margins_lfa6(orbit, gen, 9, fd)
    sl = slice(lo, cfg["n"] - hi)
    assert np.array_equal(a["y"][3:], a["y"][:3])         # the reversed links are the same series
    assert np.array_equal(a["y"][:3], b["y"][:3])
    top = np.abs(b["XYZ"][..., sl]).max()
    assert np.abs(a["XYZ"] - b["XYZ"])[..., sl].max() <= 1e-12 * top
    assert (lo, hi) == tuple(x + (gen == 20) for x in orc80.margins(orbit, gen, 9, fd))


def test_reversed_links_on_the_rotating_constellation(orc80):
    """L_-l != L_l at the 1e-4 level (Sagnac): the reversed link is the same waveform scaled by L_-l / L_l and shifted by
    (L_-l - L_l) / 2 -- Eq. (B24) P:857"""
    cfg = W.config(2, n=12000)
    hp, hc, ang, _ = W.sources(cfg, [0])
    orbit = cfg["orbit"]
    out = orc80.response_lfa6(orbit, hp, hc, ang, 15, 31, 2)
    _, _, L = orc80.orbit_tables(orbit)
    lo, hi = orc80.link_margins(orbit, 31, 2)
    sl = slice(lo + 4, 9000)                               # the inspiral part
    for l in range(3):
        yp, ym = out["y"][l, 0, sl], out["y"][3 + l, 0, sl]
        ratio = np.linalg.norm(ym) / np.linalg.norm(yp)
        assert abs(ratio - np.mean(L[3 + l, sl] / L[l, sl])) < 2e-6
        d = np.linalg.norm(ym - yp) / np.linalg.norm(yp)
        assert 1e-6 < d < 1e-3


def test_b20_against_the_full_response(orc80):
    """on the moving constellation the expansion without the symmetry is at least as close to the full response as (B25)"""
    cfg = W.config(3, n=20000)
    hp, hc, ang, _ = W.sources(cfg, [0])
    orbit = cfg["orbit"]
    full = orc80.response_full(orbit, hp, hc, ang, 15, 31, want=("XYZ",))
    lfa = orc80.response_lfa(orbit, hp, hc, ang, 15, 31, 4, want=("XYZ",))
    b20 = orc80.response_lfa6(orbit, hp, hc, ang, 15, 31, 4, want=("XYZ",))
    lo, hi = orc80.margins_lfa6(orbit, 15, 31, 4)
    sl = slice(lo, cfg["n"] - hi)
    nrm = np.linalg.norm(full["XYZ"][..., sl])
    r_lfa = np.linalg.norm((lfa["XYZ"] - full["XYZ"])[..., sl]) / nrm
    r_b20 = np.linalg.norm((b20["XYZ"] - full["XYZ"])[..., sl]) / nrm
    assert r_b20 < 1e-3 and r_b20 <= 1.05 * r_lfa, (r_b20, r_lfa)
