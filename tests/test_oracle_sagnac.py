"""Pins of oracle O15 (no GPU): the Sagnac combinations alpha, beta, gamma of SURVEY 8(f)-4 (reading G33).

Checked against what time-delay interferometry fixes, not against the oracle: laser frequency noise cancels in the
6-term combination exactly when the two round trips take the same time and in the 12-term one for any constant
L_l != L_-l; single samples re-evaluated with independent Python code; the operator identity that ties the sum
alpha + beta + gamma to X + Y + Z (pinned separately) for equal arms.
"""
import numpy as np
import pytest

import workloads as W

SENDER = [2, 0, 1, 1, 2, 0]     # links +1, +2, +3, -1, -2, -3
RECEIVER = [1, 2, 0, 2, 0, 1]
IDX = {+1: 0, +2: 1, +3: 2, -1: 3, -2: 4, -3: 5}


def static_tables(n, dt, t0, L0):
    """TABLES-mode orbit with constant light times L0 [6] (seconds)"""
    base = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN, t0=t0)
    from oracle import Oracle
    R, _, _ = Oracle("f64").orbit_tables(base)
    L = np.repeat(np.asarray(L0, dtype=np.float64)[:, None], n, axis=1)
    return dict(base, mode=W.ORBIT_TABLES, R_table=np.ascontiguousarray(R), L_table=np.ascontiguousarray(L))


def laser_links(t, L0, freqs, amps):
    """y_l(t) = p_s(t - L_l) - p_r(t): the laser-noise content of the single-link measurements"""
    def p(i, x):
        return sum(a * np.sin(2 * np.pi * f * x + 0.7 * i + k) for k, (f, a) in enumerate(zip(freqs[i], amps[i])))
    return np.array([p(SENDER[l], t - L0[l]) - p(RECEIVER[l], t) for l in range(6)])


FREQS = [[1.1e-3, 2.3e-3], [0.7e-3, 3.1e-3], [1.9e-3, 2.9e-3]]
AMPS = [[1.0, 0.4], [0.8, 0.5], [0.6, 0.7]]


def test_laser_noise_cancels_when_the_round_trips_agree(orc80):
    """L_l = L_-l, three unequal arms: T+ = T-, the 6-term alpha, beta, gamma are free of laser noise"""
    n, dt, t0 = 4000, 5.0, 3.0e5
    L0 = [8.30, 9.36, 7.27, 8.30, 9.36, 7.27]
    orbit = static_tables(n, dt, t0, L0)
    t = t0 + dt * np.arange(n)
    y = laser_links(t, L0, FREQS, AMPS)
    lo, hi = orc80.margins(orbit, 15, 31, 0)
    for gen in (15, 20):
        abc = orc80.sagnac_from_links(orbit, y, gen, 31)[:, lo:n - hi]
        assert np.abs(abc).max() < 2e-11, gen          # links are O(1), their phases (6e3 rad) carry 1e-12 of fp64 rounding
    # and the valid range is not empty or trivially zero for a signal that is not laser noise
    y2 = y.copy()
    y2[2] += np.sin(2 * np.pi * 2e-3 * t)
    assert np.abs(orc80.sagnac_from_links(orbit, y2, 15, 31)[:, lo:n - hi]).max() > 0.5


def test_sagnac_effect_needs_the_twelve_terms(orc80):
    """L_l != L_-l (the rotation of the constellation): T+ - T- = 4.5e-2 s here.  The 6-term combination keeps
    p_1(t - T+) - p_1(t - T-) ~ omega (T+ - T-); the 12-term one cancels it"""
    n, dt, t0 = 4000, 5.0, 3.0e5
    L0 = [8.30, 9.36, 7.27, 8.31, 9.38, 7.285]
    orbit = static_tables(n, dt, t0, L0)
    t = t0 + dt * np.arange(n)
    y = laser_links(t, L0, FREQS, AMPS)
    lo, hi = orc80.margins(orbit, 20, 31, 0)
    six = orc80.sagnac_from_links(orbit, y, 15, 31)[:, lo:n - hi]
    twelve = orc80.sagnac_from_links(orbit, y, 20, 31)[:, lo:n - hi]
    dT = sum(L0[:3]) - sum(L0[3:])
    # the residual of alpha is that of laser 1 alone, in closed form
    p1 = lambda x: sum(a * np.sin(2 * np.pi * f * x + k) for k, (f, a) in enumerate(zip(FREQS[0], AMPS[0])))
    want = p1(t - sum(L0[:3])) - p1(t - sum(L0[3:]))
    assert np.abs(six[0] - want[lo:n - hi]).max() < 2e-11
    assert np.abs(six).max() > 0.5 * 2 * np.pi * 1e-3 * abs(dT)
    assert np.abs(twelve).max() < 2e-11


def test_single_samples_by_brute_force(orc80):
    """alpha, beta, gamma at a few samples from analytic link series evaluated at the exact retarded times, with the beams
    walked round the triangle by spacecraft number (not by the oracle's link labels)"""
    n, dt, t0 = 2500, 5.0, 2.0e5
    L0 = [8.30, 9.36, 7.27, 8.31, 9.38, 7.285]
    orbit = static_tables(n, dt, t0, L0)
    t = t0 + dt * np.arange(n)
    fl = [1.3e-3, 2.1e-3, 0.9e-3, 1.7e-3, 2.6e-3, 0.6e-3]
    ylink = lambda l, x: np.sin(2 * np.pi * fl[l] * x + 0.3 * l)
    y = np.array([ylink(l, t) for l in range(6)])
    link_of = {(SENDER[l], RECEIVER[l]): l for l in range(6)}     # (sender, receiver) -> row

    def beam(x, route):
        """sum of the link measurements met by the beam that arrives at route[-1] at time x, having gone round `route`"""
        total = 0.0
        for k in range(len(route) - 1, 0, -1):
            l = link_of[(route[k - 1], route[k])]
            total += ylink(l, x)
            x = x - L0[l]
        return total, x

    for gen in (15, 20):
        got = orc80.sagnac_from_links(orbit, y, gen, 31)
        for ns in (600, 1234, 2100):
            for ch in range(3):
                s1 = ch
                s2, s3 = (ch + 1) % 3, (ch + 2) % 3
                plus, xp = beam(t[ns], [s1, s3, s2, s1])      # 1 -> 3 -> 2 -> 1
                minus, xm = beam(t[ns], [s1, s2, s3, s1])     # 1 -> 2 -> 3 -> 1
                want = plus - minus
                if gen == 20:
                    want += beam(xp, [s1, s2, s3, s1])[0] - beam(xm, [s1, s3, s2, s1])[0]
                assert abs(got[ch, ns] - want) < 2e-11, (gen, ns, ch, got[ch, ns], want)


def test_sum_identity_with_the_michelson_variables(orc80):
    """equal arms of exactly 2 samples (D is a shift, no interpolation error): for ANY link data
    (1 - D^2)(1 - D)(alpha + beta + gamma) = -(1 + D + D^2)(X + Y + Z)   [6-term alpha, X_1.5],
    alpha_2 = (1 - D^3) alpha_1"""
    n, dt, t0 = 600, 5.0, 0.0
    orbit = static_tables(n, dt, t0, [10.0] * 6)
    rng = np.random.default_rng(11)
    y = rng.normal(size=(6, n))
    lo, hi = orc80.margins(orbit, 20, 31, 0)
    y[:, :lo] = 0.0
    sa = orc80.sagnac_from_links(orbit, y, 15, 31)
    sx = orc80.michelson_from_links(orbit, y, 15, 31)
    D = lambda v, k=1: np.concatenate([np.zeros(2 * k), v[:-2 * k]])
    a, x = sa.sum(axis=0), sx.sum(axis=0)
    lhs = a - D(a) - D(a, 2) + D(a, 3)               # (1 - D^2)(1 - D) = 1 - D - D^2 + D^3
    rhs = -(x + D(x) + D(x, 2))
    lo15, _ = orc80.margins(orbit, 15, 31, 0)
    sl = slice(lo15 + 8, n - hi)
    assert np.abs(x[sl]).max() > 1.0
    assert np.abs(lhs - rhs)[sl].max() < 1e-13
    s2 = orc80.sagnac_from_links(orbit, y, 20, 31)
    for c in range(3):
        assert np.abs(s2[c] - (sa[c] - D(sa[c], 3)))[lo + 8:n - hi].max() < 1e-13


def test_margin_samples_are_never_read_and_full_response_plumbing(orc80):
    """sentinels in the margins of y leave every valid output unchanged; the full response puts alpha, beta, gamma where
    X, Y, Z go and applies Eq. (2.9) to them"""
    cfg = W.config(2, n=6001)
    hp, hc, ang, _ = W.source(cfg, 0)
    orbit = cfg["orbit"]
    for gen in (15, 20):
        out = orc80.response_full_sagnac(orbit, hp, hc, ang, gen, 31)
        y = out["y"][:, 0]
        abc = orc80.sagnac_from_links(orbit, y, gen, 31)
        assert np.abs(abc - out["XYZ"][:, 0]).max() < 1e-15 * np.abs(y).max()    # y went through fp64 on the way
        a, b, c = out["XYZ"][:, 0]
        assert np.allclose(out["A"][0], (c - a) / np.sqrt(2), rtol=0, atol=1e-15 * np.abs(a).max())
        assert np.allclose(out["E"][0], (a - 2 * b + c) / np.sqrt(6), rtol=0, atol=1e-15 * np.abs(a).max())
        assert np.allclose(out["T"][0], (a + b + c) / np.sqrt(3), rtol=0, atol=1e-15 * np.abs(a).max())
        lo, hi = orc80.margins(orbit, gen, 31, 0)
        ys = y.copy()
        first = np.argmax(np.abs(y).sum(axis=0) > 0)          # the link margin: y is exactly 0 there
        ys[:, :first] = 1e30
        abc2 = orc80.sagnac_from_links(orbit, ys, gen, 31)
        assert np.array_equal(abc2[:, lo:cfg["n"] - hi], abc[:, lo:cfg["n"] - hi])
        assert np.abs(abc[:, lo:cfg["n"] - hi]).max() > 0
