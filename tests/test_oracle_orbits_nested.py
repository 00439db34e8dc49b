"""Pins of the oracle parts of SURVEY 8(f)-4 (no GPU): O11 numerical orbits from tabulated knots, O12 nested TDI delays.

Each check is against something other than the oracle: polynomial trajectories (the interpolant and its derivative
are exact), the analytic orbit of O1 sampled at the knots, the textbook property of time-delay interferometry --
laser frequency noise cancels, for linearly breathing unequal arms, in the second-generation combination with properly
nested delays and not otherwise --, and a brute-force re-evaluation of single samples with independent Python code.
"""
import numpy as np
import pytest

import workloads as W

C = 299792458.0
SENDER = [2, 0, 1, 1, 2, 0]     # links +1, +2, +3, -1, -2, -3
RECEIVER = [1, 2, 0, 2, 0, 1]


def knots_orbit(n, dt, t0, knots, tk0, dtk, order):
    d = W.orbit_desc(n, dt, W.ORBIT_KNOTS, t0=t0)
    d.update(knots=np.ascontiguousarray(knots), knot_t0=float(tk0), knot_dt=float(dtk), knot_order=int(order))
    return d


# ------------------------------------------------------------------ O11 numerical orbits
@pytest.mark.parametrize("order", [3, 7])
def test_knots_polynomial_trajectory_is_exact(orc80, order):
    """positions AND the velocities that enter L_l = (|d| / c)(1 + n.V_s / c) are exact for a polynomial orbit of degree <= p"""
    rng = np.random.default_rng(order)
    dtk, tk0, nk = 1000.0, -8000.0, 40
    tk = tk0 + dtk * np.arange(nk)
    coef = rng.normal(size=(3, 3, order + 1))
    scale = np.array([1.5e11, 2.0e9, 3.0e4, 2.0e-1] + [1e-6 ** k for k in range(1, order)])[:order + 1]

    def traj(t, der=0):
        s = t / 1.0e4
        out = np.zeros((3, 3) + np.shape(t))
        for k in range(der, order + 1):
            fac = np.prod(np.arange(k, k - der, -1)) if der else 1.0
            out += (coef[..., k] * scale[k] * fac)[..., None] * s ** (k - der) / 1.0e4 ** der
        return out

    n, dt, t0 = 257, 37.0, 1234.5
    orbit = knots_orbit(n, dt, t0, traj(tk), tk0, dtk, order)
    R, nh, L = orc80.orbit_tables(orbit)
    t = t0 + dt * np.arange(n)
    Rw, Vw = traj(t), traj(t, 1)
    assert np.abs(R - Rw).max() <= 1e-15 * np.abs(Rw).max() * 40
    for l in range(6):
        d = Rw[RECEIVER[l]] - Rw[SENDER[l]]
        ln = np.linalg.norm(d, axis=0)
        want = ln / C * (1.0 + np.sum(d / ln * Vw[SENDER[l]], axis=0) / C)
        assert np.abs(L[l] - want).max() <= 1e-13 * want.max(), l
        assert np.abs(nh[l] - d / ln).max() <= 1e-12


def test_knots_reproduce_the_analytic_orbit(orc80):
    """knots sampled from O1 (first-order Keplerian, daily) -> positions, link vectors and light times of O1 at the
    sample times, to the interpolation error of order 7 over one-day knots ((Omega dt_k)^8 R ~ 1e-3 m)"""
    n, dt, t0, dtk = 4001, 5.0, 2.0e6 + 123.0, 86400.0
    nk = 20
    tk0 = np.floor(t0 / dtk) * dtk - 6 * dtk
    kep_knots = W.orbit_desc(nk, dtk, W.ORBIT_KEPLERIAN, t0=tk0, alpha0=0.4, rot0=0.9)
    Rk, _, _ = orc80.orbit_tables(kep_knots)
    orbit = knots_orbit(n, dt, t0, Rk, tk0, dtk, 7)
    orbit.update(alpha0=0.4, rot0=0.9)
    R, nh, L = orc80.orbit_tables(orbit)
    kep = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN, t0=t0, alpha0=0.4, rot0=0.9)
    R0, nh0, L0 = orc80.orbit_tables(kep)
    assert np.abs(R - R0).max() < 5e-3                      # metres, at 1.5e11
    assert np.abs(nh - nh0).max() < 1e-11
    assert np.abs(L - L0).max() < 1e-11 * L0.max()
    # and the Sagnac asymmetry L_l - L_-l comes out of the interpolant's velocity
    assert np.abs((L[:3] - L[3:]) - (L0[:3] - L0[3:])).max() < 1e-11


def test_sample_on_a_knot_is_the_knot(orc80):
    rng = np.random.default_rng(5)
    knots = 1.5e11 * rng.normal(size=(3, 3, 24))
    orbit = knots_orbit(12, 500.0, 4000.0, knots, -2000.0, 1000.0, 7)   # t_n = 4000 + 500 n: every second sample on a knot
    R, _, _ = orc80.orbit_tables(orbit)
    assert np.array_equal(R[..., ::2], knots[..., 6:12])


def test_numerical_orbit_file_is_esa_like():
    """the synthetic orbit file: arms within 1 % of 2.5e9 m, unequal at the per-mille level, breathing at metres per second"""
    orb = W.numerical_orbit(1000, 5.0, t0=1.0e7)
    K = orb["knots"]
    arms = np.array([np.linalg.norm(K[r] - K[s], axis=0) for s, r in ((2, 1), (0, 2), (1, 0))])
    assert np.all(np.abs(arms / 2.5e9 - 1.0) < 0.012)
    assert np.abs(arms[0] - arms[1]).max() > 1e-3 * 2.5e9
    rate = np.abs(np.diff(arms, axis=1)).max() / orb["knot_dt"]
    assert 0.5 < rate < 15.0                                 # the paper quotes dL/dt < 12 m/s for realistic orbits


# ------------------------------------------------------------------ O12 nested delays
def breathing_tables(n, dt, t0, rates):
    """TABLES-mode orbit whose light times are L_l(t) = L0_l + rate_l t: unequal, linearly breathing arms"""
    base = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN, t0=t0)
    from oracle import Oracle
    R, _, _ = Oracle("f64").orbit_tables(base)
    t = t0 + dt * np.arange(n)
    L0 = np.array([8.30, 8.36, 8.27, 8.301, 8.362, 8.268])
    L = L0[:, None] + np.asarray(rates)[:, None] * t[None, :]
    return dict(base, mode=W.ORBIT_TABLES, R_table=np.ascontiguousarray(R), L_table=np.ascontiguousarray(L)), L0


def laser_links(t, L, freqs, amps):
    """y_l(t) = p_s(t - L_l(t)) - p_r(t): the laser-noise content of the single-link measurements (textbook TDI)"""
    def p(i, x):
        return sum(a * np.sin(2 * np.pi * f * x + 0.7 * i + k) for k, (f, a) in enumerate(zip(freqs[i], amps[i])))
    return np.array([p(SENDER[l], t - L[l]) - p(RECEIVER[l], t) for l in range(6)])


def test_nested_equals_unnested_for_constant_delays(orc80):
    n, dt = 3000, 5.0
    orbit = W.orbit_desc(n, dt, W.ORBIT_STATIC_EQUALARM, t0=1.0e6)
    rng = np.random.default_rng(3)
    t = dt * np.arange(n)
    y = np.array([np.sin(2 * np.pi * 2e-3 * t * (1 + 0.1 * l) + l) for l in range(6)]) + 1e-3 * rng.normal(size=(6, n))
    for gen in (15, 20):
        a = orc80.michelson_from_links(orbit, y, gen, 31)
        b = orc80.michelson_nested_from_links(orbit, y, gen, 31, 3)
        assert np.abs(a - b).max() <= 1e-14 * np.abs(a).max()


def test_laser_noise_cancels_only_with_nested_second_generation(orc80):
    """Linearly breathing unequal arms (30 m/s, ten times LISA's, so that the effect stands clear of everything else):
    X_2.0 with nested delays cancels the laser noise to second order in dL/dt; with every L_l evaluated at t (the paper's
    choice for the GW response) a first-order residual omega L dL/dt remains, and X_1.5 keeps one too."""
    n, dt, t0 = 6000, 5.0, 5.0e5
    rates = np.array([1.0, -0.7, 0.5, 1.0, -0.7, 0.5]) * 1.0e-7
    orbit, _ = breathing_tables(n, dt, t0, rates)
    t = t0 + dt * np.arange(n)
    freqs = [[1.1e-3, 2.3e-3], [0.7e-3, 3.1e-3], [1.9e-3, 2.9e-3]]
    amps = [[1.0, 0.4], [0.8, 0.5], [0.6, 0.7]]
    y = laser_links(t, orbit["L_table"], freqs, amps)
    lo, hi = orc80.margins(orbit, 20, 31, 0)
    sl = slice(lo, n - hi)
    nested20 = orc80.michelson_nested_from_links(orbit, y, 20, 31, 3)[:, sl]
    plain20 = orc80.michelson_from_links(orbit, y, 20, 31)[:, sl]
    nested15 = orc80.michelson_nested_from_links(orbit, y, 15, 31, 3)[:, sl]
    first_order = 2 * np.pi * 3e-3 * 8.3 * 1e-7          # omega L dL/dt: the scale of a first-order residual
    assert np.abs(nested20).max() < 1e-3 * first_order     # second order (and interpolation error) only
    assert np.abs(plain20).max() > 0.5 * first_order
    assert np.abs(nested15).max() > 0.5 * first_order
    # each of X, Y, Z on its own
    assert all(np.abs(nested20[c]).max() < 1e-3 * np.abs(plain20[c]).max() for c in range(3))


def test_nested_single_samples_by_brute_force(orc80):
    """re-evaluate X, Y, Z at a few samples with independent code: exact chains for L_l(t) = L0_l + r_l t (a linear series is
    interpolated exactly), analytic link series evaluated at the exact retarded time"""
    n, dt, t0 = 2500, 5.0, 2.0e5
    rates = np.array([3.0, -2.0, 1.5, -1.0, 2.5, -3.5]) * 1.0e-8
    orbit, L0 = breathing_tables(n, dt, t0, rates)
    t = t0 + dt * np.arange(n)
    fl = [1.3e-3, 2.1e-3, 0.9e-3, 1.7e-3, 2.6e-3, 0.6e-3]

    def ylink(l, x):
        return np.sin(2 * np.pi * fl[l] * x + 0.3 * l)

    y = np.array([ylink(l, t) for l in range(6)])
    idx = {+1: 0, +2: 1, +3: 2, -1: 3, -2: 4, -3: 5}

    def L_at(label, x):
        return L0[idx[label]] + rates[idx[label]] * x

    def chain(x, labels):
        for lab in labels:
            x = x - L_at(lab, x)
        return x

    def cyc(label, k):
        a = abs(label)
        for _ in range(k):
            a = a % 3 + 1
        return a if label > 0 else -a

    for gen in (15, 20):
        got = orc80.michelson_nested_from_links(orbit, y, gen, 31, 3)
        for ns in (700, 1234, 2100):
            x = t[ns]
            for ch in range(3):
                p2, p3 = cyc(2, ch), cyc(3, ch)
                P, Q, U, Wl = idx[p2], idx[-p2], idx[-p3], idx[p3]
                a, b = [-p2, p2], [p3, -p3]

                def arm1(pre):   # (Q + D_-p2 P) behind the operator product `pre`
                    return ylink(Q, chain(x, pre)) + ylink(P, chain(x, pre + [-p2]))

                def arm2(pre):   # (W + D_p3 U)
                    return ylink(Wl, chain(x, pre)) + ylink(U, chain(x, pre + [p3]))

                want = arm1([]) - arm1(b) - (arm2([]) - arm2(a))
                if gen == 20:
                    want += -arm1(b + a) + arm1(a + b + b) + arm2(a + b) - arm2(b + a + a)
                assert abs(got[ch, ns] - want) < 2e-11, (gen, ns, ch, got[ch, ns], want)
