"""Seeded synthetic inputs shaped like the workloads of arXiv 2505.09600 / BASELINE.json.

This module serves BOTH the CPU oracle (tests, bench cpu_baseline) and the CUDA path
(tests, bench).  It holds none of the method's arithmetic: no projection, no
interpolation, no TDI, no hybrid weights, no t_hyb -- only waveform and parameter
generation (input data).  It imports neither `oracle` nor `paper_2505_09600_b200`.

The paper's waveforms (IMRPhenomTHM / TEHM) are not in the container;
leading-order chirps, a damped-sinusoid ringdown and Peters-Mathews harmonic sums with
the same lengths, sampling steps and spectral content stand in for them (DESIGN.md,
"input recipe").  Every source is drawn from numpy default_rng([seed, source_index]), so
a source's data does not depend on which other sources are generated with it.
"""
import math

import numpy as np
from scipy.special import jv

C_LIGHT = 299792458.0
GMSUN_S = 4.925490947e-6          # G M_sun / c^3 [s]
GPC_M = 3.085677581e25            # 1 Gpc [m]
AU_M = 149597870700.0
ARM_M = 2.5e9
YEAR_S = 31558149.7635            # sidereal year [s]
DAY_S = 86400.0

ORBIT_STATIC_EQUALARM, ORBIT_KEPLERIAN, ORBIT_TABLES = 0, 1, 2
TAPER_SIGMOID, TAPER_COSINE = 0, 1


def orbit_desc(n, dt, mode=ORBIT_KEPLERIAN, t0=0.0, arm_m=ARM_M, R_m=AU_M, period_s=YEAR_S,
               alpha0=0.0, rot0=0.0):
    return {"t0": float(t0), "dt": float(dt), "n": int(n), "arm_m": float(arm_m), "R_m": float(R_m),
            "period_s": float(period_s), "alpha0": float(alpha0), "rot0": float(rot0), "mode": int(mode)}


# ---------------------------------------------------------------------------------------
# waveforms (input data)
# ---------------------------------------------------------------------------------------
def chirp_mass_s(M_sun, q):
    eta = q / (1.0 + q) ** 2
    return M_sun * GMSUN_S * eta ** 0.6


def f_of_tau(tau, mc_s):
    """leading-order GW frequency at time tau before coalescence (same order as Eq. 4.2)"""
    return (1.0 / math.pi) * (5.0 / (256.0 * tau)) ** 0.375 * mc_s ** (-0.625)


def tau_of_f(f, mc_s):
    return 5.0 / 256.0 * (math.pi * f) ** (-8.0 / 3.0) * mc_s ** (-5.0 / 3.0)


def newtonian_chirp(t, t_c, mc_s, dist_m, cos_iota, phi_c, ringdown=None):
    """h+, hx of a quadrupole chirp; optional ringdown = dict(M_s, dt) joins a damped sinusoid.

    Before the join time t_m (GW frequency f_cut): amp = 4 (Mc c / d_L)(pi f Mc)^(2/3),
    Phi = phi_c - 2 (tau / 5 Mc)^(5/8).  After it: amplitude A_m exp(-(t-t_m)/tau_rd), frequency
    relaxing from f_cut to f_rd with the same time constant, phase continuous.
    """
    t = np.asarray(t, dtype=np.float64)
    if ringdown is not None:
        M_s, dt = ringdown["M_s"], ringdown["dt"]
        Mf = 0.95 * M_s
        f_grid = 0.2 / dt                                   # keep the data well below Nyquist
        f_rd = min(0.37367 / (2.0 * math.pi * Mf), f_grid)
        tau_rd = Mf / 0.08896
        f_isco = 1.0 / (6.0 ** 1.5 * math.pi * M_s)
        f_cut = min(f_isco, 0.9 * f_rd, 0.5 * f_grid)
        tau_cut = tau_of_f(f_cut, mc_s)
    else:
        tau_cut = None
    tau = t_c - t
    tau_in = np.maximum(tau, tau_cut if tau_cut is not None else 1e-3)
    f = (1.0 / math.pi) * (5.0 / (256.0 * tau_in)) ** 0.375 * mc_s ** (-0.625)
    amp = 4.0 * (mc_s * C_LIGHT / dist_m) * (math.pi * f * mc_s) ** (2.0 / 3.0)
    phase = phi_c - 2.0 * (tau_in / (5.0 * mc_s)) ** 0.625
    if ringdown is not None:
        x = np.maximum(-(tau - tau_cut), 0.0)               # time after the join
        decay = np.exp(-x / tau_rd)
        amp = amp * decay
        phase = phase + 2.0 * math.pi * (f_rd * x - (f_rd - f_cut) * tau_rd * (1.0 - decay))
    hp = amp * 0.5 * (1.0 + cos_iota ** 2) * np.cos(phase)
    hc = amp * cos_iota * np.sin(phase)
    return hp, hc


def _peters_rhs(F, e, M_s, eta):
    k = eta * M_s ** (5.0 / 3.0) * (2.0 * math.pi * F) ** (8.0 / 3.0)
    fe1 = (1.0 + 73.0 / 24.0 * e * e + 37.0 / 96.0 * e ** 4) / (1.0 - e * e) ** 3.5
    fe2 = (1.0 + 121.0 / 304.0 * e * e) / (1.0 - e * e) ** 2.5
    return 96.0 / 5.0 * k * F * fe1, -304.0 / 15.0 * k * e * fe2


def eccentric_knots(t_first, t_end, tau_end, M_s, q, e0, knots=1536):
    """The orbital evolution table of an eccentric inspiral: F(t), e(t), l(t) and their time derivatives at `knots` times
    (uniform in log time-to-coalescence), from the orbit-averaged Peters (1964) equations integrated backwards from the
    end of the segment with RK4.  Returns (tk, Fk, ek, lk, dFk, dek, dlk), tk increasing.  Input data: the table plays
    the role of a waveform-model parameter set for the rows that generate the strain themselves."""
    eta = q / (1.0 + q) ** 2
    mc_s = M_s * eta ** 0.6
    T_seg = t_end - t_first
    F_end = 0.5 * f_of_tau(tau_end, mc_s)
    F_start_c = 0.5 * f_of_tau(tau_end + T_seg, mc_s)
    e_end = e0 * (F_start_c / F_end) ** (19.0 / 18.0)
    # knots in s = ln(time to circular-estimate coalescence), from the end backwards
    s = np.linspace(math.log(tau_end), math.log(tau_end + T_seg), knots)
    tk = t_end + tau_end - np.exp(s)
    Fk, ek, lk = np.zeros(knots), np.zeros(knots), np.zeros(knots)
    Fk[0], ek[0] = F_end, e_end

    def rhs(state, tt):
        dF, de = _peters_rhs(state[0], state[1], M_s, eta)
        return np.array([dF, de, 2.0 * math.pi * state[0]])

    st = np.array([F_end, e_end, 0.0])
    for i in range(1, knots):
        h = tk[i] - tk[i - 1]
        k1 = rhs(st, 0)
        k2 = rhs(st + 0.5 * h * k1, 0)
        k3 = rhs(st + 0.5 * h * k2, 0)
        k4 = rhs(st + h * k3, 0)
        st = st + h / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
        Fk[i], ek[i], lk[i] = st
    tk, Fk, ek, lk = tk[::-1].copy(), Fk[::-1].copy(), ek[::-1].copy(), lk[::-1].copy()
    dFk, dek = _peters_rhs(Fk, ek, M_s, eta)
    dlk = 2.0 * math.pi * Fk
    return tk, Fk, ek, lk, dFk, dek, dlk


def eccentric_harmonics(t, t_end, tau_end, M_s, q, e0, dist_m, cos_iota, gamma, l0, nharm=10, knots=1536):
    """h+, hx = sum over harmonics n = 1..nharm of the orbital phase with Peters-Mathews
    quadrupole amplitudes (Peters & Mathews 1963 harmonic decomposition in the form of Barack &
    Cutler 2004, Eqs. 7-9); F(t), e(t), l(t) from eccentric_knots(), carried to the samples by cubic
    Hermite interpolation."""
    eta = q / (1.0 + q) ** 2
    tk, Fk, ek, lk, dFk, dek, dlk = eccentric_knots(t[0], t_end, tau_end, M_s, q, e0, knots)

    def hermite(yk, dyk):
        idx = np.clip(np.searchsorted(tk, t, side="right") - 1, 0, knots - 2)
        h = tk[idx + 1] - tk[idx]
        u = (t - tk[idx]) / h
        h00 = (1 + 2 * u) * (1 - u) ** 2
        h10 = u * (1 - u) ** 2
        h01 = u * u * (3 - 2 * u)
        h11 = u * u * (u - 1)
        return h00 * yk[idx] + h10 * h * dyk[idx] + h01 * yk[idx + 1] + h11 * h * dyk[idx + 1]

    F = hermite(Fk, dFk)
    e = hermite(ek, dek)
    ell = hermite(lk, dlk) + l0
    amp = (2.0 * math.pi * F * M_s) ** (2.0 / 3.0) * eta * M_s * C_LIGHT / dist_m
    c2g, s2g = math.cos(2 * gamma), math.sin(2 * gamma)
    ci2 = cos_iota ** 2
    hp, hc = np.zeros_like(t), np.zeros_like(t)
    cl, sl = np.cos(ell), np.sin(ell)
    cn_1, sn_1 = np.ones_like(t), np.zeros_like(t)          # cos/sin((n-1) l)
    sq = np.sqrt(1.0 - e * e)
    for n in range(1, nharm + 1):
        cn = cn_1 * cl - sn_1 * sl
        sn = sn_1 * cl + cn_1 * sl
        ne = n * e
        jm2, jm1, j0, jp1, jp2 = jv(n - 2, ne), jv(n - 1, ne), jv(n, ne), jv(n + 1, ne), jv(n + 2, ne)
        a_n = -n * amp * (jm2 - 2 * e * jm1 + (2.0 / n) * j0 + 2 * e * jp1 - jp2) * cn
        b_n = -n * amp * sq * (jm2 - 2 * j0 + jp2) * sn
        c_n = 2 * amp * j0 * cn
        hp += -(1 + ci2) * (a_n * c2g - b_n * s2g) + (1 - ci2) * c_n
        hc += 2 * cos_iota * (b_n * c2g + a_n * s2g)
        cn_1, sn_1 = cn, sn
    return hp, hc


# ---------------------------------------------------------------------------------------
# the five configs of BASELINE.json (index k = 1..5 as in SURVEY.md section 8d)
# ---------------------------------------------------------------------------------------
CONFIGS = {
    1: dict(name="cfg1_chirp_1day", n=8640, dt=10.0, batch=1, mode=ORBIT_STATIC_EQUALARM, order=9, seed=1,
            runs=[("full", 15, 0)]),
    2: dict(name="cfg2_mbhb_30day", n=518400, dt=5.0, batch=1, mode=ORBIT_KEPLERIAN, order=31, seed=2,
            runs=[("full", 20, 0), ("lfa", 20, 2), ("hybrid", 20, 2)]),
    3: dict(name="cfg3_inspiral_1yr", n=6307200, dt=5.0, batch=1, mode=ORBIT_KEPLERIAN, order=31, seed=3,
            runs=[("lfa", 15, 2), ("lfa", 15, 4), ("lfa", 20, 2), ("lfa", 20, 4)]),
    4: dict(name="cfg4_pe_batch", n=131072, dt=10.0, batch=4096, mode=ORBIT_KEPLERIAN, order=31, seed=4,
            runs=[("hybrid", 20, 2)]),
    5: dict(name="cfg5_eccentric", n=1048576, dt=5.0, batch=256, mode=ORBIT_KEPLERIAN, order=31, seed=5,
            runs=[("full", 20, 0), ("lfa", 20, 2)]),
}
HYB_F_HZ = 2.0e-3            # BASELINE.json configs 2 and 4: switch when f_GW reaches 2 mHz
HYB_WINDOW_S = 3600.0        # 1-hour cosine taper


def _angles(rng):
    cos_iota = rng.uniform(-1.0, 1.0)
    beta = math.asin(rng.uniform(-1.0, 1.0))
    lam = rng.uniform(0.0, 2.0 * math.pi)
    psi = rng.uniform(0.0, math.pi)
    phi_c = rng.uniform(0.0, 2.0 * math.pi)
    return cos_iota, beta, lam, psi, phi_c


def config(k, n=None, batch=None):
    """dict describing config k; n / batch may be reduced for small parity cases."""
    c = dict(CONFIGS[k])
    c["k"] = k
    if n is not None:
        c["n"] = int(n)
    if batch is not None:
        c["batch"] = int(batch)
    c["orbit"] = orbit_desc(c["n"], c["dt"], c["mode"])
    return c


def draw(cfg, idx):
    """The seeded parameters of source `idx` of a config, without its time series (input data only: masses,
    distance, angles, eccentricity, and the fractions that place the merger).  source() builds the series from
    exactly these draws; the tests use them to pick a stratified parity subset of a large batch."""
    k = cfg["k"]
    rng = np.random.default_rng([cfg["seed"], int(idx)])
    cos_iota, beta, lam, psi, phi_c = _angles(rng)
    p = {"cos_iota": cos_iota, "beta": beta, "lam": lam, "psi": psi, "phi_c": phi_c}
    if k == 1:
        p.update(M=2.0e6, q=1.0, dist=10.0 * GPC_M)
    elif k == 2:
        p.update(M=1.0e6, q=rng.uniform(1.0, 8.0), dist=5.0 * GPC_M)
        p["merger_h_before_end"] = rng.uniform(0.5, 2.0)
    elif k == 3:
        p.update(M=1.0e5, q=2.0, dist=5.0 * GPC_M)
    elif k == 4:
        p["M"] = 10.0 ** rng.uniform(5.0, 7.0)
        p["q"] = rng.uniform(1.0, 10.0)
        p["dist"] = rng.uniform(1.0, 20.0) * GPC_M
        p["merger_fraction"] = rng.uniform(0.9, 1.0)
    elif k == 5:
        p["M"] = 10.0 ** rng.uniform(5.0, 6.0)
        p["q"] = rng.uniform(1.0, 4.0)
        p["e0"] = rng.uniform(0.0, 0.3)
        p["dist"] = rng.uniform(1.0, 10.0) * GPC_M
        p["gamma"] = rng.uniform(0.0, math.pi)
        p["tau_end"] = rng.uniform(1.0, 12.0) * 3600.0
    else:
        raise ValueError(k)
    p["mchirp_s"] = chirp_mass_s(p["M"], p["q"])
    return p


def source(cfg, idx):
    """One source of a config: returns (hp[n], hc[n], (beta, lambda, psi), meta).

    meta carries the numbers the hybrid needs (mchirp_s, t_c, f_hyb_hz, window_s); the hybrid time
    itself (Eq. 4.2) is method arithmetic and is computed by each side with its own helper."""
    k, n, dt = cfg["k"], cfg["n"], cfg["dt"]
    t = cfg["orbit"]["t0"] + dt * np.arange(n, dtype=np.float64)
    t_end = t[-1] + dt
    p = draw(cfg, idx)
    cos_iota, beta, lam, psi, phi_c = p["cos_iota"], p["beta"], p["lam"], p["psi"], p["phi_c"]
    M, q, dist, mc = p["M"], p["q"], p["dist"], p["mchirp_s"]
    meta = {"f_hyb_hz": HYB_F_HZ, "window_s": HYB_WINDOW_S, "taper": TAPER_COSINE}
    if k == 1:
        t_c = t_end + 2.0 * DAY_S
        hp, hc = newtonian_chirp(t, t_c, mc, dist, cos_iota, phi_c)
    elif k == 2:
        rd = {"M_s": M * GMSUN_S, "dt": dt}
        t_m = t_end - p["merger_h_before_end"] * 3600.0
        t_c = t_m + _tau_cut(mc, rd)
        hp, hc = newtonian_chirp(t, t_c, mc, dist, cos_iota, phi_c, ringdown=rd)
    elif k == 3:
        t_c = t[0] + 2.0 * 365.0 * DAY_S
        hp, hc = newtonian_chirp(t, t_c, mc, dist, cos_iota, phi_c)
    elif k == 4:
        rd = {"M_s": M * GMSUN_S, "dt": dt}
        t_m = t[0] + (t_end - t[0]) * p["merger_fraction"]
        t_c = t_m + _tau_cut(mc, rd)
        hp, hc = newtonian_chirp(t, t_c, mc, dist, cos_iota, phi_c, ringdown=rd)
    else:
        tau_end = p["tau_end"]
        t_c = t_end + tau_end
        hp, hc = eccentric_harmonics(t, t_end, tau_end, M * GMSUN_S, q, p["e0"], dist, cos_iota, p["gamma"], phi_c)
    meta.update({"mchirp_s": mc, "t_c": t_c})
    return hp, hc, (beta, lam, psi), meta


def chirp_params(cfg, idx):
    """Parameters of the chirp + ringdown model of source `idx` of configs 1-4 (the numbers source() feeds to
    newtonian_chirp): dict t_c, mc_s, dist_m, cos_iota, phi_c, tau_cut, f_rd, tau_rd -- for the rows that generate the
    strain themselves.  Without a ringdown (configs 1, 3) the join sits 1 ms before coalescence."""
    k, n, dt = cfg["k"], cfg["n"], cfg["dt"]
    assert k in (1, 2, 3, 4)
    t_first = cfg["orbit"]["t0"]
    t_end = t_first + dt * n
    p = draw(cfg, idx)
    mc = p["mchirp_s"]
    out = {"mc_s": mc, "dist_m": p["dist"], "cos_iota": p["cos_iota"], "phi_c": p["phi_c"]}
    if k in (2, 4):
        rd = {"M_s": p["M"] * GMSUN_S, "dt": dt}
        Mf = 0.95 * rd["M_s"]
        t_m = t_end - p["merger_h_before_end"] * 3600.0 if k == 2 else t_first + (t_end - t_first) * p["merger_fraction"]
        tau_cut = _tau_cut(mc, rd)
        out.update(t_c=t_m + tau_cut, tau_cut=tau_cut, f_rd=min(0.37367 / (2.0 * math.pi * Mf), 0.2 / dt), tau_rd=Mf / 0.08896)
    else:
        tau_cut = 1e-3
        t_c = t_end + 2.0 * DAY_S if k == 1 else t_first + 2.0 * 365.0 * DAY_S
        out.update(t_c=t_c, tau_cut=tau_cut, f_rd=f_of_tau(tau_cut, mc), tau_rd=1.0)
    return out


def ecc_params(cfg, idx):
    """Orbital evolution table [7][nk] and scalars (M_s, eta, dist_m, cos_iota, gamma, l0) of source `idx` of config 5:
    what source() feeds to eccentric_harmonics, for the rows that generate the strain themselves."""
    assert cfg["k"] == 5
    n, dt = cfg["n"], cfg["dt"]
    t_first = cfg["orbit"]["t0"]
    t_end = t_first + dt * (n - 1) + dt
    p = draw(cfg, idx)
    M_s = p["M"] * GMSUN_S
    table = np.array(eccentric_knots(t_first, t_end, p["tau_end"], M_s, p["q"], p["e0"]))
    eta = p["q"] / (1.0 + p["q"]) ** 2
    return table, np.array([M_s, eta, p["dist"], p["cos_iota"], p["gamma"], p["phi_c"]])


def _tau_cut(mc_s, rd):
    M_s, dt = rd["M_s"], rd["dt"]
    f_grid = 0.2 / dt
    f_rd = min(0.37367 / (2.0 * math.pi * 0.95 * M_s), f_grid)
    f_isco = 1.0 / (6.0 ** 1.5 * math.pi * M_s)
    return tau_of_f(min(f_isco, 0.9 * f_rd, 0.5 * f_grid), mc_s)


def sources(cfg, indices):
    """Stack several sources: hp, hc [len(indices)][n], angles [len][3], list of meta."""
    hp = np.empty((len(indices), cfg["n"]))
    hc = np.empty_like(hp)
    ang = np.empty((len(indices), 3))
    metas = []
    for r, i in enumerate(indices):
        hp[r], hc[r], ang[r], m = source(cfg, i)
        metas.append(m)
    return hp, hc, ang, metas


# ---------------------------------------------------------------------------------------
# simple analytic test signals (used by pins and edge-case parity tests)
# ---------------------------------------------------------------------------------------
def monochromatic(n, dt, f_hz, a_plus=1.0, a_cross=0.7, phi_p=0.3, phi_c=1.1, t0=0.0):
    t = t0 + dt * np.arange(n, dtype=np.float64)
    w = 2.0 * math.pi * f_hz
    return a_plus * np.cos(w * t + phi_p), a_cross * np.cos(w * t + phi_c)


def frozen_tables(orbit, R_snapshot, L_snapshot):
    """ORBIT_TABLES description with the same positions / light times at every sample."""
    o = dict(orbit)
    o["mode"] = ORBIT_TABLES
    n = o["n"]
    o["R_table"] = np.repeat(np.asarray(R_snapshot, dtype=np.float64).reshape(3, 3, 1), n, axis=2)
    o["L_table"] = np.repeat(np.asarray(L_snapshot, dtype=np.float64).reshape(6, 1), n, axis=1)
    return o


# ---------------------------------------------------------------------------------------
# numerical orbit files (input data for SURVEY 8(f)-4; "realistic ESA orbits")
# ---------------------------------------------------------------------------------------
ORBIT_KNOTS = 3


def numerical_orbit(n, dt, t0=0.0, knot_dt=DAY_S, knot_order=7, seed=11, arm_m=ARM_M, R_m=AU_M, period_s=YEAR_S,
                    alpha0=0.0, rot0=0.0, scatter=5e-3):
    """An orbit FILE as a mission would deliver it: spacecraft positions [3][3][nk] tabulated every knot_dt seconds.

    The spacecraft move on exact Keplerian ellipses (Kepler's equation solved by Newton iteration) of the usual
    cartwheel construction -- semi-major axis R, eccentricity and inclination from alpha = L / (2 R), phases 120
    degrees apart -- with the eccentricity, inclination and phase of every spacecraft scattered by `scatter`
    (relative; seeded), so that the three arms differ at the per-cent level and breathe by metres per second, as the
    arms of ESA's numerically optimised orbits do.  The ellipses stand in for such a file: they are input data only
    (neither the oracle nor the library knows how the knots were made)."""
    rng = np.random.default_rng([seed, 4])
    margin = (knot_order + 1) // 2 + 1
    k0 = math.floor(t0 / knot_dt) - margin
    nk = math.ceil((t0 + n * dt) / knot_dt) + margin - k0 + 1
    tk0 = k0 * knot_dt
    tk = tk0 + knot_dt * np.arange(nk)
    a = arm_m / (2.0 * R_m)
    nu = math.pi / 3.0 + 5.0 / 8.0 * a
    e_nom = math.sqrt(1.0 + 4.0 * a * math.cos(nu) / math.sqrt(3.0) + 4.0 * a * a / 3.0) - 1.0
    inc_nom = math.atan(a * math.sin(nu) / (math.sqrt(3.0) / 2.0 + a * math.cos(nu)))
    om = 2.0 * math.pi / period_s
    knots = np.zeros((3, 3, nk))
    for i in range(3):
        e = e_nom * (1.0 + scatter * rng.standard_normal())
        inc = inc_nom * (1.0 + scatter * rng.standard_normal())
        sig = 2.0 * math.pi * i / 3.0 + rot0 + scatter * 1e-1 * rng.standard_normal()
        Mean = om * tk + alpha0 - sig
        psi = Mean.copy()
        for _ in range(12):                                   # psi + e sin psi = Mean
            psi -= (psi + e * np.sin(psi) - Mean) / (1.0 + e * np.cos(psi))
        xr = R_m * (np.cos(psi) + e) * math.cos(inc)
        yr = R_m * math.sqrt(1.0 - e * e) * np.sin(psi)
        zr = R_m * (np.cos(psi) + e) * math.sin(inc)
        knots[i, 0] = math.cos(sig) * xr - math.sin(sig) * yr
        knots[i, 1] = math.sin(sig) * xr + math.cos(sig) * yr
        knots[i, 2] = zr
    d = orbit_desc(n, dt, ORBIT_KNOTS, t0=t0, arm_m=arm_m, R_m=R_m, period_s=period_s, alpha0=alpha0, rot0=rot0)
    d.update(knots=np.ascontiguousarray(knots), knot_t0=float(tk0), knot_dt=float(knot_dt), knot_order=int(knot_order))
    return d
