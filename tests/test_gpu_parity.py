"""GPU parity: the CUDA path (through the C ABI) against the long-double oracle, element by element, on
the same seeded inputs.  Bar: per-channel relative L2 <= 1e-11 over the non-margin samples (BASELINE.json
north_star); margins must be exactly 0.0."""
import numpy as np
import pytest
import torch

import workloads as W
from parity_util import TOL, fp64_floor, hybrid_params, record, series_floor, strict_check, to_numpy

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ltdi():
    import paper_2505_09600_b200 as m
    assert torch.cuda.is_available(), "GPU parity tests need a CUDA device"
    return m


def run_case(ltdi, orc, cfg, which, gen, fd, order=None, taper=W.TAPER_COSINE, idx=None, ld_pad=0):
    n, batch = cfg["n"], cfg["batch"]
    order = order or cfg["order"]
    idx = list(range(batch)) if idx is None else idx
    hp, hc, ang, metas = W.sources(cfg, idx)
    orbit = cfg["orbit"]
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(orbit, device=dev)
    if ld_pad:
        pad = np.full((len(idx), ld_pad), 7.0)   # columns beyond n must never be read or written
        dhp = torch.from_numpy(np.concatenate([hp, pad], 1)).to(dev)
        dhc = torch.from_numpy(np.concatenate([hc, pad], 1)).to(dev)
    else:
        dhp, dhc = torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev)
    def oracle(o):
        if which == "full":
            return o.response_full(orbit, hp, hc, ang, gen, order)
        if which == "lfa":
            return o.response_lfa(orbit, hp, hc, ang, gen, order, fd)
        return o.response_hybrid(orbit, hp, hc, ang, gen, order, fd, hybrid_params(metas, o.hyb_time, taper, cfg["dt"]))

    ref = oracle(orc)
    if which == "full":
        out = ltdi.response_full(orb, dhp, dhc, ang, gen, order, True, True)
    elif which == "lfa":
        out = ltdi.response_lfa(orb, dhp, dhc, ang, gen, order, fd, True, True)
    else:
        out = ltdi.response_hybrid(orb, dhp, dhc, ang, gen, order, fd,
                                   hybrid_params(metas, ltdi.hyb_time, taper, cfg["dt"]), True, True)
    torch.cuda.synchronize()
    out = to_numpy(out)
    for k in out:
        out[k] = out[k][..., :n]
    fd_eff = 0 if which == "full" else fd     # the full response has no stencil rim
    lo, hi = orc.margins(orbit, gen, order, fd_eff)
    assert (lo, hi) == ltdi.margins(orbit, gen, order, fd_eff)
    # the fp64 floor of the algorithm on this input: the oracle's double build against its long-double build
    from oracle import Oracle
    ref64 = oracle(Oracle("f64"))
    ref["floor"] = fp64_floor(ref, ref64, lo, n, hi)
    ref["floor_XYZ"] = series_floor(ref["XYZ"], ref64["XYZ"], lo, n, hi)
    ref["floor_y"] = series_floor(ref["y"], ref64["y"], lo, n, hi)
    return out, ref, lo, hi


def check(out, ref, lo, hi, n, tol=TOL):
    """1e-11 per channel (T against the largest channel) and per link / Michelson series: parity_util.strict_check"""
    return strict_check(out, ref, lo, hi, n, tol)


def test_orbit_delay_kernel(ltdi, orc80):
    """S0: positions to one fp64 rounding; link vectors and light times as hi + lo pairs to 2e-17 (the oracle's own
    long-double rounding of R_r - R_s is 4e-18): the double-double orbit kernel.  Late in the mission (t = 1 yr) the
    fp64 rounding of t_n alone would be 7e-16 in n_l."""
    for mode, t0 in ((W.ORBIT_KEPLERIAN, 1.0e7), (W.ORBIT_KEPLERIAN, 3.1e7), (W.ORBIT_STATIC_EQUALARM, 1.0e7)):
        orbit = W.orbit_desc(70001, 5.0, mode, t0=t0, alpha0=0.3, rot0=1.1)
        R, nh, L = orc80.orbit_tables(orbit)
        nh_hi, nh_lo, L_hi, L_lo = orc80.orbit_tables_split(orbit)
        orb = ltdi.Orbits(orbit)
        rows, lo = orb.rows().cpu().numpy(), orb.rows_lo().double().cpu().numpy()
        assert np.abs(rows[0:9].reshape(3, 3, -1) - R).max() <= np.spacing(np.abs(R).max())     # 3e-5 m at 1 AU
        dn = (rows[9:18].reshape(3, 3, -1) - nh_hi[:3]) + (lo[0:9].reshape(3, 3, -1) - nh_lo[:3])
        dL = (rows[18:24] - L_hi) + (lo[9:15] - L_lo)
        assert np.abs(dn).max() <= 2e-17, np.abs(dn).max()
        assert np.abs(dL).max() <= 2e-17 * L.max(), np.abs(dL).max() / L.max()
        assert np.abs(rows[9:18].reshape(3, 3, -1) - nh[:3]).max() <= 1.2e-16       # the hi parts alone: one rounding
        assert np.array_equal(nh[3:], -nh[:3])        # n_-l = -n_l is what the table layout assumes


def test_orbit_tables_mode_link_vectors(ltdi, orc80):
    """LTDI_ORBIT_TABLES: n_l = (R_r - R_s) / |R_r - R_s| from the caller's fp64 positions, formed without rounding the
    difference; light times passed through (low parts zero)"""
    n = 5000
    base = W.orbit_desc(n, 5.0, W.ORBIT_KEPLERIAN, t0=2.0e6)
    R, _, L = orc80.orbit_tables(base)
    orbit = dict(base, mode=W.ORBIT_TABLES, R_table=np.ascontiguousarray(R), L_table=np.ascontiguousarray(L))
    nh_hi, nh_lo, L_hi, L_lo = orc80.orbit_tables_split(orbit)
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(orbit, torch.from_numpy(orbit["R_table"]).to(dev), torch.from_numpy(orbit["L_table"]).to(dev))
    rows, lo = orb.rows().cpu().numpy(), orb.rows_lo().double().cpu().numpy()
    dn = (rows[9:18].reshape(3, 3, -1) - nh_hi[:3]) + (lo[0:9].reshape(3, 3, -1) - nh_lo[:3])
    assert np.abs(dn).max() <= 2e-17
    assert np.array_equal(rows[18:24], L) and np.all(lo[9:15] == 0.0) and np.array_equal(rows[0:9].reshape(3, 3, -1), R)


def test_config1_full_tdi15(ltdi, orc80):
    cfg = W.config(1)
    out, ref, lo, hi = run_case(ltdi, orc80, cfg, "full", 15, 0)
    check(out, ref, lo, hi, cfg["n"])


@pytest.mark.parametrize("which,gen,taper", [("full", 20, 0), ("full", 15, 0), ("lfa", 20, 0), ("lfa", 15, 0),
                                             ("hybrid", 20, W.TAPER_COSINE), ("hybrid", 20, W.TAPER_SIGMOID),
                                             ("hybrid", 15, W.TAPER_COSINE)])
def test_config2_merger(ltdi, orc80, which, gen, taper):
    """config 2 shortened to its last 40 000 samples (several tiles, ragged tail, merger + ringdown)"""
    cfg = W.config(2, n=40007)
    out, ref, lo, hi = run_case(ltdi, orc80, cfg, which, gen, 2, taper=taper)
    check(out, ref, lo, hi, cfg["n"])


@pytest.mark.parametrize("gen", [15, 20])
@pytest.mark.parametrize("fd", [2, 4])
def test_config3_long_inspiral_lfa(ltdi, orc80, gen, fd):
    cfg = W.config(3, n=30011)
    out, ref, lo, hi = run_case(ltdi, orc80, cfg, "lfa", gen, fd)
    check(out, ref, lo, hi, cfg["n"])


def test_config4_batch_hybrid(ltdi, orc80):
    """config 4 slice: 40 sources (the > 32 sources parameter path) of 20 001 samples, per-source windows"""
    cfg = W.config(4, n=20001, batch=40)
    out, ref, lo, hi = run_case(ltdi, orc80, cfg, "hybrid", 20, 2)
    check(out, ref, lo, hi, cfg["n"])


@pytest.mark.parametrize("which", ["full", "lfa"])
def test_config5_eccentric(ltdi, orc80, which):
    cfg = W.config(5, n=65536, batch=2)
    out, ref, lo, hi = run_case(ltdi, orc80, cfg, which, 20, 2)
    check(out, ref, lo, hi, cfg["n"])


@pytest.mark.parametrize("order", [1, 5, 13, 63])
def test_generic_lagrange_orders(ltdi, orc80, order):
    cfg = W.config(2, n=5003, batch=2)
    for which in ("full", "lfa"):
        out, ref, lo, hi = run_case(ltdi, orc80, cfg, which, 20, 4, order=order, ld_pad=13)
        check(out, ref, lo, hi, cfg["n"])


def test_series_shorter_than_the_margins_is_all_zero(ltdi, orc80):
    cfg = W.config(2, n=200)
    out, ref, lo, hi = run_case(ltdi, orc80, cfg, "full", 20, 0)
    assert lo + hi > cfg["n"]
    for c in "AET":
        assert np.all(out[c] == 0.0) and np.all(ref[c] == 0.0)


def test_frozen_tables_mode(ltdi, orc80):
    """LTDI_ORBIT_TABLES with caller-supplied positions and light times"""
    n, dt = 4000, 5.0
    snap = W.orbit_desc(1, 1.0, W.ORBIT_KEPLERIAN, t0=0.37 * W.YEAR_S)
    R, _, L = orc80.orbit_tables(snap)
    orbit = W.frozen_tables(W.orbit_desc(n, dt), R[:, :, 0], L[:, 0])
    hp, hc = W.monochromatic(n, dt, 3e-3)
    ang = [(0.3, 1.0, 0.7)]
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(orbit, torch.from_numpy(orbit["R_table"]).to(dev), torch.from_numpy(orbit["L_table"]).to(dev))
    out = to_numpy(ltdi.response_full(orb, torch.from_numpy(hp[None]).to(dev), torch.from_numpy(hc[None]).to(dev),
                                      ang, 20, 31, True, True))
    ref = orc80.response_full(orbit, hp[None], hc[None], ang, 20, 31)
    lo, hi = orc80.margins(orbit, 20, 31, 0)
    from oracle import Oracle
    ref64 = Oracle("f64").response_full(orbit, hp[None], hc[None], ang, 20, 31)
    ref["floor"] = fp64_floor(ref, ref64, lo, n, hi)
    ref["floor_XYZ"] = series_floor(ref["XYZ"], ref64["XYZ"], lo, n, hi)
    ref["floor_y"] = series_floor(ref["y"], ref64["y"], lo, n, hi)
    check(out, ref, lo, hi, n)


def test_errors_from_the_device_entry_points(ltdi):
    dev = torch.device("cuda:0")
    orbit = W.orbit_desc(3000, 5.0)
    orb = ltdi.Orbits(orbit, device=dev)
    h = torch.zeros(1, 3000, dtype=torch.float64, device=dev)
    with pytest.raises(ltdi.LtdiError):
        ltdi.response_full(orb, h, h, [(0, 0, 0)], 17, 31)
    with pytest.raises(ltdi.LtdiError):
        ltdi.response_lfa(orb, h, h, [(0, 0, 0)], 20, 31, 3)
    with pytest.raises(ltdi.LtdiError):
        ltdi.response_full(orb, h[:, :2000].contiguous(), h[:, :2000].contiguous(), [(0, 0, 0)], 20, 31)  # ld < n
    with pytest.raises(ltdi.LtdiError):
        ltdi.response_hybrid(orb, h, h, [(0, 0, 0)], 20, 31, 2,
                             {"t_hyb": 0.0, "window_s": -1.0, "sigma_s": 1.0, "taper": 0})


def test_host_pipeline_matches_device_call(ltdi):
    """ltdi_response_host (host buffers in and out) gives bit-identical A, E, T"""
    dev = torch.device("cuda:0")
    cfg = W.config(2, n=9000, batch=3)
    hp, hc, ang, metas = W.sources(cfg, [0, 1, 2])
    orb = ltdi.Orbits(cfg["orbit"], device=dev)
    ref = ltdi.response_lfa(orb, torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev), ang, 20, 31, 2)
    pipe = ltdi.HostPipeline(orb, 3, 9000)
    A, E, T = pipe.run(ltdi.RESPONSE_LFA, torch.from_numpy(hp).pin_memory(), torch.from_numpy(hc).pin_memory(), ang,
                       20, 31, 2)
    torch.cuda.synchronize()
    assert torch.equal(A, ref["A"].cpu()) and torch.equal(E, ref["E"].cpu()) and torch.equal(T, ref["T"].cpu())


def test_host_call_cut_into_pieces_matches_device_call(ltdi):
    """a batch above 128 MiB per series goes through ltdi_response_host as a pipeline of pieces (upload / kernels / download
    on three streams): bitwise the device call, for the hybrid with one window per source (the per-source arrays are
    offset piece by piece), with a shared window, and for the LFA; two calls back to back on one stream and two slots"""
    dev = torch.device("cuda:0")
    n, batch = 40000, 520                     # 166 MB per series: 2 pieces of 260 sources
    cfg = W.config(4, n=n, batch=8)
    hp8, hc8, ang8, metas8 = W.sources(cfg, list(range(8)))
    rep = batch // 8
    hp, hc = np.tile(hp8, (rep, 1)), np.tile(hc8, (rep, 1))
    scale = 1.0 + 0.01 * np.arange(batch)[:, None]          # every source different
    hp, hc = hp * scale, hc * scale
    ang = np.tile(ang8, (rep, 1))
    metas = [metas8[i % 8] for i in range(batch)]
    hyb = hybrid_params(metas, ltdi.hyb_time, W.TAPER_COSINE, cfg["dt"])
    for i, h in enumerate(hyb):                              # and every window different
        h["t_hyb"] += 10.0 * cfg["dt"] * (i % 7)
    orb = ltdi.Orbits(cfg["orbit"], device=dev)
    dhp, dhc = torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev)
    hp_h, hc_h = torch.from_numpy(hp).pin_memory(), torch.from_numpy(hc).pin_memory()
    keep = lambda d: [d[c].cpu() for c in "AET"]
    want = [keep(ltdi.response_hybrid(orb, dhp, dhc, ang, 20, 31, 2, hyb)),
            keep(ltdi.response_hybrid(orb, dhp, dhc, ang, 20, 31, 2, hyb[3])),
            keep(ltdi.response_lfa(orb, dhp, dhc, ang, 20, 31, 2))]
    calls = [(ltdi.RESPONSE_HYBRID, hyb), (ltdi.RESPONSE_HYBRID, hyb[3]), (ltdi.RESPONSE_LFA, None)]
    for depth in (1, 2):
        pipe = ltdi.HostPipeline(orb, batch, n, depth=depth)
        for (which, h), w in zip(calls, want):
            out = pipe.run(which, hp_h, hc_h, ang, 20, 31, 2, h)
            pipe.synchronize()
            torch.cuda.synchronize()
            for a, b in zip(out, w):
                assert torch.equal(a, b), (depth, which)
        # back to back without a synchronisation in between: the second call must not overtake the first one's copies
        outs = []
        for (which, h) in calls[:2]:
            outs.append([t for t in pipe.run(which, hp_h, hc_h, ang, 20, 31, 2, h)])
            if depth == 1:
                pipe.synchronize()
                outs[-1] = [t.clone() for t in outs[-1]]
        pipe.synchronize()
        torch.cuda.synchronize()
        if depth == 2:
            for o, w in zip(outs, want[:2]):
                for a, b in zip(o, w):
                    assert torch.equal(a, b), depth
        del pipe


def test_prepared_anchors_give_bitwise_the_same_result(ltdi):
    """ltdi_orbits_prepare(): TDI weights computed once per time grid; the responses must not change by a bit,
    and a prepare for another generation / order must be ignored"""
    cfg = W.config(2, n=30011, batch=3)
    hp, hc, ang, metas = W.sources(cfg, [0, 1, 2])
    dev = torch.device("cuda:0")
    dhp, dhc = torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev)
    hyb = hybrid_params(metas, ltdi.hyb_time, W.TAPER_COSINE, cfg["dt"])

    def run(orb):
        out = []
        for gen in (15, 20):
            out.append(to_numpy(ltdi.response_full(orb, dhp, dhc, ang, gen, 31, True, False)))
            out.append(to_numpy(ltdi.response_lfa(orb, dhp, dhc, ang, gen, 31, 2, True, False)))
            out.append(to_numpy(ltdi.response_hybrid(orb, dhp, dhc, ang, gen, 31, 2, hyb, True, False)))
        torch.cuda.synchronize()
        return out

    plain = run(ltdi.Orbits(cfg["orbit"], device=dev))
    for gen, order in ((20, 31), (15, 31), (20, 9), (20, 13)):
        prepared = run(ltdi.Orbits(cfg["orbit"], device=dev).prepare(gen, order))
        for a, b in zip(plain, prepared):
            for k in ("A", "E", "T", "XYZ"):
                assert np.array_equal(a[k], b[k]), (gen, order, k)


def test_host_pipeline_with_two_slots_matches_single_slot(ltdi):
    """depth = 2 rotates streams / scratch / pinned outputs: same bits as the one-stream pipeline"""
    cfg = W.config(2, n=9000, batch=3)
    hp, hc, ang, metas = W.sources(cfg, [0, 1, 2])
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(cfg["orbit"], device=dev)
    hp_h, hc_h = torch.from_numpy(hp).pin_memory(), torch.from_numpy(hc).pin_memory()
    hyb = hybrid_params(metas, ltdi.hyb_time, W.TAPER_COSINE, cfg["dt"])
    calls = [(ltdi.RESPONSE_FULL, 2, None), (ltdi.RESPONSE_LFA, 2, None), (ltdi.RESPONSE_HYBRID, 2, hyb),
             (ltdi.RESPONSE_LFA, 4, None)]
    one = ltdi.HostPipeline(orb, 3, 9000)
    want = []
    for which, fd, h in calls:
        out = one.run(which, hp_h, hc_h, ang, 20, 31, fd, h)
        one.synchronize()
        want.append([t.clone() for t in out])
    two = ltdi.HostPipeline(orb, 3, 9000, depth=2)
    for rep in range(2):          # the second pass reuses slots that still hold results
        got = []
        for i, (which, fd, h) in enumerate(calls):
            out = two.run(which, hp_h, hc_h, ang, 20, 31, fd, h)
            if i >= 1:            # the previous call's slot is complete only after its event
                two.slots[(two.calls - 2) % 2]["event"].synchronize()
                got.append([t.clone() for t in two.slots[(two.calls - 2) % 2]["out"]])
        two.synchronize()
        got.append([t.clone() for t in out])
        for w, g in zip(want, got):
            for a, b in zip(w, g):
                assert torch.equal(a, b)


@pytest.mark.parametrize("dt", [0.05, 0.5, 1.0, 2.0, 3.3, 4.6, 5.0, 7.5, 12.0, 30.0, 60.0])
def test_sampling_steps_sweep_the_shared_memory_plans(ltdi, orc80, dt):
    """the halo widths, and with them the shared-memory carve-up of every kernel, depend on dt: sweep it through the
    opt-in threshold (48 KB), the tuned path and, for very small dt, the fall-back to the generic kernel; Keplerian
    orbit, two sources, all three responses, both generations, orders 31 and 9"""
    from oracle import Oracle
    orc64 = Oracle("f64")
    lo_max = max(orc80.margins(W.orbit_desc(10, dt), 20, 31, 4))
    n = int(2 * lo_max + 1500) if dt >= 0.5 else int(2 * lo_max + 300)
    orbit = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN, t0=1.234e7)
    # well sampled (50 samples per cycle), but never below 2 mHz: the full TDI 2.0 response cancels as (omega L / c)^3
    # at low frequency and NO fp64 evaluation meets 1e-11 there (the oracle's own double build: 1e-11 at 0.7 mHz,
    # 1e-9 at 0.1 mHz, hard part 1) -- which is the regime the paper gives to the LFA
    f = max(0.02 / dt, 2.0e-3)
    hp0, hc0 = W.monochromatic(n, dt, f, t0=orbit["t0"])
    hp1, hc1 = W.monochromatic(n, dt, 0.6 * f, a_plus=0.4, a_cross=-1.1, phi_p=2.0, phi_c=0.1, t0=orbit["t0"])
    hp, hc = np.stack([hp0, hp1]), np.stack([hc0, hc1])
    ang = [(0.3, 1.0, 0.7), (-0.9, 4.0, 2.2)]
    tmid = orbit["t0"] + 0.55 * n * dt
    hyb = [{"t_hyb": tmid, "window_s": 40 * dt, "sigma_s": dt, "taper": W.TAPER_COSINE},
           {"t_hyb": tmid - 100 * dt, "window_s": 64 * dt, "sigma_s": 1.6 * dt, "taper": W.TAPER_SIGMOID}]
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(orbit, device=dev)
    dhp, dhc = torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev)
    cases = [("full", 20, 31, 0), ("lfa", 20, 31, 2), ("hybrid", 20, 31, 4), ("full", 15, 9, 0), ("hybrid", 15, 9, 2)]
    if dt < 0.5:
        cases = cases[:3]          # the oracle takes a second per response here
    for which, gen, order, fd in cases:
        if which == "full":
            out = ltdi.response_full(orb, dhp, dhc, ang, gen, order, True, True)
            ref, ref64 = (o.response_full(orbit, hp, hc, ang, gen, order) for o in (orc80, orc64))
        elif which == "lfa":
            out = ltdi.response_lfa(orb, dhp, dhc, ang, gen, order, fd, True, True)
            ref, ref64 = (o.response_lfa(orbit, hp, hc, ang, gen, order, fd) for o in (orc80, orc64))
        else:
            out = ltdi.response_hybrid(orb, dhp, dhc, ang, gen, order, fd, hyb, True, True)
            ref, ref64 = (o.response_hybrid(orbit, hp, hc, ang, gen, order, fd, hyb) for o in (orc80, orc64))
        torch.cuda.synchronize()
        out = to_numpy(out)
        lo, hi = orc80.margins(orbit, gen, order, fd)
        assert (lo, hi) == ltdi.margins(orbit, gen, order, fd)
        ref["floor"] = fp64_floor(ref, ref64, lo, n, hi)
        ref["floor_XYZ"] = series_floor(ref["XYZ"], ref64["XYZ"], lo, n, hi)
        ref["floor_y"] = series_floor(ref["y"], ref64["y"], lo, n, hi)
        check(out, ref, lo, hi, n)


def test_unsupported_shape_is_reported(ltdi):
    """dt = 0.02 s: the link series a hybrid TDI 2.0 tile needs (7.2 L / c = 3000 samples back, for nine series) do
    not fit the 227 KB of shared memory: the call must say LTDI_EUNSUPPORTED, not launch (include/lisatdi.h)"""
    n, dt = 60000, 0.02
    orb = ltdi.Orbits(W.orbit_desc(n, dt))
    h = torch.zeros(1, n, dtype=torch.float64, device="cuda:0")
    with pytest.raises(ltdi.LtdiError) as e:
        ltdi.response_hybrid(orb, h, h, [(0.1, 0.2, 0.3)], 20, 31, 2,
                             {"t_hyb": 600.0, "window_s": 1.0, "sigma_s": 0.1, "taper": 0})
    assert e.value.code == ltdi.EUNSUPPORTED


@pytest.mark.parametrize("order", [31, 9])
def test_fast_varying_tables_take_the_exact_weight_paths(ltdi, orc80, order):
    """LTDI_ORBIT_TABLES with light times that breathe by 1 % within minutes and spacecraft that wobble by a light
    second: the TDI delays drift by far more than the first-order anchors allow and cross integer shifts inside
    tiles (exact per-sample weights in tdi_kernel), and the two samples of a link pair get different integer shifts
    (single-sample interpolator in link_kernel).  Same bar as everywhere else."""
    from oracle import Oracle
    orc64 = Oracle("f64")
    n, dt = 6000, 5.0
    base = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN, t0=2.0e6)
    R, _, L = orc80.orbit_tables(base)
    t = base["t0"] + dt * np.arange(n)
    rng = np.random.default_rng(11)
    R = R + 3.0e8 * np.sin(2 * np.pi * t / 487.0 + rng.uniform(0, 6, (3, 3, 1)))          # [3][3][n]
    L = L * (1.0 + 1.0e-2 * np.sin(2 * np.pi * t / 1733.0 + rng.uniform(0, 6, (6, 1))))    # [6][n]
    orbit = dict(base, mode=W.ORBIT_TABLES, R_table=np.ascontiguousarray(R), L_table=np.ascontiguousarray(L))
    hp0, hc0 = W.monochromatic(n, dt, 4e-3, t0=base["t0"])
    hp1, hc1 = W.monochromatic(n, dt, 1.1e-2, a_plus=0.3, a_cross=0.9, t0=base["t0"])
    hp, hc = np.stack([hp0, hp1]), np.stack([hc0, hc1])
    ang = [(0.3, 1.0, 0.7), (-0.9, 4.0, 2.2)]
    hyb = {"t_hyb": base["t0"] + 0.5 * n * dt, "window_s": 600.0, "sigma_s": 15.0, "taper": W.TAPER_SIGMOID}
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(orbit, torch.from_numpy(orbit["R_table"]).to(dev), torch.from_numpy(orbit["L_table"]).to(dev))
    dhp, dhc = torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev)
    for which, gen, fd in (("full", 20, 0), ("full", 15, 0), ("lfa", 20, 2), ("lfa", 15, 4), ("hybrid", 20, 2)):
        if which == "full":
            out = ltdi.response_full(orb, dhp, dhc, ang, gen, order, True, True)
            ref, ref64 = (o.response_full(orbit, hp, hc, ang, gen, order) for o in (orc80, orc64))
        elif which == "lfa":
            out = ltdi.response_lfa(orb, dhp, dhc, ang, gen, order, fd, True, True)
            ref, ref64 = (o.response_lfa(orbit, hp, hc, ang, gen, order, fd) for o in (orc80, orc64))
        else:
            out = ltdi.response_hybrid(orb, dhp, dhc, ang, gen, order, fd, hyb, True, True)
            ref, ref64 = (o.response_hybrid(orbit, hp, hc, ang, gen, order, fd, hyb) for o in (orc80, orc64))
        torch.cuda.synchronize()
        out = to_numpy(out)
        lo, hi = orc80.margins(orbit, gen, order, fd)
        ref["floor"] = fp64_floor(ref, ref64, lo, n, hi)
        ref["floor_XYZ"] = series_floor(ref["XYZ"], ref64["XYZ"], lo, n, hi)
        ref["floor_y"] = series_floor(ref["y"], ref64["y"], lo, n, hi)
        check(out, ref, lo, hi, n)


@pytest.mark.parametrize("shared_window", [True, False])
def test_parameter_slices_of_large_batches(ltdi, orc80, shared_window):
    """600 sources (two parameter launches of 512 + 88) of 3001 samples: 8 distinct sources tiled 75 times; one
    hybrid window for all (n_hyb = 1) or one per source; the first copies match the oracle, the replicas the first"""
    cfg = W.config(4, n=3001, batch=8)
    hp, hc, ang, metas = W.sources(cfg, list(range(8)))
    reps, n, dt = 75, cfg["n"], cfg["dt"]
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(cfg["orbit"], device=dev)
    dhp, dhc = torch.from_numpy(hp).to(dev).repeat(reps, 1), torch.from_numpy(hc).to(dev).repeat(reps, 1)
    tmid = cfg["orbit"]["t0"] + 0.6 * n * dt
    mk = lambda i: {"t_hyb": tmid + 40.0 * dt * i, "window_s": 64 * dt, "sigma_s": 1.6 * dt, "taper": i % 2}
    hyb8 = [mk(0)] * 8 if shared_window else [mk(i) for i in range(8)]
    hyb_gpu = mk(0) if shared_window else hyb8 * reps
    out = to_numpy(ltdi.response_hybrid(orb, dhp, dhc, np.tile(ang, (reps, 1)), 20, 31, 2, hyb_gpu, True, True))
    torch.cuda.synchronize()
    for k in ("A", "E", "T"):
        v = out[k].reshape(reps, 8, n)
        assert np.array_equal(v, np.broadcast_to(v[0], v.shape)), k
    first = {k: (v[:8] if v.ndim == 2 else v[:, :8]) for k, v in out.items()}
    from oracle import Oracle
    ref = orc80.response_hybrid(cfg["orbit"], hp, hc, ang, 20, 31, 2, hyb8)
    ref64 = Oracle("f64").response_hybrid(cfg["orbit"], hp, hc, ang, 20, 31, 2, hyb8)
    lo, hi = orc80.margins(cfg["orbit"], 20, 31, 2)
    ref["floor"] = fp64_floor(ref, ref64, lo, n, hi)
    ref["floor_XYZ"] = series_floor(ref["XYZ"], ref64["XYZ"], lo, n, hi)
    ref["floor_y"] = series_floor(ref["y"], ref64["y"], lo, n, hi)
    check(first, ref, lo, hi, n)


def test_decayed_ringdown_tail_keeps_relative_accuracy(ltdi, orc80):
    """A heavy binary that merges in the middle of the segment: the ring-down decays by hundreds of e-folds, and a
    window in that tail (1e-100 of the peak) must still match the oracle RELATIVE to its own norm -- the case that
    catches reduced-precision shortcuts in the interpolation (fp32 underflow) which a whole-series norm hides."""
    from oracle import Oracle
    orc64 = Oracle("f64")
    n, dt = 20001, 10.0
    orbit = W.orbit_desc(n, dt, W.ORBIT_KEPLERIAN, t0=3.0e6)
    t = orbit["t0"] + dt * np.arange(n)
    M_s = 8.0e6 * W.GMSUN_S
    mc = W.chirp_mass_s(8.0e6, 2.0)
    rd = {"M_s": M_s, "dt": dt}
    t_m = t[0] + 0.5 * n * dt
    hp, hc = W.newtonian_chirp(t, t_m + W._tau_cut(mc, rd), mc, 3.0 * W.GPC_M, 0.3, 1.0, ringdown=rd)
    hp, hc = hp[None], hc[None]
    assert 0.0 < np.abs(hp[0, -2000:]).max() < 1e-60 * np.abs(hp).max()      # decayed, but not to zero
    ang = [(0.4, 2.0, 0.9)]
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(orbit, device=dev)
    dhp, dhc = torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev)
    hyb = {"t_hyb": t[0] + 0.3 * n * dt, "window_s": 3600.0, "sigma_s": 90.0, "taper": W.TAPER_COSINE}
    for which in ("full", "hybrid"):
        if which == "full":
            out = to_numpy(ltdi.response_full(orb, dhp, dhc, ang, 20, 31))
            ref, ref64 = (o.response_full(orbit, hp, hc, ang, 20, 31, want=()) for o in (orc80, orc64))
        else:
            out = to_numpy(ltdi.response_hybrid(orb, dhp, dhc, ang, 20, 31, 2, hyb))
            ref, ref64 = (o.response_hybrid(orbit, hp, hc, ang, 20, 31, 2, hyb, want=()) for o in (orc80, orc64))
        lo, hi = orc80.margins(orbit, 20, 31, 2 if which == "hybrid" else 0)
        for a, b in ((n - hi - 1500, n - hi), (n - hi - 4000, n - hi - 2500), (int(0.55 * n), int(0.55 * n) + 1500)):
            for c in "AE":
                w80, w64, g = ref[c][0, a:b], ref64[c][0, a:b], out[c][0, a:b]
                nrm = np.linalg.norm(w80)
                assert nrm > 0
                err, floor = np.linalg.norm(g - w80) / nrm, np.linalg.norm(w64 - w80) / nrm
                record(label=[which], series=c, window=[int(a), int(b)], err=float(err), floor=float(floor), bar=TOL)
                assert err <= TOL, (which, c, (a, b), err, floor)


# ---- higher-order and alternative LFA (Eqs. (B4), (B13), (B14)) ------------------------------------

def run_lfa_ext(ltdi, orc, cfg, gen, fd, terms, point, order=None, idx=None):
    n = cfg["n"]
    order = order or cfg["order"]
    idx = list(range(cfg["batch"])) if idx is None else idx
    hp, hc, ang, _ = W.sources(cfg, idx)
    orbit = cfg["orbit"]
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(orbit, device=dev)
    ref = orc.response_lfa_ext(orbit, hp, hc, ang, gen, order, fd, terms, point)
    out = ltdi.response_lfa_ext(orb, torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev), ang, gen, order, fd,
                                terms, point, True, True)
    torch.cuda.synchronize()
    out = to_numpy(out)
    lo, hi = orc.margins_lfa_ext(orbit, gen, order, fd, terms)
    assert (lo, hi) == ltdi.margins_lfa_ext(orbit, gen, order, fd, terms)
    return out, ref, lo, hi


@pytest.mark.parametrize("gen,fd,terms,point", [(20, 2, 2, 0), (20, 4, 2, 0), (15, 2, 2, 0), (15, 4, 2, 0),
                                                (20, 2, 1, 1), (20, 2, 1, 2), (15, 4, 1, 1), (15, 4, 1, 2)])
def test_lfa_ext_config2(ltdi, orc80, gen, fd, terms, point):
    """m = 1 term of Eq. (B4) and the backward / forward expansion points on config 2's merger (tuned path, p = 31)"""
    cfg = W.config(2, n=40007)
    out, ref, lo, hi = run_lfa_ext(ltdi, orc80, cfg, gen, fd, terms, point)
    check(out, ref, lo, hi, cfg["n"])


@pytest.mark.parametrize("terms,point", [(2, 0), (1, 1), (1, 2)])
def test_lfa_ext_config3_gen20(ltdi, orc80, terms, point):
    """the worst-conditioned case (config 3, TDI 2.0: Eq. (B33) amplifies the noise of y by 2.45 / (omega dt)^2)"""
    cfg = W.config(3, n=30011)
    out, ref, lo, hi = run_lfa_ext(ltdi, orc80, cfg, 20, 2, terms, point)
    check(out, ref, lo, hi, cfg["n"])


def test_lfa_ext_terms1_is_the_lfa_bitwise(ltdi):
    cfg = W.config(2, n=20011)
    hp, hc, ang, _ = W.sources(cfg, [0])
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(cfg["orbit"], device=dev)
    dhp, dhc = torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev)
    for order in (31, 5):
        a = to_numpy(ltdi.response_lfa(orb, dhp, dhc, ang, 20, order, 2, True, True))
        b = to_numpy(ltdi.response_lfa_ext(orb, dhp, dhc, ang, 20, order, 2, 1, ltdi.LFA_CENTRAL, True, True))
        for k in a:
            assert np.array_equal(a[k], b[k]), (order, k)


@pytest.mark.parametrize("order,terms,point", [(5, 2, 0), (5, 1, 1), (9, 2, 0), (9, 1, 2)])
def test_lfa_ext_other_orders_and_batch(ltdi, orc80, order, terms, point):
    """generic kernel (p = 5) and the tuned p = 9 path, a batch of sources with a ragged length"""
    cfg = W.config(4, n=9001, batch=3)
    out, ref, lo, hi = run_lfa_ext(ltdi, orc80, cfg, 20, 4 if order == 9 else 2, terms, point, order=order)
    check(out, ref, lo, hi, cfg["n"])


def test_lfa_ext_argument_errors(ltdi):
    cfg = W.config(2, n=5003)
    hp, hc, ang, _ = W.sources(cfg, [0])
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(cfg["orbit"], device=dev)
    dhp, dhc = torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev)
    for terms, point in ((0, 0), (3, 0), (2, 1), (2, 2), (1, 3), (1, -1)):
        with pytest.raises(ltdi.LtdiError):
            ltdi.response_lfa_ext(orb, dhp, dhc, ang, 20, 31, 2, terms, point)


# ---- SURVEY 8(f)-2, second part: Eq. (B20) / (B30), six LFA links, no link-reversal symmetry (oracle O14) ----------

@pytest.mark.parametrize("k,n,batch,order,gen,fd", [(2, 40007, 1, 31, 15, 2), (2, 40007, 1, 31, 20, 2), (2, 40007, 1, 31, 20, 4),
                                                    (1, None, 1, 9, 15, 2), (4, 9001, 3, 9, 20, 4), (4, 9001, 3, 5, 15, 4)])
def test_lfa6_b20_b30(ltdi, orc80, k, n, batch, order, gen, fd):
    cfg = W.config(k, n=n, batch=batch) if n else W.config(k)
    idx = list(range(cfg["batch"]))
    hp, hc, ang, _ = W.sources(cfg, idx)
    orbit = cfg["orbit"]
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(orbit, device=dev)
    ref = orc80.response_lfa6(orbit, hp, hc, ang, gen, order, fd)
    out = to_numpy(ltdi.response_lfa6(orb, torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev), ang, gen, order, fd, True, True))
    lo, hi = orc80.margins_lfa6(orbit, gen, order, fd)
    assert (lo, hi) == ltdi.margins_lfa6(orbit, gen, order, fd)
    check(out, ref, lo, hi, cfg["n"])


@pytest.mark.parametrize("which", ["full", "lfa", "hybrid"])
def test_one_series_split_in_time(ltdi, which):
    """the pieces time_shard() hands to the ranks of a multi-GPU job, run here one after the other on one
    device, stitch to the whole-series response (the sub-grids start at a t0 rounded to fp64, so 1e-13, not bitwise);
    on a numerical orbit file as well, whose knots every piece shares"""
    dev = torch.device("cuda:0")
    cfg = W.config(2, n=60013)
    hp, hc, ang, metas = W.sources(cfg, [0])
    gen, order, fd = 20, 31, 2
    hyb = hybrid_params(metas, ltdi.hyb_time, W.TAPER_COSINE, cfg["dt"])
    for orbit in (cfg["orbit"], W.numerical_orbit(cfg["n"], cfg["dt"], t0=cfg["orbit"]["t0"])):
        def call(desc, p, c):
            orb = ltdi.Orbits(desc, device=dev)
            p, c = torch.from_numpy(np.ascontiguousarray(p)).to(dev), torch.from_numpy(np.ascontiguousarray(c)).to(dev)
            if which == "full":
                return to_numpy(ltdi.response_full(orb, p, c, ang, gen, order))
            if which == "lfa":
                return to_numpy(ltdi.response_lfa(orb, p, c, ang, gen, order, fd))
            return to_numpy(ltdi.response_hybrid(orb, p, c, ang, gen, order, fd, hyb))
        whole = call(orbit, hp, hc)
        lo, hi = ltdi.margins(orbit, gen, order, 0 if which == "full" else fd)
        world = 3
        got = {c: np.zeros(cfg["n"]) for c in "AET"}
        for rank in range(world):
            sub, src, dst, a, b = ltdi.time_shard(orbit, lo, hi, world, rank)
            r = call(sub, hp[:, src], hc[:, src])
            for c in "AET":
                got[c][a:b] = r[c][0, dst]
        scale = max(np.linalg.norm(whole[c]) for c in "AET")
        for c in "AET":
            assert np.linalg.norm(got[c] - whole[c][0]) <= 1e-13 * scale, (which, c)


def test_second_device_gives_the_same_bits(ltdi):
    """the library's per-device state (constant tables, shared-memory attributes, side streams, the static scratch of
    ltdi_response_static) is set up for every device it is used on: the responses on cuda:1, called after cuda:0, are bitwise
    those of cuda:0.  Needs two visible devices (skipped on the one-GPU boxes of this pool)."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    cfg = W.config(2, n=20011, batch=2)
    hp, hc, ang, metas = W.sources(cfg, [0, 1])
    results = []
    for index in (0, 1):
        dev = torch.device("cuda", index)
        hyb = hybrid_params(metas, ltdi.hyb_time, W.TAPER_COSINE, cfg["dt"])
        orb = ltdi.Orbits(cfg["orbit"], device=dev)
        dhp, dhc = torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev)
        out = []
        with torch.cuda.device(dev):
            out.append(to_numpy(ltdi.response_full(orb, dhp, dhc, ang, 20, 31)))
            out.append(to_numpy(ltdi.response_hybrid(orb, dhp, dhc, ang, 20, 31, 2, hyb)))
            out.append(to_numpy(ltdi.response_lfa(orb, dhp, dhc, ang, 20, 5, 2)))          # generic kernel: constant tables
            out.append(to_numpy(ltdi.response_static(ltdi.RESPONSE_LFA, orb, dhp, dhc, ang, 20, 31, 2)))
            torch.cuda.synchronize(dev)
        results.append(out)
    for a, b in zip(*results):
        for c in "AET":
            assert np.array_equal(a[c], b[c]), c
