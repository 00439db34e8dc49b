"""GPU parity of SURVEY 8(f)-4, third part: the full response in the Sagnac combinations alpha, beta, gamma
(ltdi_response_full_sagnac) against the long-double oracle O15, at the bar of the hot path."""
import numpy as np
import pytest
import torch

import workloads as W
from parity_util import strict_check, to_numpy

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ltdi():
    import paper_2505_09600_b200 as m
    assert torch.cuda.is_available(), "GPU parity tests need a CUDA device"
    return m


def run(ltdi, orc, cfg, orbit, gen, order):
    hp, hc, ang, _ = W.sources(cfg, list(range(cfg["batch"])))
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(orbit, device=dev)
    out = ltdi.response_full_sagnac(orb, torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev), ang, gen, order, True, True)
    torch.cuda.synchronize()
    ref = orc.response_full_sagnac(orbit, hp, hc, ang, gen, order)
    lo, hi = orc.margins(orbit, gen, order, 0)
    return to_numpy(out), ref, lo, hi


@pytest.mark.parametrize("k,n,batch,gen", [(1, None, 1, 15), (2, 30011, 1, 20), (2, 30011, 1, 15), (4, 9001, 3, 20),
                                           (5, 20003, 2, 20)])
def test_sagnac_on_the_analytic_orbit(ltdi, orc80, k, n, batch, gen):
    """config 1 in its own generation (BASELINE.json: TDI 1.5): at 1 mHz the 12-term combination is 4e-4 of the links and the
    oracle's own double build is 1.9e-10 from its long-double build there, which a plain-fp64 kernel cannot beat"""
    cfg = W.config(k, n=n, batch=batch) if n else W.config(k)
    out, ref, lo, hi = run(ltdi, orc80, cfg, cfg["orbit"], gen, cfg["order"])
    strict_check(out, ref, lo, hi, cfg["n"])
    # the combination is not the Michelson one: alpha differs from X at the level of the signal
    assert np.abs(out["XYZ"]).max() > 0


@pytest.mark.parametrize("order", [5, 9])
def test_sagnac_other_orders_and_the_orbit_file(ltdi, orc80, order):
    cfg = W.config(2, n=20011)
    cfg["order"] = order
    orbit = W.numerical_orbit(cfg["n"], cfg["dt"], t0=cfg["orbit"]["t0"])
    out, ref, lo, hi = run(ltdi, orc80, cfg, orbit, 20, order)
    strict_check(out, ref, lo, hi, cfg["n"])


def test_sagnac_differs_from_michelson_and_errors(ltdi):
    cfg = W.config(2, n=8001)
    hp, hc, ang, _ = W.sources(cfg, [0])
    dev = torch.device("cuda:0")
    orb = ltdi.Orbits(cfg["orbit"], device=dev)
    dhp, dhc = torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev)
    s = to_numpy(ltdi.response_full_sagnac(orb, dhp, dhc, ang, 20, 31, True, False))
    m = to_numpy(ltdi.response_full(orb, dhp, dhc, ang, 20, 31, True, False))
    assert np.abs(s["XYZ"] - m["XYZ"]).max() > 0.1 * np.abs(m["XYZ"]).max()
    with pytest.raises(ltdi.LtdiError):
        ltdi.response_full_sagnac(orb, dhp, dhc, ang, 17, 31)
    with pytest.raises(ltdi.LtdiError):
        ltdi.response_full_sagnac(orb, dhp, dhc, ang, 20, 8)
