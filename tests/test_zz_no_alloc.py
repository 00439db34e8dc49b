"""ltdi_response_static: the responses with the library's scratch in a static device array (no allocation by the call),
against the existing calls that take a workspace from the caller, at the tolerance of the parity tests (1e-11 relative
L2 per channel; T against the largest channel).  Collected last on purpose: the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

import workloads as W
from parity_util import hybrid_params

pytestmark = pytest.mark.gpu
TOL = 1e-11


@pytest.fixture(scope="module")
def ltdi():
    import paper_2505_09600_b200 as m
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return m


def close(got, want):
    top = max(float(torch.linalg.norm(want[c])) for c in "AET")
    assert top > 0.0
    worst = 0.0
    for c in "AET":
        ref = float(torch.linalg.norm(want[c]))
        err = float(torch.linalg.norm(got[c] - want[c]))
        worst = max(worst, err / (ref if c != "T" and ref > 0 else top))
    return worst


def case(ltdi, k, n, batch, which, gen, order=None, fd=2):
    dev = torch.device("cuda:0")
    cfg = W.config(k, n=n, batch=batch) if n else W.config(k)
    hp, hc, ang, metas = W.sources(cfg, list(range(cfg["batch"])))
    order = order or cfg["order"]
    orb = ltdi.Orbits(cfg["orbit"], device=dev)
    dhp, dhc = torch.from_numpy(hp).to(dev), torch.from_numpy(hc).to(dev)
    hyb = hybrid_params(metas, ltdi.hyb_time, W.TAPER_COSINE, cfg["dt"]) if which == "hybrid" else None
    code = {"full": ltdi.RESPONSE_FULL, "lfa": ltdi.RESPONSE_LFA, "hybrid": ltdi.RESPONSE_HYBRID}[which]

    def existing():
        if which == "full":
            r = ltdi.response_full(orb, dhp, dhc, ang, gen, order)
        elif which == "lfa":
            r = ltdi.response_lfa(orb, dhp, dhc, ang, gen, order, fd)
        else:
            r = ltdi.response_hybrid(orb, dhp, dhc, ang, gen, order, fd, hyb)
        return {c: r[c].clone() for c in "AET"}

    def static():
        return ltdi.response_static(code, orb, dhp, dhc, ang, gen, order, fd, hyb)
    return existing, static


def test_two_calls_in_a_row_match_the_workspace_path(ltdi):
    """different responses, grids, batch sizes and Lagrange orders one after the other, with no synchronisation in between
    (same stream: they serialise): the second call finds the first one's contents in the shared array, laid out differently"""
    cases = [case(ltdi, 2, 30011, 3, "hybrid", 20),
             case(ltdi, 4, 9001, 2, "full", 20),
             case(ltdi, 1, None, 1, "full", 15),          # order 9, static equal arms
             case(ltdi, 2, 20011, 2, "lfa", 20, fd=4),
             case(ltdi, 2, 12007, 1, "full", 20, order=5)]   # the generic tile kernel
    want = [existing() for existing, _ in cases]
    got = [static() for _, static in cases]                # back to back
    again = [static() for _, static in cases[:2]]
    torch.cuda.synchronize()
    for i, (g, w) in enumerate(zip(got, want)):
        assert close(g, w) <= TOL, (i, close(g, w))
    for i, (g, w) in enumerate(zip(again, want[:2])):
        assert close(g, w) <= TOL, ("again", i, close(g, w))


def test_sizes_beyond_the_static_array_are_refused(ltdi):
    dev = torch.device("cuda:0")
    n, batch = 131072, 64                                  # 12 link rows x 64 x 1 MiB: 800 MB of scratch
    cfg = W.config(4, n=n, batch=2)
    orb = ltdi.Orbits(cfg["orbit"], device=dev)
    import ctypes as C
    need = C.c_size_t()
    assert ltdi.lib().ltdi_workspace_bytes(ltdi.RESPONSE_HYBRID, n, batch, 20, 31, C.byref(need)) == ltdi.OK
    assert need.value > ltdi.STATIC_SCRATCH_BYTES
    hp = torch.zeros(batch, n, dtype=torch.float64, device=dev)
    ang = np.tile(np.array([[0.1, 0.2, 0.3]]), (batch, 1))
    hyb = {"t_hyb": cfg["orbit"]["t0"] + 0.5 * n * cfg["dt"], "window_s": 3600.0, "sigma_s": 90.0, "taper": W.TAPER_COSINE}
    out = {c: torch.full((batch, n), 7.0, dtype=torch.float64, device=dev) for c in "AET"}
    before = ltdi.launch_count()
    with pytest.raises(ltdi.LtdiError) as e:
        ltdi.response_static(ltdi.RESPONSE_HYBRID, orb, hp, hp, ang, 20, 31, 2, hyb, out=out)
    assert e.value.code == ltdi.EWORKSPACE
    assert ltdi.launch_count() == before and float(out["A"].min()) == 7.0     # nothing was launched or written
    with pytest.raises(ltdi.LtdiError):
        ltdi.response_static(7, orb, hp, hp, ang, 20, 31)
    # and the entry point still works afterwards
    existing, static = case(ltdi, 2, 9001, 2, "hybrid", 20)
    w, g = existing(), static()
    torch.cuda.synchronize()
    assert close(g, w) <= TOL
