"""Helpers of the GPU parity tests: run the CUDA path and the long-double oracle on the same seeded
inputs and compare channel by channel (relative L2 over the non-margin samples)."""
import json
import os

import numpy as np

import workloads as W

TOL = 1e-11           # BASELINE.json north_star: per-channel relative L2 <= 1e-11 in fp64
NEAR_NULL = 1e-6      # a channel this far below the largest one is judged against the largest
FLOOR_FACTOR = 3.0    # bar = max(TOL, FLOOR_FACTOR x fp64 floor of the algorithm)


def fp64_floor(ref80, ref64, lo, n, hi, keys=("A", "E", "T")):
    """relative L2 of the oracle's double build against its long-double build, per channel: the error any
    plain-fp64 evaluation of the paper's formulas carries on this input (T = (X + Y + Z) / sqrt 3 cancels,
    and the second difference of the gen-2.0 LFA divides the rounding noise of y by (omega dt)^2)"""
    out = {}
    for k in keys:
        d, nrm = rel_l2(ref64[k], ref80[k], lo, n - hi)
        out[k] = d / nrm if nrm > 0 else 0.0
    return out


def series_floor(ref80, ref64, lo, n, hi):
    r80, r64 = np.asarray(ref80), np.asarray(ref64)
    top = max(np.linalg.norm(r80[i][..., lo:n - hi]) for i in range(r80.shape[0]))
    return [float(np.linalg.norm((r64[i] - r80[i])[..., lo:n - hi]) / top) if top > 0 else 0.0
            for i in range(r80.shape[0])]


def rel_l2(got, want, lo, hi_end):
    g = np.asarray(got)[..., lo:hi_end]
    w = np.asarray(want)[..., lo:hi_end]
    return float(np.linalg.norm(g - w)), float(np.linalg.norm(w))


def channel_errors(gpu, ref, lo, n, hi, keys=("A", "E", "T")):
    """{key: (relative L2, flagged_near_null)}; a near-null channel (T of the LFA for equal arms is
    identically 0) is measured against the largest channel norm, as SURVEY.md 8(d) states."""
    norms, diffs = {}, {}
    for k in keys:
        diffs[k], norms[k] = rel_l2(gpu[k], ref[k], lo, n - hi)
    top = max(norms.values())
    out = {}
    for k in keys:
        near_null = norms[k] < NEAR_NULL * top
        den = top if near_null else norms[k]
        out[k] = (diffs[k] / den if den > 0 else diffs[k], near_null)
    return out


def series_errors(got, want, lo, n, hi):
    """relative L2 per leading index (links or X, Y, Z), against the largest series norm"""
    got, want = np.asarray(got), np.asarray(want)
    top = max(np.linalg.norm(want[i][..., lo:n - hi]) for i in range(want.shape[0]))
    return [float(np.linalg.norm((got[i] - want[i])[..., lo:n - hi]) / top) if top > 0 else 0.0
            for i in range(want.shape[0])]


def hybrid_params(metas, hyb_time, taper=W.TAPER_COSINE, dt=None):
    """per-source hybrid windows: t_hyb from Eq. (4.2) evaluated by the side that calls (hyb_time is
    that side's helper), cosine 1 h window (configs 2, 4) or the paper's sigmoid T = 800 dt, sigma = T / 40"""
    out = []
    for m in metas:
        th = hyb_time(m["f_hyb_hz"], m["mchirp_s"], m["t_c"])
        if taper == W.TAPER_COSINE:
            out.append({"t_hyb": th, "window_s": m["window_s"], "sigma_s": m["window_s"] / 40.0, "taper": taper})
        else:
            T = 800.0 * dt
            out.append({"t_hyb": th, "window_s": T, "sigma_s": T / 40.0, "taper": taper})
    return out


def to_numpy(out):
    return {k: (None if v is None else v.detach().cpu().numpy()) for k, v in out.items()}


REPORT = os.path.join(os.environ.get("GRAFT_REPO_ROOT", os.path.dirname(os.path.dirname(os.path.abspath(__file__)))),
                      "gpurun_out", "parity_report.jsonl")


def record(**row):
    """append one parity measurement (achieved error, fp64 floor of the oracle's double build, bar) to
    gpurun_out/parity_report.jsonl; the committed summary under profiles/ is made from this file"""
    row = {"test": os.environ.get("PYTEST_CURRENT_TEST", "").split(" ")[0], **row}
    try:
        os.makedirs(os.path.dirname(REPORT), exist_ok=True)
        with open(REPORT, "a") as f:
            f.write(json.dumps(row, default=float) + "\n")
    except OSError:
        pass
