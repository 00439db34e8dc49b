#!/usr/bin/env python
"""bench.py -- throughput of the time-domain LISA response hot path on B200 (one JSON line).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg2|cfg4s|...]

A *step* is one pass of the whole hot path over one batch of synthetic input:
the orbit/delay kernel, then the full, LFA and hybrid responses (TDI 2.0, Lagrange order 31) of the
workload.  The default workload is BASELINE.json configs[1] ("cfg2": one MBHB merger, 30 days at dt = 5 s,
518 400 samples).  metric = TDI output samples/s: (samples x sources x 3 responses x ranks) / step time.

--impl reference times the CPU oracle (oracle/, as it stands, double build) on a bounded sample of the
same workload on the host cores; it is the deliberately slow baseline, not a target.
"""
import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

GEN, FD = 20, 2
# algorithmic flops per output sample (SURVEY.md 8(a)/(d), M = order + 1 taps; stated in DESIGN.md):
#   full 2.0: 72 M + 252 M + 200,  LFA: 60 M + 150
FLOPS_FULL = lambda M: 72 * M + 252 * M + 200
FLOPS_LFA = lambda M: 60 * M + 150
# the same model split per kernel: flops per output sample of one launch
KERNEL_FLOPS = {
    ("full", "link_full"): lambda M: 72 * M + 200,    # S2 + S3: 9 retarded times x (weights 4M + two dots 4M)
    ("full", "tdi"): lambda M: 252 * M,               # S4 + S5: 3 channels x 14 interpolations x 6M
    ("lfa", "link_lfa"): lambda M: 24 * M + 150,      # S6: 3 retarded times x 8M
    ("lfa", "tdi"): lambda M: 36 * M,                 # S7: 3 channels x 2 interpolations x 6M
}

# flops the kernels actually execute per output sample: the TDI kernel shares the weights of a
# term over an anchor tile and spends 2 DFMA (4 flop) per tap and sample where the model above counts 6 flop of
# per-sample weights and dot product; the link kernels execute what the model counts
KERNEL_EXEC_FLOPS = {
    ("full", "tdi"): lambda M: 3 * 14 * 4 * M,
    ("lfa", "tdi"): lambda M: 3 * 2 * 4 * M,
}

# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` capture
# (profiles/), cfg2 only; None where no capture exists for the kernel
TRAFFIC = {"full/tdi": 74.6e6 + 3.2e6}    # profiles/r01f_cfg2.md, tdi_kernel<32,FULL>, cfg2
# sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active of the same capture (context, cfg2 only; with the
# device filled, cfg4s: link_full 67.6, tdi full 70.6, link_lfa 57.7, tdi LFA 48.1)
FP64_PIPE_PCT_NCU = {"full/orbit": 53.6, "full/anchor": 12.0, "full/link_full": 62.4, "full/tdi": 65.8,
                     "lfa/link_lfa": 48.5, "lfa/tdi": 43.0, "hybrid/link_full": 45.8, "hybrid/tdi": 42.1}

WORKLOADS = {
    # name: (config index, n, batch)  -- None = BASELINE.json size
    "cfg2": (2, None, None),
    "cfg1": (1, None, None),
    "cfg1f": (1, None, 4096),    # config 1 with the device filled: 4096 sources with fresh angles
    "cfg3": (3, None, None),     # 1 year at dt = 5 s, one source
    "cfg4s": (4, None, 256),     # a 256-source slice of config 4 (the full 4096 x 131072 needs 21 GB of buffers)
    "cfg4": (4, None, None),     # config 4 at full size: 4096 sources (about 90 GB of device and 35 GB of pinned memory)
    "cfg5s": (5, None, 16),
}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def make_inputs(workload, rank):
    import workloads as W
    k, n, batch = WORKLOADS[workload]
    cfg = W.config(k, n=n, batch=batch)
    idx = [rank * cfg["batch"] + i for i in range(cfg["batch"])]   # every rank gets its own sources
    hp, hc, ang, metas = W.sources(cfg, idx)
    return cfg, hp, hc, ang, metas


def windows(metas, hyb_time):
    return [{"t_hyb": hyb_time(m["f_hyb_hz"], m["mchirp_s"], m["t_c"]), "window_s": m["window_s"],
             "sigma_s": m["window_s"] / 40.0, "taper": m["taper"]} for m in metas]


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe) through NVML
    from a polling thread (the timed region of the single-source workloads lasts tens of milliseconds, too
    short for `nvidia-smi -lms`); falls back to one nvidia-smi query if NVML cannot be loaded."""
    REASONS = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

    def __init__(self, index, period_s=0.002):
        import threading
        self.rows, self.stop_flag, self.nvml, self.h = [], threading.Event(), None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            visible = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(visible.split(",")[index]) if visible and visible.split(",")[index].isdigit() else index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.nvml = pynvml
        except Exception:
            self.nvml = None
        self.index, self.period = index, period_s
        self.thread = threading.Thread(target=self._poll, daemon=True)
        self.thread.start()

    def _poll(self):
        nv = self.nvml
        while nv is not None and not self.stop_flag.is_set():
            try:
                self.rows.append((nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM),
                                  nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h),
                                  nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0))
            except Exception:
                break
            time.sleep(self.period)

    def stop(self):
        self.stop_flag.set()
        self.thread.join(timeout=2)
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": len(self.rows)}
        nv = self.nvml
        if nv is not None and self.rows:
            out["sm_mhz"] = float(np.median([r[0] for r in self.rows]))
            out["sm_max_mhz"] = float(nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM))
            out["power_w_max"] = max(r[2] for r in self.rows)
            out["reasons"] = [k for k, bit in self.REASONS.items() if any(r[1] & bit for r in self.rows)]
            out["how"] = "NVML polled every %g ms during the timed region" % (1e3 * self.period)
            return out
        try:
            q = "clocks.sm,clocks.max.sm,power.draw"
            r = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                               capture_output=True, text=True, timeout=10).stdout.strip().split(",")
            out.update(sm_mhz=float(r[0]), sm_max_mhz=float(r[1]), power_w_max=float(r[2]),
                       how="one nvidia-smi query after the timed region (NVML unavailable)")
        except Exception:
            pass
        return out


def cpu_baseline(cfg, hp, hc, ang, metas, budget_samples):
    """The oracle as it stands (double build, OpenMP) on a bounded tail sample of source 0."""
    import workloads as W
    from oracle import Oracle
    orc = Oracle("f64")
    n = min(cfg["n"], budget_samples)
    a = cfg["n"] - n
    orbit = W.orbit_desc(n, cfg["dt"], cfg["mode"], t0=cfg["orbit"]["t0"] + a * cfg["dt"])
    h0, h1 = np.ascontiguousarray(hp[:1, a:]), np.ascontiguousarray(hc[:1, a:])
    hyb = windows(metas[:1], orc.hyb_time)
    order = cfg["order"]
    t0 = time.perf_counter()
    orc.response_full(orbit, h0, h1, ang[:1], GEN, order, want=())
    orc.response_lfa(orbit, h0, h1, ang[:1], GEN, order, FD, want=())
    orc.response_hybrid(orbit, h0, h1, ang[:1], GEN, order, FD, hyb, want=())
    sec = time.perf_counter() - t0
    return {"value": 3 * n / sec, "unit": "TDI samples/s", "cores": orc.num_threads(), "kind": "oracle",
            "sample": f"last {n} samples of source 0 of {cfg['name']}: full + LFA + hybrid, TDI 2.0, order {order}, "
                      f"double build, {sec:.1f} s"}, sec


def run_reference(args, rank):
    if rank != 0:
        return
    cfg, hp, hc, ang, metas = make_inputs(args.workload, 0)
    sample = 20000
    for _ in range(args.warmup):
        cpu_baseline(cfg, hp, hc, ang, metas, 2000)
    secs, base = [], None
    for _ in range(args.steps):
        base, s = cpu_baseline(cfg, hp, hc, ang, metas, sample)
        secs.append(s)
    n = min(cfg["n"], sample)
    value = 3 * n * len(secs) / sum(secs)
    base["value"] = value
    line = {"impl": "reference", "metric": "TDI output samples/s (full + LFA + hybrid)", "value": value,
            "unit": "TDI samples/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * sum(secs) / len(secs), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "sample": base["sample"]},
            "cpu_baseline": base,
            "e2e": {"value": value, "unit": "TDI samples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        return run_reference(args, rank)

    import torch
    import torch.distributed as dist
    import paper_2505_09600_b200 as ltdi
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg, hp, hc, ang, metas = make_inputs(args.workload, rank)
    n, batch, order = cfg["n"], cfg["batch"], cfg["order"]
    M = order + 1
    hyb = windows(metas, ltdi.hyb_time)
    hp_host, hc_host = torch.from_numpy(hp).pin_memory(), torch.from_numpy(hc).pin_memory()
    d_hp, d_hc = hp_host.to(dev), hc_host.to(dev)
    ws = ltdi.Workspace(batch, n, dev)
    orb = ltdi.Orbits(cfg["orbit"], device=dev)
    anchors = orb.prepare(GEN, order)._anchors      # reused by every step: the step allocates only the orbit table
    flush = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)   # 256 MB > 126 MB L2

    ev = lambda: torch.cuda.Event(enable_timing=True)
    per_call = {"orbit": [], "full": [], "lfa": [], "hybrid": []}

    def step(record):
        nonlocal orb
        marks = [ev() for _ in range(5)]
        marks[0].record()
        orb = ltdi.Orbits(cfg["orbit"], device=dev).prepare(GEN, order, buffer=anchors)    # S0 (+ TDI weights)
        marks[1].record()
        ltdi.response_full(orb, d_hp, d_hc, ang, GEN, order, workspace=ws)                 # S1-S5
        marks[2].record()
        ltdi.response_lfa(orb, d_hp, d_hc, ang, GEN, order, FD, workspace=ws)              # S6-S7
        marks[3].record()
        ltdi.response_hybrid(orb, d_hp, d_hc, ang, GEN, order, FD, hyb, workspace=ws)      # S8
        marks[4].record()
        if record:
            return marks
        return None

    for _ in range(args.warmup):
        flush.zero_()
        step(False)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = ClockSampler(local_rank) if rank == 0 else None
    launches0 = ltdi.launch_count()
    all_marks = []
    wall0 = time.perf_counter()
    for _ in range(args.steps):
        flush.zero_()                      # evict the 126 MB L2 between timed steps (outside the events)
        all_marks.append(step(True))
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    launches = ltdi.launch_count() - launches0
    if world > 1:
        dist.barrier()
    clk = clocks.stop() if clocks else None
    step_ms = []
    for m in all_marks:
        step_ms.append(m[0].elapsed_time(m[4]))
        for name, i in (("orbit", 0), ("full", 1), ("lfa", 2), ("hybrid", 3)):
            per_call[name].append(m[i].elapsed_time(m[i + 1]))
    total_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_ms = float(total_ms.item())
    ms_per_step = total_ms / args.steps
    samples_per_step = 3 * n * batch * world
    value = samples_per_step / (ms_per_step * 1e-3)

    # per-kernel device times: the same K steps again with the library's per-kernel CUDA events switched on
    # (events recorded on the launching stream around every kernel; ltdi_profile_* in include/lisatdi.h)
    ltdi.profile_reset()
    ltdi.profile_enable(True)
    for _ in range(args.steps):
        flush.zero_()
        step(False)
    torch.cuda.synchronize()
    ltdi.profile_enable(False)
    prof = ltdi.profile_read()

    # end to end: host buffers in, host A, E, T out, through ltdi_response_host (copies inside the timed region)
    # two slots: the device->host copy of one response overlaps the upload and the kernels of the next
    pipe = ltdi.HostPipeline(orb, batch, n, depth=2)
    for _ in range(2):
        pipe.run(ltdi.RESPONSE_FULL, hp_host, hc_host, ang, GEN, order)
    pipe.synchronize()
    torch.cuda.synchronize()
    e0, e1 = ev(), ev()
    k_e2e = max(3, min(args.steps, 10))
    e0.record()
    for _ in range(k_e2e):
        pipe.run(ltdi.RESPONSE_FULL, hp_host, hc_host, ang, GEN, order)
        pipe.run(ltdi.RESPONSE_LFA, hp_host, hc_host, ang, GEN, order, FD)
        pipe.run(ltdi.RESPONSE_HYBRID, hp_host, hc_host, ang, GEN, order, FD, hyb)
    pipe.join()
    e1.record()
    e1.synchronize()
    e2e_ms = torch.tensor([e0.elapsed_time(e1) / k_e2e], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(e2e_ms, op=dist.ReduceOp.MAX)
    e2e_value = samples_per_step / (float(e2e_ms.item()) * 1e-3)

    # next row: FFT -> noise-weighted inner products of the full and the hybrid response (steps
    # iv-v of P:408); reported beside the step, not part of `value`
    keep = lambda d: {k: v.clone() for k, v in d.items() if k in "AET"}
    r_full = keep(ltdi.response_full(orb, d_hp, d_hc, ang, GEN, order, workspace=ws))
    r_hyb = keep(ltdi.response_hybrid(orb, d_hp, d_hc, ang, GEN, order, FD, hyb, workspace=ws))
    ovl = ltdi.Overlap(n, n, batch, dev)
    psd = ovl.psd(cfg["dt"], GEN)
    for _ in range(2):
        ovl.products(r_full, r_hyb, cfg["dt"], psd, 1e-4, 2e-2)
    torch.cuda.synchronize()
    k_ovl = max(3, min(args.steps, 20))
    o0, o1 = ev(), ev()
    o0.record()
    for _ in range(k_ovl):
        o_out, o_snr = ovl.products(r_full, r_hyb, cfg["dt"], psd, 1e-4, 2e-2)
    o1.record()
    o1.synchronize()
    ovl_ms = o0.elapsed_time(o1) / k_ovl
    o_out, o_snr = o_out.cpu().numpy(), o_snr.cpu().numpy()
    overlap_row = {"ms_per_call": ovl_ms, "samples_per_s": 2.0 * n * batch / (ovl_ms * 1e-3),
                   "what": "6 FFTs (A, E, T of the full and of the hybrid response) + Eq. (5.1) products, overlap, "
                           "mismatch, SNR per source; band 1e-4 .. 2e-2 Hz, Sangria PSD with galactic foreground",
                   "spectrum_gbs": 6.0 * 16.0 * (n // 2 + 1) * batch / (ovl_ms * 1e-3) / 1e9,
                   "mismatch_hybrid_vs_full_AET_source0": [float(x) for x in o_out[0, :, 4]],
                   "max_mismatch_AE": float(np.nanmax(o_out[:, :2, 4])),
                   "snr_full_source0": float(o_snr[0, 0]),
                   "lnL_full_as_data_hybrid_as_template_source0": float(o_snr[0, 2])}
    del r_full, r_hyb, ovl

    if rank == 0:
        # roofline of the dominant kernel: the fused response kernel in its full-response launch
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except OSError:
            pass
        dfma_rate = ltdi.fp64_probe(device=dev)
        peak_tflops = 2.0 * dfma_rate / 1e12
        # per launch: device ms (mean over the profiled steps) and achieved algorithmic TFLOP/s per kernel
        kernels = {}
        for resp, ks in prof.items():
            for name, (ms, cnt) in ks.items():
                per_step = ms / args.steps                      # all launches of this kernel in one step
                ent = {"ms_per_step": per_step, "launches_per_step": cnt / args.steps}
                fl = KERNEL_FLOPS.get((resp, name))
                if fl is not None:
                    ent["tflops"] = fl(M) * n * batch / (per_step * 1e-3) / 1e12
                    ent["frac_of_dfma_peak"] = ent["tflops"] / peak_tflops
                    fe = KERNEL_EXEC_FLOPS.get((resp, name))
                    if fe is not None:   # the same with the flops the kernel really executes
                        ent["frac_executed_flops"] = fe(M) * n * batch / (per_step * 1e-3) / 1e12 / peak_tflops
                if name == "orbit":
                    ent["gbs"] = 192.0 * n / (per_step * 1e-3) / 1e9
                    ent["frac_of_hbm_measured"] = ent["gbs"] / peaks["hbm_gbs"] if peaks.get("hbm_gbs") else None
                kernels[f"{resp}/{name}"] = ent
        dom = max(kernels, key=lambda k: kernels[k]["ms_per_step"])       # the dominant kernel of the step
        if "tflops" not in kernels[dom]:
            dom = max((k for k in kernels if "tflops" in kernels[k]), key=lambda k: kernels[k]["ms_per_step"])
        achieved = kernels[dom]["tflops"]
        full_ms = float(np.mean(per_call["full"]))
        roofline = {"bound": "alu", "kernel": dom + " (response/kernel; see include/lisatdi.h LTDI_KERNEL_*)",
                    "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s", "frac": achieved / peak_tflops,
                    "frac_executed_flops": kernels[dom].get("frac_executed_flops"),
                    "note": "achieved = algorithmic flops of the SURVEY 8(d) model (per-sample weights 4M + dot 2M per "
                            "interpolation); the TDI kernel executes 4M of them (weights shared over an anchor tile), "
                            "so frac can exceed the FP64 pipe utilisation ncu reports (fp64_pipe_pct_ncu_cfg2) and 1",
                    "traffic": TRAFFIC.get(dom) if args.workload == "cfg2" else None,
                    "fp64_pipe_pct_ncu_cfg2": FP64_PIPE_PCT_NCU,
                    "peak_source": "DFMA chain probe measured in this run (2 flop per DFMA); nominal 148 SM x 64 DFMA/clk",
                    "timed_with": "per-kernel CUDA events on the launching stream (ltdi_profile_*), over %d steps "
                                  "identical to the timed ones, run right after them" % args.steps,
                    "peak_nominal": 148 * 64 * 2 * ((clk or {}).get("sm_max_mhz") or 1965.0) * 1e6 / 1e12,
                    "hbm_gbs_measured": peaks.get("hbm_gbs"),
                    "kernels": kernels,
                    "per_call_ms": {k: float(np.mean(v)) for k, v in per_call.items()},
                    "full_call_tflops": FLOPS_FULL(M) * n * batch / (full_ms * 1e-3) / 1e12,
                    "lfa_call_tflops": FLOPS_LFA(M) * n * batch / (float(np.mean(per_call["lfa"])) * 1e-3) / 1e12}
        line = {"metric": "TDI output samples/s (full + LFA + hybrid)", "value": value, "unit": "TDI samples/s",
                "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic",
                "config": {"workload": cfg["name"], "samples": n, "sources_per_gpu": batch, "dt_s": cfg["dt"],
                           "tdi": "2.0", "lagrange_order": order, "fd_order": FD, "responses": "full+lfa+hybrid",
                           "orbit_kernel_in_step": True, "l2": "flushed between steps (256 MB write)",
                           "wall_s_timed_region": wall},
                "clocks": clk, "gpu_launches": int(launches),
                "e2e": {"value": e2e_value, "unit": "TDI samples/s", "h2d_bytes_per_step": 3 * pipe.h2d_bytes,
                        "d2h_bytes_per_step": 3 * pipe.d2h_bytes},
                "roofline": roofline, "next_rows": {"overlap": overlap_row}}
        if world == 1 and not args.no_cpu_baseline:
            # ~10 s of CPU work: the oracle over the last <= 600 000 samples of source 0, repeated until 10 s have passed
            base, sec, reps = None, 0.0, 0
            while sec < 10.0 and reps < 4096:
                base, s1 = cpu_baseline(cfg, hp, hc, ang, metas, 600000)
                sec += s1
                reps += 1
            nsmp = min(cfg["n"], 600000)
            base["value"] = 3 * nsmp * reps / sec
            base["sample"] = base["sample"].rsplit(",", 1)[0] + f", {reps} passes, {sec:.1f} s"
            line["cpu_baseline"] = base
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
