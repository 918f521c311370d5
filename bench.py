"""bench.py -- throughput of the multi-mode difference-map (DM) iteration on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl ours|reference]

A "step" is one whole DM iteration (psi update S1-S6, object S7, probe S8, error row S9 of
DESIGN.md) over one synthetic fly-scan data set shaped like BASELINE.json config I (default
configs[1]: 2500 views of 128x128, K=2).  Prints ONE JSON line (contract in DESIGN.md
"Measurement").  N > 1 (torchrun): independent replicas, one per GPU, no data-path collective
(north_star: the path is single-GPU).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "dm_mode_views_per_s"
UNIT = "mode-views/s"


def measured_traffic(workload: str, path: int):
    """DRAM bytes per launch of the psi-update kernel from the committed ncu --set full captures
    (profiles/traffic.json, written by hand from the reports named there); None if not captured."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(p):
        return json.load(open(p)).get(f"{workload}:path{path}", {}).get("dram_bytes_per_launch")
    return None


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed regions run."""

    def __init__(self, index: int, period_s: float = 0.02):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons = index, period_s, [], set()
        self.max_mhz, self._halt, self.ok = None, threading.Event(), False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # pragma: no cover
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._halt.is_set():
            try:
                mhz = int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                util = nv.nvmlDeviceGetUtilizationRates(self.h).gpu
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.samples.append((mhz, util))
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._halt.set()
        if self.is_alive():
            self.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        loaded = [m for m, u in self.samples if u > 0] or [m for m, _ in self.samples]
        return {"sm_mhz": float(np.median(loaded)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def sample_cfg(cfg, target_mode_views: int):
    """Same N, K, L, step, jitter, probe, noise; raster cropped to ~target mode-views (bounded CPU work)."""
    from paper_1808_10375_b200 import synth  # noqa: F401
    nv = max(4, target_mode_views // (cfg.K * cfg.L))
    ny = max(2, min(cfg.ny, int(round(nv ** 0.5))))
    nx = max(2, min(cfg.nx, nv // ny))
    return cfg.scaled(ny, nx)


def time_oracle(cfg, steps: int, warmup: int, target_mode_views: int, threads: int = 0):
    """The oracle as it stands (oracle/dm_oracle.c, FP64, OpenMP over views / pixels) on the host
    cores, on a bounded sample of the workload.  Returns (mode-views/s, ms/step, cores, sample text)."""
    import oracle
    from paper_1808_10375_b200 import synth
    sc = sample_cfg(cfg, target_mode_views)
    pr = synth.make_problem(sc)
    all_threads = oracle.num_threads()
    if threads:
        oracle.set_num_threads(threads)
    o = oracle.OracleDM(sc.N, sc.K, sc.L, sc.obj_h, sc.obj_w, pr.positions)
    o.set_data(pr.intensities, pr.probe0, pr.object0)
    o.iterate(warmup)
    t0 = time.perf_counter()
    o.iterate(steps)
    dt = time.perf_counter() - t0
    cores = oracle.num_threads()
    o.close()
    if threads:
        oracle.set_num_threads(all_threads)
    sample = (f"{sc.name}: {sc.ny}x{sc.nx} raster ({sc.n_views} views, {sc.mode_views} mode-views) of "
              f"{cfg.name}, same N={sc.N} K={sc.K} L={sc.L}, {steps} iteration(s) after {warmup} warm-up")
    return sc.mode_views * steps / dt, 1e3 * dt / steps, cores, sample


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # size the per-step sample so that the whole run stays within ~2 minutes of wall time
    rate, _, _, _ = time_oracle(cfg, 1, 0, 64)
    budget = int(120.0 * rate / max(1, args.steps + args.warmup))
    v, ms, cores, sample = time_oracle(cfg, args.steps, args.warmup, max(64, min(args.ref_mode_views, budget)))
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "N": cfg.N, "K": cfg.K, "L": cfg.L, "sample": sample},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args, cfg):
    import torch
    from paper_1808_10375_b200 import dm, synth

    from paper_1808_10375_b200.replicas import ReplicaGroup
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    grp = ReplicaGroup("nccl", torch.device("cuda", local))
    world, rank = grp.world, grp.rank
    dm.lib()

    # every rank reconstructs its own data set (replicas; seed = rank)
    pr = synth.make_problem(cfg, seed=grp.seed)
    plan = dm.DMPlan(cfg.N, cfg.n_views, cfg.K, cfg.L, cfg.obj_h, cfg.obj_w, pr.positions,
                     path=args.path, **({"lag": args.lag} if args.lag else {})).alloc_workspace()
    I_h = torch.from_numpy(pr.intensities).pin_memory()
    P_h = torch.from_numpy(pr.probe0).pin_memory()
    O_h = torch.from_numpy(pr.object0).pin_memory()
    Pout_h = torch.empty_like(P_h).pin_memory()
    Oout_h = torch.empty_like(O_h).pin_memory()
    I_d, P_d, O_d = I_h.cuda(), P_h.cuda(), O_h.cuda()
    stream = torch.cuda.current_stream()

    barrier, max_over_ranks = grp.barrier, grp.max_over_ranks

    sampler = ClockSampler(local)
    sampler.start()

    # ---- device-resident arm: inputs already in HBM, K iterations timed with CUDA events ----
    plan.set_data(I_d, P_d, O_d)
    plan.iterate(args.warmup)
    plan.set_profiling(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    plan.iterate(args.steps)
    e1.record(stream)
    barrier()
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    phase_ms, n_prof = plan.phase_ms()
    plan.set_profiling(False)
    info = plan.info()

    # ---- end-to-end arm: HOST (pinned) buffers through dm_solve_host, copies inside the timing ----
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    for _ in range(2):
        plan.solve_host(I_h, P_h, O_h, 1, Pout_h, Oout_h)
    barrier()
    e0.record(stream)
    for _ in range(e2e_steps):
        plan.solve_host(I_h, P_h, O_h, 1, Pout_h, Oout_h)
    e1.record(stream)
    barrier()
    ms_e2e = max_over_ranks(e0.elapsed_time(e1))
    clocks = sampler.stop()

    if rank != 0:
        grp.close()
        return

    MV, NN = cfg.mode_views, cfg.N * cfg.N
    ms_step = ms_total / args.steps
    value = grp.aggregate(MV, args.steps, ms_total)
    peak, peak_src = measured_peaks()
    psi_bytes = MV * NN * 16 + cfg.n_views * NN * 4          # psi read + write + sqrt(I) read
    psi_ms = phase_ms[0] / max(n_prof, 1)
    achieved = psi_bytes / (psi_ms * 1e-3) / 1e9
    bmin = 3 * MV * NN * 8 + cfg.n_views * NN * 4            # whole iteration
    h2d = I_h.numel() * 4 + P_h.numel() * 8 + O_h.numel() * 8
    d2h = Pout_h.numel() * 8 + Oout_h.numel() * 8
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "iterations_per_s": 1e3 / ms_step,
        "config": {"workload": cfg.name, "N": cfg.N, "n_views": cfg.n_views, "K": cfg.K, "L": cfg.L,
                   "object": [cfg.obj_h, cfg.obj_w], "mode_views": MV, "path": info["path"],
                   "parallelism": "replicas" if world > 1 else "single-gpu",
                   "l2": f"inputs larger than L2 (psi {MV * NN * 8 / 2**20:.0f} MiB streamed every step)"
                         if MV * NN * 8 > 2 * 126 * 2**20 else "psi fits L2: latency-bound case, no flush"},
        "roofline": {"bound": "hbm", "kernel": "psi update (S1-S6)", "achieved": achieved, "peak": peak,
                     "unit": "GB/s", "frac": achieved / peak, "traffic": measured_traffic(cfg.name, info["path"]),
                     "peak_source": peak_src,
                     "bytes_per_launch": psi_bytes, "ms_per_launch": psi_ms},
        "iteration_roofline": {"bytes_min": bmin, "achieved_gbs": bmin / (ms_step * 1e-3) / 1e9,
                               "frac_of_measured_hbm": bmin / (ms_step * 1e-3) / 1e9 / peak},
        "phase_ms_per_step": {k: float(v) / max(n_prof, 1) for k, v in
                              zip(("psi_update", "object", "probe", "errors"), phase_ms)},
        "e2e": {"value": grp.aggregate(MV, e2e_steps, ms_e2e), "unit": UNIT, "steps": e2e_steps,
                "ms_per_step": ms_e2e / e2e_steps, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "call": "dm_solve_host(n_iter=1): H2D intensities+P0+O0 (pinned), set_data, 1 iteration, D2H P+O"},
        "gpu_launches": info["launches_per_iter"] * args.steps,
        "clocks": clocks,
    }
    if world == 1 and not args.no_cpu_baseline:
        v, ms, cores, sample = time_oracle(cfg, 1, 1, args.ref_mode_views)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                "ms_per_step": ms}
        # one host thread, smaller sample: context for the paper's single-core figure
        v1, ms1, c1, sample1 = time_oracle(cfg, 1, 0, max(64, args.ref_mode_views // 16), threads=1)
        line["cpu_baseline_1thread"] = {"value": v1, "unit": UNIT, "cores": c1, "kind": "oracle", "sample": sample1,
                                        "ms_per_step": ms1}
    print(json.dumps(line), flush=True)
    grp.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json config index (default 1)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--path", type=int, default=0, help="0 auto, 1 staged, 2 fused")
    ap.add_argument("--lag", type=int, default=0, help="path 4: phase lag in views (0 = derived)")
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--ref-mode-views", type=int, default=4096,
                    help="size of the bounded oracle sample (mode-views per iteration)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    from paper_1808_10375_b200 import synth
    cfg = synth.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        if args.warmup < 3:
            args.warmup = 3
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
