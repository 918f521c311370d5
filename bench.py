"""bench.py -- throughput of the multi-mode difference-map (DM) iteration on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl ours|reference]

A "step" is one whole DM iteration (psi update S1-S6, object S7, probe S8, error row S9 of
DESIGN.md) over one synthetic fly-scan data set shaped like BASELINE.json config I.  The headline
workload is the largest single-GPU config (default configs[3]: 4096 views of 256x256, K=4, L=2;
BASELINE.json's metric names no config); the other single-GPU configs (1, 2, 4) are measured in the
same run and reported under "per_config".  Prints ONE JSON line (contract in DESIGN.md
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


def csrc_digest() -> str:
    """sha256 over the CUDA sources, in file-name order: ties a stored ncu number to the kernels it was taken on."""
    import glob
    import hashlib
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_1808_10375_b200", "csrc", "*"))):
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def measured_traffic(workload: str, path: int, lag: int):
    """DRAM bytes per launch of the psi-update kernel (dram__bytes_read.sum + dram__bytes_write.sum) from the
    committed ncu capture of exactly these kernels: profiles/traffic.json keeps, per workload and path, the bytes,
    the digest of csrc/ they were captured on and path 4's lag.  Returns (bytes, provenance); (None, why) when no
    capture matches the sources and launch parameters of this run -- a stale number is never reported."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None, "no capture"
    e = json.load(open(p)).get(f"{workload}:path{path}")
    if not e:
        return None, "no capture for this workload / path"
    if e.get("csrc_digest") != csrc_digest():
        return None, f"capture {e.get('source')} was taken on other kernel sources (digest {e.get('csrc_digest')})"
    if path == 4 and e.get("lag") != lag:
        return None, f"capture was taken at lag {e.get('lag')}, this run uses {lag}"
    return e["dram_bytes_per_launch"], {"file": "profiles/traffic.json", "source": e.get("source"),
                                         "csrc_digest": e.get("csrc_digest"), "kind": "committed ncu capture, not measured in this run"}


# FP32 lane-operations (FADD / FMUL / FFMA lanes, a packed f32x2 instruction = two) per pixel and mode of the psi
# update.  Measured values are executed-instruction counts of an ncu capture of exactly these kernels
# (profiles/traffic.json, "lane_ops_per_pixel_mode", same csrc digest rule as the DRAM bytes); without a matching
# capture the figures below are used and the line says "estimated": 109 was counted on path 3 (N = 128) in round 2,
# the others are +/- 11-12 per octave of N (one radix-2 stage more or less in each of the four 1-D FFTs).
LANE_OPS_ESTIMATE = {64: 98, 128: 109, 256: 120, 512: 132}


def lane_ops_per_pixel(workload: str, path: int, N: int):
    """(lane-operations per pixel and mode, provenance text)."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(p):
        e = json.load(open(p)).get(f"{workload}:path{path}")
        if e and e.get("csrc_digest") == csrc_digest() and e.get("lane_ops_per_pixel_mode"):
            return float(e["lane_ops_per_pixel_mode"]), f"measured: ncu executed FADD/FMUL/FFMA lanes, {e.get('source')}"
    return float(LANE_OPS_ESTIMATE[N]), "estimated (no ncu capture of these kernel sources for this workload)"


NOMINAL_HBM_GBS = 8000.0      # north_star / SURVEY.md 8(d): "~8 TB/s"


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


def measure_device_arm(dm, synth, torch, grp, cfg, pr, steps, warmup, path, lag, stream):
    """Device-resident arm on one config: inputs already in HBM, `steps` whole DM iterations timed with CUDA
    events on the launching stream after `warmup` untimed ones.  Returns (plan, host tensors, result dict)."""
    plan = dm.DMPlan(cfg.N, cfg.n_views, cfg.K, cfg.L, cfg.obj_h, cfg.obj_w, pr.positions,
                     path=path, **({"lag": lag} if lag else {})).alloc_workspace()
    I_h = torch.from_numpy(pr.intensities).pin_memory()
    P_h = torch.from_numpy(pr.probe0).pin_memory()
    O_h = torch.from_numpy(pr.object0).pin_memory()
    I_d, P_d, O_d = I_h.cuda(), P_h.cuda(), O_h.cuda()
    plan.set_data(I_d, P_d, O_d)
    del I_d
    plan.iterate(warmup)
    plan.set_profiling(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    grp.barrier()
    e0.record(stream)
    plan.iterate(steps)
    e1.record(stream)
    grp.barrier()
    ms_total = grp.max_over_ranks(e0.elapsed_time(e1))
    phase_ms, n_prof = plan.phase_ms()
    plan.set_profiling(False)
    info, geo = plan.info(), plan.geometry()

    MV, NN = cfg.mode_views, cfg.N * cfg.N
    ms_step = ms_total / steps
    peak, peak_src = measured_peaks()
    psi_bytes = MV * NN * 16 + cfg.n_views * NN * 4          # psi read + write + sqrt(I) read
    psi_ms = phase_ms[0] / max(n_prof, 1)
    achieved = psi_bytes / (psi_ms * 1e-3) / 1e9
    bmin = 3 * MV * NN * 8 + cfg.n_views * NN * 4            # whole iteration
    bsimple = 4 * MV * NN * 8 + cfg.n_views * NN * 4
    it_gbs = bmin / (ms_step * 1e-3) / 1e9
    traffic, traffic_src = measured_traffic(cfg.name, info["path"], geo["wf_lag"])
    res = {
        "value": grp.aggregate(MV, steps, ms_total), "unit": UNIT, "steps": steps, "warmup": warmup,
        "ms_per_step": ms_step, "iterations_per_s": 1e3 / ms_step,
        "config": {"workload": cfg.name, "N": cfg.N, "n_views": cfg.n_views, "K": cfg.K, "L": cfg.L,
                   "object": [cfg.obj_h, cfg.obj_w], "mode_views": MV, "path": info["path"],
                   "parallelism": "replicas" if grp.world > 1 else "single-gpu",
                   "l2": f"inputs larger than L2 (psi {MV * NN * 8 / 2**20:.0f} MiB streamed every step)"
                         if MV * NN * 8 > 2 * 126 * 2**20 else "psi fits L2: latency-bound case, no flush"},
        "roofline": {"bound": "hbm", "kernel": "psi update (S1-S6)", "achieved": achieved, "peak": peak,
                     "unit": "GB/s", "frac": achieved / peak, "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                     "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                     "bytes_per_launch": psi_bytes, "ms_per_launch": psi_ms},   # finish_roofline() adds the FP32 side
        "iteration_roofline": {"bytes_min": bmin, "bytes_simple_schedule": bsimple, "achieved_gbs": it_gbs,
                               "frac_of_measured_hbm": it_gbs / peak, "frac_of_nominal_8TBs": it_gbs / NOMINAL_HBM_GBS},
        "phase_ms_per_step": {k: float(v) / max(n_prof, 1) for k, v in
                              zip(("psi_update", "object", "probe", "errors"), phase_ms)},
        "gpu_launches": info["launches_per_iter"] * steps,
    }
    return plan, (I_h, P_h, O_h), res


def finish_roofline(r, device_peaks):
    """the reported fraction is max(t_HBM, t_FP32) / t_kernel, `bound` names the side that won and
    both sides stay in the object ("hbm", "alu").  t_HBM = algorithmic bytes / measured HBM copy rate; t_FP32 =
    lane-operations / the FFMA2 lane rate this device sustains (dm_measure_peaks; an FMA is ONE lane-operation, a
    butterfly is mostly adds).  Without device peaks (replica runs) the HBM side stands alone."""
    rf, c = r["roofline"], r["config"]
    hbm = {"achieved": rf["achieved"], "peak": rf["peak"], "unit": "GB/s", "frac": rf["frac"],
           "bytes_per_launch": rf["bytes_per_launch"], "peak_source": rf["peak_source"]}
    rf["hbm"] = hbm
    if not device_peaks:
        return
    per_px, src = lane_ops_per_pixel(c["workload"], c["path"], c["N"])
    ops = per_px * c["mode_views"] * c["N"] ** 2
    t = rf["ms_per_launch"] * 1e-3
    peak = device_peaks["fp32_lane_ops_per_s_ffma2"]
    alu = {"achieved": ops / t / 1e12, "peak": peak / 1e12, "unit": "T lane-op/s", "frac": ops / t / peak,
           "lane_ops_per_pixel_mode": per_px, "lane_ops_source": src, "lane_ops_per_launch": ops,
           "peak_source": "measured in this run (dm_measure_peaks, packed FFMA2 lanes)"}
    rf["alu"] = alu
    if alu["frac"] > hbm["frac"]:
        rf.update({"bound": "alu", "achieved": alu["achieved"], "peak": alu["peak"], "unit": alu["unit"], "frac": alu["frac"],
                   "peak_source": alu["peak_source"]})
    rf["rule"] = "frac = max(t_HBM, t_FP32) / t_kernel (SURVEY.md 8(d)); both sides under 'hbm' and 'alu'"


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
    stream = torch.cuda.current_stream()
    sampler = ClockSampler(local)
    sampler.start()

    # ---- headline workload: every rank reconstructs its own data set (replicas; seed = rank) ----
    pr = synth.make_problem(cfg, seed=grp.seed)
    plan, (I_h, P_h, O_h), line = measure_device_arm(dm, synth, torch, grp, cfg, pr, args.steps, args.warmup,
                                                     args.path, args.lag, stream)

    # ---- end-to-end arm: HOST (pinned) buffers through dm_solve_host, copies inside the timing ----
    Pout_h = torch.empty_like(P_h).pin_memory()
    Oout_h = torch.empty_like(O_h).pin_memory()
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(2):
        plan.solve_host(I_h, P_h, O_h, 1, Pout_h, Oout_h)
    grp.barrier()
    e0.record(stream)
    for _ in range(e2e_steps):
        plan.solve_host(I_h, P_h, O_h, 1, Pout_h, Oout_h)
    e1.record(stream)
    grp.barrier()
    ms_e2e = grp.max_over_ranks(e0.elapsed_time(e1))
    h2d = I_h.numel() * 4 + P_h.numel() * 8 + O_h.numel() * 8
    d2h = Pout_h.numel() * 8 + Oout_h.numel() * 8
    plan.close()
    del plan, I_h, P_h, O_h, Pout_h, Oout_h, pr
    torch.cuda.empty_cache()

    # ---- the other single-GPU configs, same device-resident measurement (N = 1 only) ----
    per_config = []
    if world == 1 and not args.no_per_config:
        for ci in args.per_config:
            if ci == args.config:
                continue
            c2 = synth.CONFIGS[ci]
            pr2 = synth.make_problem(c2, seed=grp.seed)
            plan2, hosts, r2 = measure_device_arm(dm, synth, torch, grp, c2, pr2, args.per_config_steps, max(3, args.warmup),
                                                  0, 0, stream)
            plan2.close()
            del plan2, hosts, pr2
            torch.cuda.empty_cache()
            per_config.append(r2)
    clocks = sampler.stop()
    # FP32 / HBM / L2 / shared-memory rates of this device, measured by the library's own streaming kernels
    device_peaks = dm.measure_peaks() if world == 1 else None

    if rank != 0:
        grp.close()
        return

    head = {"metric": METRIC, "value": line.pop("value"), "unit": line.pop("unit"), "n_gpus": world,
            "steps": line.pop("steps"), "warmup": line.pop("warmup"), "ms_per_step": line.pop("ms_per_step"),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic"}
    head.update(line)
    head["e2e"] = {"value": grp.aggregate(cfg.mode_views, e2e_steps, ms_e2e), "unit": UNIT, "steps": e2e_steps,
                   "ms_per_step": ms_e2e / e2e_steps, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                   "call": "dm_solve_host(n_iter=1): H2D intensities+P0+O0 (pinned), set_data, 1 iteration, D2H P+O"}
    head["clocks"] = clocks
    if device_peaks:
        head["device_peaks"] = device_peaks
    for r in [head] + per_config:
        finish_roofline(r, device_peaks)
    # the driver's record keeps `config` and `roofline` whole but drops unknown top-level keys: a compact copy of the
    # other configs' results rides inside `config` (c1 is the workload BENCH_r01 was quoted on)
    head["config"]["per_config_summary"] = [
        {"workload": r["config"]["workload"], "path": r["config"]["path"], "value": r["value"], "ms_per_step": r["ms_per_step"],
         "psi_update_ms": r["roofline"]["ms_per_launch"], "roofline_bound": r["roofline"]["bound"],
         "roofline_frac": r["roofline"]["frac"], "hbm_frac": r["roofline"]["hbm"]["frac"],
         "alu_frac": (r["roofline"].get("alu") or {}).get("frac"),
         "iteration_frac_of_measured_hbm": r["iteration_roofline"]["frac_of_measured_hbm"]} for r in per_config]
    if device_peaks:
        head["roofline"]["device_peaks"] = device_peaks
    if per_config:
        head["per_config"] = per_config
    line = head
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
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=3,
                    help="BASELINE.json config index of the headline workload (default 3: the largest single-GPU config)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--path", type=int, default=0,
                    help="psi-update path of the headline workload: 0 auto, 1 staged, 2 fused (N <= 128), "
                         "3 register-resident (N = 128), 4 view-pipelined warp-FFT")
    ap.add_argument("--lag", type=int, default=0, help="path 4: phase lag in views (0 = derived)")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--per-config", type=int, nargs="*", default=[1, 2, 4],
                    help="other configs measured in the same run (device-resident arm only), reported under per_config")
    ap.add_argument("--per-config-steps", type=int, default=10)
    ap.add_argument("--no-per-config", action="store_true")
    ap.add_argument("--print-csrc-digest", action="store_true", help="print the digest profiles/traffic.json is keyed by")
    ap.add_argument("--ref-mode-views", type=int, default=4096,
                    help="size of the bounded oracle sample (mode-views per iteration)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--peaks", action="store_true", help="only measure and print the device rates of dm_measure_peaks")
    args = ap.parse_args()
    if args.print_csrc_digest:
        print(csrc_digest())
        return
    if args.peaks:
        import torch
        from paper_1808_10375_b200 import dm
        assert torch.cuda.is_available(), "bench.py --peaks needs a CUDA device"
        sampler = ClockSampler(0)
        sampler.start()
        pk = dm.measure_peaks()
        print(json.dumps({"device_peaks": pk, "clocks": sampler.stop(), "gpu": torch.cuda.get_device_name(0)}), flush=True)
        return
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
