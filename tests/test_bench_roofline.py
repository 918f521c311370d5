"""bench.py's roofline object follows SURVEY.md 8(d): frac = max(t_HBM, t_FP32) / t_kernel, `bound` names the
side that won, both sides stay in the object.  Host arithmetic only (no GPU)."""
import bench


def _result(N=128, mode_views=5000, ms=0.6, hbm_peak=6500.0):
    bytes_ = mode_views * N * N * 16 + (mode_views // 2) * N * N * 4
    ach = bytes_ / (ms * 1e-3) / 1e9
    return {"config": {"workload": "c1-flyscan2", "path": 3, "N": N, "mode_views": mode_views},
            "roofline": {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak,
                         "bytes_per_launch": bytes_, "ms_per_launch": ms, "peak_source": "test"}}


def test_roofline_takes_the_larger_bound_and_keeps_both():
    r = _result()
    per_px, src = bench.lane_ops_per_pixel("c1-flyscan2", 3, 128)
    assert per_px > 0 and (src.startswith("measured") or src.startswith("estimated"))
    ops = per_px * 5000 * 128 * 128
    # an FP32 peak so low that the ALU side must win, then one so high that HBM must win
    for peak, want in ((ops / 0.5e-3, "alu"), (ops / 0.01e-3, "hbm")):
        rr = _result()
        bench.finish_roofline(rr, {"fp32_lane_ops_per_s_ffma2": peak})
        rf = rr["roofline"]
        assert rf["bound"] == want
        assert abs(rf["frac"] - max(rf["hbm"]["frac"], rf["alu"]["frac"])) < 1e-12
        t = rf["ms_per_launch"] * 1e-3
        assert abs(rf["hbm"]["frac"] - (rf["bytes_per_launch"] / (rf["hbm"]["peak"] * 1e9)) / t) < 1e-12
        assert abs(rf["alu"]["frac"] - (ops / peak) / t) < 1e-12
        assert rf["achieved"] / rf["peak"] == rf["frac"] or abs(rf["achieved"] / rf["peak"] - rf["frac"]) < 1e-12
    # replica runs have no device peaks: the HBM side stands alone
    bench.finish_roofline(r, None)
    assert r["roofline"]["bound"] == "hbm" and "alu" not in r["roofline"]


def test_unmatched_capture_is_labelled_estimated():
    per_px, src = bench.lane_ops_per_pixel("no-such-workload", 4, 256)
    assert per_px == bench.LANE_OPS_ESTIMATE[256] and src.startswith("estimated")
