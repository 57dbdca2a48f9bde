"""-m "not gpu": bench.py's flat summary (host logic).  The driver's record keeps the scalar keys
of `roofline` and drops nested objects, so both halves of BASELINE.json's metric -- "% of FP64 /
HBM roofline" -- and every leg's fraction must be there as flat scalars copied from the legs."""
import types

import bench


def test_flat_summary_copies_every_leg_into_scalars():
    roofline = {
        "frac": 0.915,
        "per_turn": {"frac": 1.07, "achieved": 7000.0, "ms_per_turn": 0.0458, "frac_of_nominal_8TBs": 0.875,
                     "value": 2.2e11, "traffic": 261_000_000, "peak": 6545.6,
                     "beyond_l2": {"rows": [{"frac": 1.04}, {"frac": 0.98}, {"frac": 0.94}]}},
        "configs": {"configs[2]": {"roofline": {"frac": 0.936}},
                    "configs[4] leapfrog fp32": {"roofline": {"frac": 0.883}},
                    "configs[4] ruth4 fp64": {"roofline": {"frac": 0.922}}},
        "next": {"f2_ramp_fused": {"roofline": {"frac": 0.842}},
                 "f4_slice_histogram": {"us_per_call": 16.8, "roofline": {"frac": 0.73}}},
        "f1_chunk_sweep": {"rows": [{"turns_per_launch": 1, "kernel": "fused", "us_per_launch": 8.2},
                                    {"turns_per_launch": 4, "kernel": "fused", "us_per_launch": 9.0},
                                    {"turns_per_launch": 1, "kernel": "per_turn graph=1", "us_per_launch": 3.9}]},
    }
    cx = types.SimpleNamespace(traffic={"fused_source": "profiles/ncu_traffic.json, captured at abc1234"})
    flat = bench.flat_summary(roofline, cx)
    assert all(not isinstance(v, (dict, list)) for v in flat.values())
    assert flat["per_turn_frac"] == 1.07 and flat["per_turn_gbs"] == 7000.0 and flat["per_turn_us"] == 45.8
    assert abs(flat["per_turn_dram_frac"] - 261e6 / 45.8e-6 / 1e9 / 6545.6) < 1e-3
    assert (flat["per_turn_beyond_l2_frac_min"], flat["per_turn_beyond_l2_frac_max"]) == (0.94, 1.04)
    assert flat["cfg2_frac"] == 0.936 and flat["cfg4_lf_f32_frac"] == 0.883 and flat["cfg4_ruth4_f64_frac"] == 0.922
    assert flat["f2_ramp_frac"] == 0.842 and flat["f4_hist_frac"] == 0.73 and flat["f4_hist_us"] == 16.8
    assert flat["f1_us_per_launch_1turn_fused"] == 8.2
    assert flat["f1_us_per_launch_1turn_per_turn_graph"] == 3.9
    assert flat["traffic_source"].endswith("abc1234")
    assert "cfg4_ec_f64_frac" not in flat and "f3_fused_frac" not in flat      # legs that did not run


def test_flat_summary_survives_failed_legs():
    cx = types.SimpleNamespace(traffic={})
    flat = bench.flat_summary({"per_turn": {"error": "RuntimeError: boom"}, "configs": {"error": "x"}}, cx)
    assert flat == {"traffic_source": None}


def test_ncu_traffic_file_names_the_commit_of_every_capture():
    t = bench.ncu_traffic()
    assert t["fused"] > 0 and "captured at" in t["fused_source"] and "captured at" in t["per_turn_source"]
