"""Host-side logic of bench.py (no GPU): the committed ncu tables it reads, the issue-slot roofline
arithmetic, the staleness check of those tables, and the reference arm's JSON line."""
import json
import os
import subprocess
import sys

import bench

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SOLVE = ["analytic-fast", "sz-fast", "newton-fast", "nested-fast", "analytic", "sz", "newton", "nested"]


def test_instruction_table_has_a_row_per_variant():
    t = bench.profile_table("instruction_counts.txt")
    for name in SOLVE + ["plic_volume", "blank", "roundtrip:analytic-fast"]:
        row = t[name]
        inst, lanes, packed = float(row[0]), float(row[1]), float(row[2])
        assert 0.1 < inst < 20 and 1 <= lanes <= 32 and 0 <= packed < inst, (name, row)
    # the packed fp32x2 kernels are the PLIC_FAST ones; the precise kernels are scalar code
    assert all(float(t[n][2]) > 0 for n in SOLVE[:4]) and all(float(t[n][2]) == 0 for n in SOLVE[4:])
    assert int(t["@cells"][0]) == 1 << 26 and len(t["@csrc_sha1"][0]) == 12


def test_traffic_table_matches_the_algorithmic_bytes():
    t = bench.profile_table("dram_traffic.txt")
    cells = int(t["@cells"][0])
    for name in SOLVE + ["plic_volume"]:
        assert 0.95 <= float(t[name][0]) / (bench.BYTES_PER_CELL * cells) <= 1.02, name   # no wasted re-reads
    traffic, src = bench.ncu_traffic("analytic-fast", cells)
    assert traffic == float(t["analytic-fast"][0]) and "dram_traffic.txt" in src
    none, why = bench.ncu_traffic("analytic-fast", cells // 2)
    assert none is None and "cells" in why


def test_issue_fields_count_a_packed_instruction_twice():
    clk = {"sm_mhz": 1100, "sm_mean_mhz": 1000.0}              # the mean of the window is the denominator
    e = {"hbm_frac": 0.5}
    # 2 warp-instructions per cell, 0.5 of them packed: 2.5 slots; 148 SMs x 4 x 1 GHz = 592 G slots/s
    bench.issue_fields(e, ["2.0", "32.0", "0.5", "k"], N=592_000_000, ms=2.5, sms=148, clk=clk)
    assert abs(e["issue_slots_per_cell"] - 2.5) < 1e-12 and abs(e["issue_frac"] - 1.0) < 1e-9
    assert e["bound"] == "issue" and e["issue_clock_mhz"] == 1000.0
    e = {"hbm_frac": 0.9}
    bench.issue_fields(e, ["2.0", "32.0", "0.5", "k"], N=592_000_000, ms=5.0, sms=148, clk=1000)
    assert abs(e["issue_frac"] - 0.5) < 1e-9 and e["bound"] == "hbm"
    e = {"hbm_frac": 0.9}
    bench.issue_fields(e, None, 1, 1.0, 148, clk)               # no row, or no clock sample: nothing claimed
    assert e["issue_frac"] is None and "bound" not in e
    bench.issue_fields(e, ["2.0", "32.0", "0.5", "k"], 1, 1.0, 148, {"sm_mhz": None})
    assert e["issue_frac"] is None and "bound" not in e


def test_issue_fraction_above_one_is_a_model_error_not_a_bound():
    e = {"hbm_frac": 0.5}
    bench.issue_fields(e, ["2.0", "32.0", "0.5", "k"], N=592_000_000, ms=2.0, sms=148, clk=1000)
    assert e["issue_frac"] > 1.0 and e["issue_model_error"] is True and e["bound"] is None


def test_instruction_counts_are_used_only_on_the_workload_they_were_captured_on():
    t = bench.profile_table("instruction_counts.txt")
    assert t["@workload"] == ["configs[1]"]
    for name in SOLVE:
        assert bench.counts_row(t, name, "configs[1]") == t[name]
    for other in ("configs[2]", "configs[3]"):
        for name in ("analytic", "sz", "newton", "nested"):      # map_compact: executed counts depend on the data
            assert t[name][3].startswith("map_compact") and bench.counts_row(t, name, other) is None
        for name in ("analytic-fast", "sz-fast", "newton-fast", "nested-fast"):     # branch-free
            assert bench.counts_row(t, name, other) == t[name]
    assert bench.counts_row(t, "no-such-kernel", "configs[1]") is None


def test_table_staleness_follows_the_kernel_sources():
    d = bench.csrc_digest()
    assert len(d) == 12 and int(d, 16) >= 0
    assert not bench.table_is_stale({"@csrc_sha1": [d]})
    assert bench.table_is_stale({"@csrc_sha1": ["0" * 12]}) and bench.table_is_stale({})


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--log2n", "20"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == bench.METRIC and line["unit"] == bench.UNIT
    assert line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle" and line["gpu_launches"] == 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"]


def _synthetic_full_line():
    """An object of the shape and size run_ours builds (33 KB in round 2: too long for a driver that
    keeps a bounded tail of stdout)."""
    variant = {"value": 331.0123456789, "ms_per_step": 0.20271234567, "launches": 100, "bytes_per_cell": 20,
               "hbm_gbs_per_gpu": 6620.123456789, "hbm_frac": 1.0137812345, "hbm_frac_nominal": 0.8275123,
               "sm_mhz": 1507, "roofline_frac": 1.0137812345, "per_launch": {"n": 20, "median_ms": 0.2031234,
                                                                              "best_ms": 0.20112345},
               "warp_inst_per_cell": 2.059, "lanes_per_inst": 31.9, "packed_warp_inst_per_cell": 0.672,
               "issue_slots_per_cell": 2.731, "issue_frac": 0.93712345, "bound": "hbm",
               "algorithmic_thread_inst_per_cell": 61, "issue_frac_algorithmic": 0.7123456}
    methods = {k: dict(variant) for k in SOLVE + ["plic_volume", "blank"]}
    big = {k: {m: dict(variant) for m in SOLVE} for k in ("a", "b")}
    return {
        "metric": bench.METRIC, "value": 331.0123456789, "unit": bench.UNIT, "n_gpus": 1, "steps": 100, "warmup": 5,
        "ms_per_step": 0.20271234567, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": bench.WORKLOAD % 26, "cells_per_gpu": 1 << 26, "method": "analytic-fast",
                   "l2": "inputs larger than L2", "launch": {"grid": 32768, "block": 256, "cells_per_thread": 4}},
        "clocks": {"sm_mhz": 1507, "sm_min_mhz": 1500, "sm_max_mhz": 1965, "reasons": ["sw_power_cap"],
                   "samples": 10, "note": "x" * 300},
        "gpu_launches": 100, "gpu_launches_all_timed_regions": 4000,
        "e2e": {"value": 3.19, "unit": bench.UNIT, "h2d_bytes_per_step": 16 << 26, "d2h_bytes_per_step": 4 << 26,
                "steps": 10, "frac_of_link": 0.93, "pcie": {"gen": 5, "width": 16}, "bound": "y" * 200},
        "roofline": {"bound": "hbm", "achieved": 6620.1, "peak": 6530.0, "unit": "GB/s", "frac": 1.0138,
                     "traffic": 1324311112.0, "kernel": "analytic-fast", "peak_note": "z" * 250},
        "stream_ceiling": dict(variant), "methods": methods, "burst": dict(variant),
        "storage": {k + "/f16": dict(variant) for k in SOLVE}, "pipe_rates": big, "paper_benchmark": big,
        "curvature": dict(variant), "divergence": {"methods": big}, "config4": {"methods": big},
        "cpu_baseline": {"value": 0.0257, "unit": bench.UNIT, "cores": 16, "kind": "oracle", "sample": "s" * 120},
        "cpu_baseline_1core": {"value": 0.0016, "unit": bench.UNIT, "cores": 1, "kind": "oracle", "sample": "s" * 120},
        "summary": {"cols": "c" * 100, "rows": {k: [0.2018, 1.018, 0.937, "hbm", 0.188, 1.0, 0.7408, 1.11] for k in SOLVE},
                    "storage_ms": {k + "/f16": 0.1569 for k in SOLVE}},
    }


CONTRACT_KEYS = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                 "scaling", "vs_baseline", "dtype", "data", "config", "clocks", "gpu_launches", "e2e", "roofline",
                 "cpu_baseline")


def test_stdout_line_is_short_enough_for_a_driver_that_keeps_a_tail(tmp_path):
    full = _synthetic_full_line()
    assert len(json.dumps(full)) > 30000                       # the size that broke the round-2 record
    path = bench.write_detail(full, str(tmp_path / "sub" / "detail.json"))
    assert json.load(open(path)) == json.loads(json.dumps(full))
    line = bench.compact_line(full, path)
    text = json.dumps(line)
    assert len(text) < bench.LINE_LIMIT <= 8192
    back = json.loads(text)
    for k in CONTRACT_KEYS:
        assert k in back, k
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in back["roofline"], k
    for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"):
        assert k in back["e2e"], k
    assert back["cpu_baseline"]["kind"] == "oracle" and back["clocks"]["reasons"] == ["sw_power_cap"]
    assert not any(k in back for k in bench.DETAIL_KEYS)
    assert back["detail"]["file"] == path and set(back["detail"]["keys"]) == set(bench.DETAIL_KEYS)
    assert back["value"] == 331.012 and "summary" in back      # 6 significant digits
    # a pathologically long optional part is dropped rather than breaking the bound; the contract keys stay
    full["summary"]["rows"] = {str(i): ["w" * 50] * 8 for i in range(40)}
    full["burst"]["note"] = "n" * 5000
    worst = bench.compact_line(full, None)
    assert len(json.dumps(worst)) < bench.LINE_LIMIT
    assert all(k in worst for k in CONTRACT_KEYS)
    assert bench.write_detail(full, "") is None


def test_run_ours_prints_exactly_one_line():
    """No second print of a JSON object in the GPU arm: the compact line is the only stdout line."""
    src = open(os.path.join(ROOT, "bench.py")).read()
    body = src[src.index("def run_ours("):src.index("# ---- what goes to stdout")]
    assert body.count("print(") == 1 and "print(json.dumps(compact_line(line, detail_path))" in body
