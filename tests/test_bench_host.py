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
    e = {"hbm_frac": 0.5}
    # 2 warp-instructions per cell, 0.5 of them packed: 2.5 slots; 148 SMs x 4 x 1 GHz = 592 G slots/s
    bench.issue_fields(e, ["2.0", "32.0", "0.5", "k"], N=592_000_000, ms=2.5, sms=148, mhz=1000)
    assert abs(e["issue_slots_per_cell"] - 2.5) < 1e-12 and abs(e["issue_frac"] - 1.0) < 1e-9
    assert e["bound"] == "issue"
    e = {"hbm_frac": 0.9}
    bench.issue_fields(e, ["2.0", "32.0", "0.5", "k"], N=592_000_000, ms=5.0, sms=148, mhz=1000)
    assert abs(e["issue_frac"] - 0.5) < 1e-9 and e["bound"] == "hbm"
    e = {"hbm_frac": 0.9}
    bench.issue_fields(e, None, 1, 1.0, 148, 1000)          # no row, or no clock sample: nothing claimed
    bench.issue_fields(e, ["2.0", "32.0", "0.5", "k"], 1, 1.0, 148, None)
    assert "issue_frac" not in e


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
