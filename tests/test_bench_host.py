"""Host-side logic of bench.py that needs no GPU: the ncu counters it reports come from the committed profile summaries,
the workload table covers BASELINE.json's configs, and every profile names the command that made it."""
from __future__ import annotations

import csv
import glob
import json
import os

import bench

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_ncu_counters_come_from_profiles():
    path = os.path.join(ROOT, "profiles", "r02_ncu_per_launch.csv")
    rows = list(csv.DictReader(open(path)))
    assert {"workload", "variant", "kernel", "dram_bytes", "warp_inst", "source"} <= set(rows[0])
    for r in rows:
        assert os.path.exists(os.path.join(ROOT, r["source"])), r["source"]
        assert float(r["dram_bytes"]) > 0 and float(r["warp_inst"]) > 0
    # the default line and its companions find their rows
    for wl in ("c5", "s512", "c5u"):
        assert bench.ncu_value(wl, "global", "dram_bytes") > 1e9
        assert bench.ncu_value(wl, "global", "warp_inst") > 1e8
    assert bench.ncu_value("c5", "no-such-variant", "dram_bytes") is None
    # algorithmic bytes of a coherent field = measured DRAM traffic (no wasted re-reads): 28 B x 2^27 cells for configs[4]
    spec = bench.workload_spec("c5")
    assert abs(bench.ncu_value("c5", "global", "dram_bytes") / (bench.bytes_per_cell(spec) * 2 ** 27) - 1.0) < 0.02


def test_workloads_cover_the_baseline_configs():
    cfg = json.load(open(os.path.join(ROOT, "BASELINE.json")))["configs"]
    assert len(cfg) == 5
    for name in ("c2", "c3", "c4-32", "c4-256", "c5", "c5u", "s512", "s512d", "s512f"):
        spec = bench.workload_spec(name)
        assert spec["nsub"] >= 1 and len(spec["n"]) in (3, 4) and bench.bytes_per_cell(spec) in (24, 28, 32)
    assert bench.workload_spec("c5")["n"] == [48] * 4 and bench.workload_spec("c5")["nsub"] == 4


def test_every_profile_names_its_command():
    for f in glob.glob(os.path.join(ROOT, "profiles", "*_full.txt")):
        first = open(f).readline()
        assert first.startswith("command: ncu "), f
    for f in glob.glob(os.path.join(ROOT, "profiles", "*.csv")):
        assert os.path.exists(f[:-4] + ".md"), f"{f} needs a .md beside it naming its command"
