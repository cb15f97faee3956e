"""Host-side arithmetic of bench.py that the reported roofline rests on (no GPU): algorithmic bytes per
site as SURVEY.md 8(d) counts them, and the rule that `roofline.traffic` is read from a committed capture
summary (or is null with the reason), never a literal in bench.py."""
import json
import os

import numpy as np

import bench
from paper_1311_2404_b200 import workloads as W


def test_algorithmic_bytes_per_site():
    w = W.c1_taylor_green(32)
    assert bench.algorithmic_bytes_per_site(w) == 2 * 9 * 4 + 1                      # 73
    w = W.c2_channel(16, 256, 4)                                                     # SOLID rows y = 0, 255
    assert abs(bench.algorithmic_bytes_per_site(w) - ((1 - 2 / 256) * 152 + 1)) < 1e-12
    for prec, s in ((W.F32, 4), (W.F64, 8)):
        w = W.c3_mrt_obstacles(64, 48, 40, precision=prec)
        phi = float((w.mask == W.SOLID).mean())
        assert 0.04 < phi < 0.06
        assert abs(bench.algorithmic_bytes_per_site(w) - ((1 - phi) * 2 * 19 * s + 1)) < 1e-12
        assert abs(bench.algorithmic_bytes_per_site(w) - (145.4 if s == 4 else 289.8)) < 2.0 * s / 4
    assert bench.algorithmic_bytes_per_site(W.c5_shan_chen(8, 8, 8)) == 472           # two-pass floor, fp32
    assert bench.algorithmic_bytes_per_site(W.c4_duct(8, 8, 8, precision=W.F64)) < 2 * 19 * 8 + 1


def test_traffic_comes_from_the_committed_capture_or_is_null(tmp_path, monkeypatch):
    missing = tmp_path / "none.json"
    monkeypatch.setattr(bench, "TRAFFIC_FILE", str(missing))
    t, src = bench.ncu_traffic("c2")
    assert t is None and "no committed capture" in src
    f = tmp_path / "t.json"
    f.write_text(json.dumps({"commit": "abc1234", "configs": {"c2": {"dram_bytes_per_step": 2.5e9, "kernel": "step_kernel<...>"}}}))
    monkeypatch.setattr(bench, "TRAFFIC_FILE", str(f))
    t, src = bench.ncu_traffic("c2")
    assert t == 2.5e9 and "abc1234" in src
    assert bench.ncu_traffic("c9")[0] is None
    # the shipped file, if present, must name its commit and hold per-step byte counts
    shipped = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "profiles", "r02_traffic.json")
    if os.path.exists(shipped):
        d = json.load(open(shipped))
        assert len(d["commit"]) >= 7 and "command" in d
        for k, v in d["configs"].items():
            assert v["dram_bytes_per_step"] > 1e6 and v["kernel"]
