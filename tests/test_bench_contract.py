"""bench.py host logic (no GPU): the flop convention against SURVEY.md section 8 size table, and the reference arm's JSON line."""
import io
import json
import contextlib

import bench


def test_flop_convention_matches_survey_table():
    # ladder cMAC vv^2*oo, ring cMAC (ov)^3, "all sigma terms, flop" per config
    for (o, v, ladder, ring, total) in [(4, 20, 2.17e5, 5.12e5, 9.25e6), (10, 80, 4.49e8, 5.12e8, 9.08e9),
                                        (24, 200, 1.09e11, 1.11e11, 1.89e12), (34, 300, 1.13e12, 1.06e12, 1.85e13)]:
        cm = bench.sigma_cmacs(o, v)
        assert abs(cm["T11"] - ladder) / ladder < 0.01
        assert abs(cm["T8"] - ring) / ring < 0.01
        assert abs(bench.sigma_flops(o, v) - total) / total < 0.01


def test_reference_arm_prints_one_json_line_with_the_contract_keys(monkeypatch):
    monkeypatch.setattr(bench, "ORACLE_SAMPLE", (3, 5))
    args = type("A", (), dict(config=4, steps=2, warmup=1, gpus=1))()
    buf = io.StringIO()
    with contextlib.redirect_stdout(buf):
        bench.run_reference(args)
    lines = [l for l in buf.getvalue().splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in d, key
    assert d["impl"] == "reference" and d["vs_baseline"] is None and d["value"] > 0
    assert d["steps"] == 2 and d["warmup"] == 1                    # the arm honours --steps / --warmup as given
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and "workload" in d["config"]
