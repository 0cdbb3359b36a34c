"""Host-side logic of bench.py that needs no GPU: the algorithmic work counts behind `roofline`, the source hash that
ties the ncu figures in profiles/ to the kernels, and the stale-capture rule."""
import json
import os

import bench

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_algorithmic_counts_follow_design_section_7():
    n, m, k = 1_048_576, 52.16, 42
    a = bench.algorithmic(0, n, m * n, k)
    assert a["force_slots"] == n * (6 * m + 48 * k) and a["dens_slots"] == n * (6 * m + 25 * k)
    assert a["force_bytes"] == n * (4 * m + 4 + 32 + 24 + 24 + 24)
    s = bench.algorithmic(0, n, m * n, k, bench.SURVEY_SLOTS)
    assert s["force_slots"] == n * (13 * m + 95 * k)                 # SURVEY.md section 8(d)'s estimate
    t = bench.algorithmic(1, n, 58.0 * n, 58)
    assert t["force_slots"] == n * 58 * (8 + 18)


def test_source_hash_and_stale_rule(tmp_path, monkeypatch):
    h = bench.csrc_sha()
    assert len(h) == 16 and h == bench.csrc_sha()
    from paper_1212_6332_b200 import ncu_summary
    assert ncu_summary.csrc_sha() == h                                # the writer and the reader of profiles/ncu_*.json agree
    # a capture of other sources reads as stale, never as current
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    os.makedirs(tmp_path / "profiles")
    os.makedirs(tmp_path / "paper_1212_6332_b200" / "csrc")
    (tmp_path / "paper_1212_6332_b200" / "csrc" / "a.cu").write_text("x")
    (tmp_path / "profiles" / "ncu_3a.json").write_text(json.dumps({"csrc_sha": "0" * 16, "source": "s", "kernels": {}}))
    cap = bench.ncu_capture("3a")
    assert cap["stale"] is True and "kernels" not in cap
    (tmp_path / "profiles" / "ncu_3a.json").write_text(json.dumps({"csrc_sha": bench.csrc_sha(), "source": "s", "kernels": {"force": {}}}))
    assert bench.ncu_capture("3a")["kernels"] == {"force": {}}
    assert bench.ncu_capture("nope") is None


def test_committed_captures_name_their_command():
    for w in ("3a", "4", "1"):
        p = os.path.join(ROOT, "profiles", f"ncu_{w}.json")
        if os.path.exists(p):
            cap = json.load(open(p))
            assert cap["command"].startswith("ncu ") and "bench.py" in cap["command"]
            assert os.path.exists(os.path.join(ROOT, cap["source"]))
            assert {"force", "density"} <= set(cap["kernels"])
