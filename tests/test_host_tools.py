"""Host-side helpers of bench.py and of the profile summaries (no GPU): the parity block of the bench line, the
summary of a committed ncu launch list, and the rule that a stored DRAM counter is reported only for the kernel
sources it was captured from."""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
from paper_1810_02916_b200 import profiling  # noqa: E402


def test_parity_block_metric_and_fractional_error():
    rng = np.random.default_rng(0)
    ref = rng.standard_normal((1000, 3))
    ref[0] = 1e-9                                     # a tiny acceleration: the metric divides by the rms there, frac_err does not
    got = ref * (1 + 1e-6)
    got[1] = ref[1] * 1.5
    p = bench.parity_block(got.astype(np.float64), ref)
    rms = np.sqrt((ref ** 2).sum(axis=1).mean())
    e1 = 0.5 * np.linalg.norm(ref[1]) / max(np.linalg.norm(ref[1]), rms)
    assert p["n_sinks"] == 1000 and abs(p["max"] - e1) < 1e-12 and not p["pass"]
    assert abs(p["frac_err_median"] - 1e-6) < 1e-9 and abs(p["frac_gt_1e-4"] - 1e-3) < 1e-12
    assert bench.parity_block(ref * (1 + 1e-7), ref)["pass"]


def test_launch_list_summary_of_the_committed_csv(tmp_path):
    out = tmp_path / "l.md"

    class A:
        csv = os.path.join(ROOT, "profiles", "r02_launches_c4.csv")
        title, command, note = "t", "c", ""
    A.out = str(out)
    profiling.cmd_launches(A)
    text = out.read_text()
    rows = [l for l in text.splitlines() if l.startswith("| `k_")]
    assert any("k_forces_warp" in r for r in rows) and any("k_radix_scatter" in r for r in rows)
    share = float([r for r in rows if "k_forces_warp" in r][0].split("|")[5].strip().rstrip("%"))
    assert share > 90.0                               # the interaction kernel dominates the step


def test_traffic_is_reported_only_for_the_sources_it_was_captured_from(tmp_path, monkeypatch):
    rec = {"W": {"dram_bytes_read": 3.0, "dram_bytes_write": 4.0, "kernel_source_sha256": profiling.kernel_source_hash()}}
    f = tmp_path / "t.json"
    f.write_text(json.dumps(rec))
    monkeypatch.setattr(profiling, "TRAFFIC_JSON", str(f))
    assert profiling.read_traffic("W") == 7.0 and profiling.read_traffic("other") is None
    rec["W"]["kernel_source_sha256"] = "0" * 64
    f.write_text(json.dumps(rec))
    assert profiling.read_traffic("W") is None
