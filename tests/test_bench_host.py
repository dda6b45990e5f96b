"""Host-side logic of bench.py that needs no GPU: the byte accounting behind `roofline` and `whole_eval`, the rule that
decides whether L2 is flushed between steps (printed in `config`, identical in both arms), the reference arm's line."""
import json
import subprocess
import sys
import os

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
from paper_1910_07054_b200 import workloads as W  # noqa: E402


def test_algorithmic_bytes_of_the_storages_at_config_4():
    w = W.config(4)
    nk = 2 * 256 * 257
    spec = 192 * nk * 8
    plain = bench.algorithmic_bytes(w)
    assert plain["bank"] == 6 * 64 * 64 * nk * 4 and plain["coupling"] == plain["bank"] + 2 * spec
    mir = bench.algorithmic_bytes(w, None, True)
    assert mir["bank"] == 6 * 64 * 64 * 257 * 257 * 4
    rec = bench.algorithmic_bytes(w, None, True, True)
    # SURVEY.md:196-197: unordered layer pairs, ky-mirrored: 3.30 GB of bank, 3.70 GB for the coupling launch
    assert rec["bank"] == 6 * 2080 * 257 * 257 * 4
    assert abs(rec["coupling"] / 1e9 - 3.70) < 0.01
    assert rec["whole"] == rec["bank"] + 4 * spec + 4 * 192 * 256 * 257 * 8 + 2 * 192 * 256 * 256 * 4


def test_fused_path_moves_no_spectra():
    w = W.config(2)
    staged, fused = bench.algorithmic_bytes(w), bench.algorithmic_bytes(w, fused=True)
    spec = 18 * 2 * 64 * 65 * 8
    assert staged["whole"] - fused["whole"] == 4 * spec and fused["bank"] == staged["bank"]


def test_l2_rule_depends_on_the_workload_only():
    assert bench.l2_mode(W.config(1)).startswith("L2 flushed")
    assert bench.l2_mode(W.config(2)).startswith("L2 flushed")
    for k in (3, 4, 5):
        assert bench.l2_mode(W.config(k)).startswith("inputs larger than L2")
    assert bench.workload_config(W.config(4))["l2"] == bench.l2_mode(W.config(4))


def test_reference_arm_prints_the_contract_line_on_config_1():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "3", "--warmup", "1"], capture_output=True, text=True, check=True).stdout
    line = json.loads([l for l in out.splitlines() if l.startswith("{")][-1])
    assert line["impl"] == "reference" and line["metric"] == bench.METRIC and line["higher_is_better"] is True
    assert line["config"] == bench.workload_config(W.config(1))
    cb = line["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores_timed"] == 1 and cb["value"] == line["value"] and "all_cores" in cb
    assert line["e2e"] == {"value": line["value"], "unit": bench.UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["gpu_launches"] == 0
    # one meaning per key: the steps that ran, a whole evaluation per step, value = 1000 / ms_per_step, nothing extrapolated
    assert line["steps"] == 3 and line["steps_requested"] == 3 and line["extrapolated"] is False and line["extrapolation"] is None
    assert abs(line["value"] * line["ms_per_step"] / 1e3 - 1.0) < 1e-9
    assert abs(line["timed_s"] - line["steps"] * line["ms_per_step"] / 1e3) < 1e-9
    # like for like: `value` times the evaluation with the tensor spectra pre-built; the evaluation that also
    # transforms the tensor planes is reported beside it and is the slower one
    assert cb["with_tensor_fft"]["s_per_eval"] > cb["s_per_eval"] and "oracle_tensor_spectra_s" in cb
