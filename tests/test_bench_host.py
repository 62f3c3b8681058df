"""Host logic of bench.py (no GPU): the algorithmic-byte model against SURVEY.md section 8(d)'s table, and the
`--impl reference` arm's JSON line."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
from kf_inputs import workloads  # noqa: E402


@pytest.mark.parametrize("name,gb", [("cfg1", 0.01687), ("cfg2", 1.0774), ("cfg3", 4.7736), ("cfg4", 4.2971)])
def test_algorithmic_bytes_match_the_survey_table(name, gb):
    # KV read (4096 B per context token and layer) + q + appended rows + outputs +
    # range partials written and re-read; "context S" = tokens resident at attend time
    wl = workloads.by_name(name)
    total, kv = bench.algorithmic_bytes(wl, [s - 1 for s in wl.contexts], wl.n_layers)
    assert kv == sum(wl.contexts) * 4096
    assert total / 1e9 == pytest.approx(gb, rel=2e-3)
    assert kv / total > 0.99                     # everything but the KV read is below 1%


def test_cfg5_bytes_per_layer_step():
    wl = workloads.by_name("cfg5")
    total, kv = bench.algorithmic_bytes(wl, [s - 1 for s in wl.contexts], wl.n_layers)
    assert total / wl.n_layers / 1e9 == pytest.approx(37.07, rel=3e-3)      # 37.07 GB per layer-step
    assert kv == wl.n_layers * sum(wl.contexts) * 4096


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2",
                          "--warmup", "1", "--workload", "cfg1"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-1000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == bench.METRIC and line["unit"] == "GB/s"
    assert line["value"] > 0 and line["vs_baseline"] is None and line["higher_is_better"] is True
    assert line["e2e"] == {"value": line["value"], "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    cb = line["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == line["value"] and "cfg1" in cb["sample"]
