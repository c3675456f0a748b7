"""bench.py prints ONE JSON line that carries the keys the measurement contract asks for
(DESIGN.md section 7).  Run on a small parity config so that it takes seconds."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_json_line_contract():
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--config", "water_96k", "--steps", "5", "--warmup", "3",
           "--cpu-baseline-atoms", "96000", "--cpu-baseline-steps", "1"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["metric"] == "rbe_kspace_ns_per_atom_step" and d["unit"] == "ns/atom/step"
    assert d["n_gpus"] == 1 and d["steps"] == 5 and d["warmup"] == 3 and d["higher_is_better"] is False
    assert d["scaling"] == "weak" and d["vs_baseline"] is None and d["dtype"] == "f32" and d["data"] == "synthetic"
    assert d["config"]["workload"] == "water_96k" and "l2" in d["config"]
    assert d["value"] > 0 and abs(d["value"] - d["ms_per_step"] * 1e6 / 96000) < 1e-9 * d["value"] + 1e-12
    r = d["roofline"]
    assert r["bound"] == "alu" and r["peak"] > 0 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and "traffic" in r
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > d["value"] and "sample" in c
    e = d["e2e"]
    assert e["value"] > d["value"] and e["h2d_bytes_per_step"] >= 12 * 96000 and e["d2h_bytes_per_step"] == 12 * 96000
    assert e["float4_ms_per_step"] > 0
    assert d["gpu_launches"] == 1 * 5 and d["config"]["launch"]["step_fused"] == 1      # one cooperative launch per step
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert d["graph_step"]["gpu_launches_per_step"] == 2 and d["short_range"]["ms_per_call"] > 0
    # hygiene keys of round 2: peaks measured in the same run, executed-work fractions, both kernels, one-thread oracle
    lanes = d["peaks"]["lanes_per_sm_per_clk"]
    assert 14.0 <= lanes["mufu"] <= 16.5 and 110.0 <= lanes["ffma"] <= 130.0 and 55.0 <= lanes["imad"] <= 66.0
    assert r["kernel"] == "step_kernel" and r["executed"]["mufu_per_pair"] == 2.5 and "measured in this run" in r["peak_source"]
    assert [k["kernel"] for k in d["roofline_kernels"]] == ["sf_kernel", "f_kernel"]
    assert c["one_thread"]["value"] > 0 and c["speedup_all_threads_vs_one"] > 0
    assert d["kernels_ms"]["two_launch_step"] > 0 and d["kernels_ms"]["step_call"] == d["ms_per_step"]
    # honesty keys of round 3: the timed step checked against the oracle inside the run, the step without charge pairing,
    # one whole MD step
    pr = d["parity_in_run"]
    assert pr["passed"] is True and pr["timed_step_reproduced_bitwise"] is True and pr["atoms"] == 96000
    assert pr["F_relL2"] <= 2e-5 and pr["rho_err"] <= 1e-6
    un = r["unpaired"]
    assert un["ms_per_step"] > 0 and un["executed_mufu_per_pair"] == 3.0 and abs(un["value"] - un["ms_per_step"] * 1e6 / 96000) < 1e-9
    st = d["static_step"]
    assert st["ms_per_step"] > 0 and st["gpu_launches_per_step"] == 1 and st["ms_per_step"] < 2 * d["ms_per_step"]
    assert r["executed"]["xu_per_pair"] is None or r["executed"]["xu_per_pair"] > 0 if "xu_per_pair" in r["executed"] else True
    md = d["md_step"]
    assert md["ms_per_step"] > d["short_range"]["ms_per_call"] * 0.2 and md["graph_launches_per_step"] == 1 and md["finite"] is True
    assert md["kernels_per_step"] == 11 and 90_000 <= md["N"] <= 100_000
