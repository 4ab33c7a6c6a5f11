"""bench.py's JSON contract, exercised on a tiny workload (GPU): every required key is present, the e2e arm moves the
bytes it claims and reproduces the device-resident energy, the launch counter is non-zero, and the streamed
(aux-block by aux-block) mode reproduces the resident energy bit for bit."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.strip().splitlines() if ln.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]  # exactly ONE JSON line
    return json.loads(lines[0])


def test_bench_line_contract_and_streamed_mode():
    wl = "custom:24,150,203"
    d = _bench("--workload", wl, "--steps", "2", "--warmup", "3")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "roofline", "cpu_baseline", "clocks", "e2e", "gpu_launches"):
        assert k in d, k
    assert d["unit"] == "TFLOP/s" and d["dtype"] == "f64" and d["n_gpus"] == 1 and d["vs_baseline"] is None
    assert d["config"]["workload"] == wl and d["value"] > 0 and d["gpu_launches"] > 0
    r = d["roofline"]
    assert r["bound"] == "tensor" and r["unit"] == "TFLOP/s" and 30.0 < r["peak"] < 45.0
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    e = d["e2e"]
    nbytes = 8 * (203 * (174 * 175 // 2) + 174 * 24 + 174 * 150 + 24 + 150 + 24 * 24)
    assert e["h2d_bytes_per_step"] == nbytes and e["d2h_bytes_per_step"] == 8 + 8 * 24 * 24
    assert e["same_result_as_device_arm"] and 0 < e["value"] <= d["value"] * 1.05
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0
    s = _bench("--workload", wl, "--streamed", "--stream-gb", "0.002")  # 16 aux rows per block
    assert s["config"]["inputs_resident"] is False and s["config"]["aux_block_rows"] == 16
    assert s["E_frag"] == d["E_frag"]  # same kernels, same order of aux rows inside B: identical bits
