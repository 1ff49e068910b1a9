"""bench.py's driver contract on a small workload: one JSON line with the keys the driver reads (value, e2e with the bytes it
copies, roofline with achieved / peak / frac, cpu_baseline, clocks, gpu_launches) and the legs beside them (vcycle, pcg, convdiff)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "2", "--scale", "2", "--steps", "2", "--warmup", "3",
                          "--kernel-reps", "5", "--roofline-idle", "0.1"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "e2e", "roofline", "cpu_baseline", "clocks", "gpu_launches", "vcycle", "pcg", "convdiff"):
        assert key in line, key
    assert line["n_gpus"] == 1 and line["steps"] == 2 and line["dtype"] == "f32" and line["data"] == "synthetic"
    assert line["value"] > 0 and line["gpu_launches"] > 0 and line["config"]["workload"].startswith("cfg2")
    assert line["e2e"]["value"] > 0 and line["e2e"]["h2d_bytes_per_step"] > 0 and line["e2e"]["d2h_bytes_per_step"] > 0
    r = line["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1 and line["cpu_baseline"]["value"] > 0
    cd = line["convdiff"]
    assert cd["roofline"]["bound"] == "alu" and cd["ms"] > 0 and cd["cpu_baseline"]["value"] > 0
    assert line["config"]["converged"] is True and line["pcg"]["converged"] is True
    # the level-0 kernels timed in the state the timed steps leave the board in, beside the burst figure; where the rest of a step goes
    assert r["in_step"]["ms"] > 0 and abs(r["in_step"]["frac"] - r["in_step"]["achieved"] / r["peak"]) < 1e-9
    bd = line["breakdown_ms"]
    assert all(bd[k] > 0 for k in ("set_coeff", "divergence", "solve", "gradient")) and bd["solve_cycles"] == line["config"]["cycles_run"]
    assert line["vcycle_256"] is None            # rides on the default config-4 run only
