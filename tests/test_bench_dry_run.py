"""bench.py's own code path, executed against the host model (no GPU): the line it prints has the keys the contract names.
The numbers in that line are meaningless here (tests/emu/bench_dry.py says why); the structure and the parity flags are not."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_line_has_the_contract_keys_and_matches_the_oracle():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "emu", "bench_dry.py"), "--events", "10", "--steps", "2",
                          "--warmup", "3", "--cpu-events", "4"], capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert key in line, key
    assert line["metric"] == "events_per_s" and line["n_gpus"] == 1 and line["steps"] == 2 and line["warmup"] >= 3
    assert line["vs_baseline"] is None and line["dtype"] == "int32" and line["data"] == "synthetic"
    assert line["config"]["workload"] == "cfg3_100k_events_pileup40" and line["config"]["events"] == 10
    assert line["gpu_launches"] == 3 * 2                                      # fast kernel, general kernel (deferred list), assign: per step
    for key in ("bound", "achieved", "peak", "unit", "frac", "traffic", "frac_pipeline", "kernel"):
        assert key in line["roofline"], key
    assert line["roofline"]["traffic"] is None                                # not the full workload: no ncu figure applies
    for key in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"):
        assert key in line["e2e"], key
    assert line["e2e"]["same_as_device_results"] is True
    for key in ("value", "unit", "cores", "kind", "sample"):
        assert key in line["cpu_baseline"], key
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["gpu_outputs_identical_on_sample"] is True
