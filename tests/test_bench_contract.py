"""The reference arm of bench.py (`--impl reference`: the oracle on the host cores) runs without a GPU and prints the
contract's JSON line; the roofline bookkeeping of bench.py is consistent with the flop counts DESIGN.md states."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--n-markers", "4096",
                        "--nx", "16", "--steps", "3", "--warmup", "1", "--ref-sample", "2048"],
                       capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "particle-steps/s" and line["value"] > 0
    assert line["higher_is_better"] is True and line["dtype"] == "f64" and line["data"] == "synthetic"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "configs[1]" in line["config"]["workload"]


def test_flop_and_byte_counts_match_design():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.algorithmic_flops(1) == 1041 and bench.algorithmic_flops(0) == 328      # DESIGN.md section 6, K1
    assert bench.algorithmic_flops(1, mode=1) == 1156
    assert bench.algorithmic_flops(2) - bench.algorithmic_flops(1) == 2 * (10 * 20 + 2 * 38) + 73
    assert bench.algorithmic_bytes_push(1, ordered=True) == 144
    assert abs(bench.FP64_NOMINAL_TFLOPS - 37.22) < 0.01
