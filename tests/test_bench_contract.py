"""CPU-only checks of bench.py's bookkeeping: the algorithmic flops per psi evaluation that the roofline fraction is
built on (SURVEY.md section 8(d) lists them for the five configs), and the JSON line of the reference arm."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench                                                      # noqa: E402
from paper_2208_05637_b200 import workloads as wl                 # noqa: E402


@pytest.mark.parametrize("cfg,expected", [(1, 2 * (842 + 320)), (2, 2 * (11185 + 2816)), (3, 2 * (41580 + 8192)),
                                          (4, 375830), (5, 423346)])
def test_algorithmic_flops_per_evaluation(cfg, expected):
    """2 nnz(M1, M2, M3) + 2 ((n-2) h + 4 h) with the sorted default degrees — the numbers SURVEY.md 8(d) states."""
    w = wl.WORKLOADS[cfg]
    params = wl.make_made_params(w.n_qubits, w.hidden, w.seed_weights)
    assert bench.algorithmic_flops_per_eval(params) == expected


def test_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` times the oracle on the host cores and prints ONE JSON line with the contract's keys
    (cfg 1 so that it runs in a second)."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--cfg", "1",
                          "--steps", "1", "--warmup", "0", "--oracle-samples", "8"],
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "pairs/s" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["gpu_launches"] == 0 and d["vs_baseline"] is None
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["value"] == d["value"]
    assert "workload" in d["config"]
