"""bench.py contract pieces that can be checked without a GPU: the reference arm prints one JSON line with the
agreed keys; the roofline constants agree with DESIGN.md."""
import json
import subprocess
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600, cwd=str(ROOT))
    assert out.returncode == 0, out.stderr[-500:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "attempted site updates/s" and d["unit"] == "Gupd/s"
    assert d["higher_is_better"] is True and d["value"] > 0 and d["steps"] == 1
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": "Gupd/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "config3" in d["config"]["workload"]


def test_roofline_constants_match_design():
    sys.path.insert(0, str(ROOT))
    import bench
    assert bench.WORKLOAD == dict(L=1 << 17, tile=64, p=1.0, q=0.0, seed=42)      # BASELINE config 3
    assert bench.MCS_PER_STEP * 10 == 100                                         # default K = 10 steps = 100 MCS
    assert bench.ALG_BYTES_PER_UPDATE == 0.5 and bench.ALG_ALU_OPS_PER_UPDATE == 11.5
    design = (ROOT / "DESIGN.md").read_text()
    assert "**11.5**" in design and "18.6 T lane-ops/s" in design
