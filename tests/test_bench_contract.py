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


def test_algorithmic_units_follow_from_the_method():
    """What the mathematics fixes about the roofline inputs: config 3 of BASELINE.json, one launch of the tiled update
    kernel = one colour = L^2/4 attempted updates, each 2-bit site read once and written once per MCS = L^2/8
    bytes per launch, five 32-bit shared-memory loads and one XOR reduction per attempt, one sigma_y bit per site for
    the measurement (eq. 3 walks plane Y only)."""
    sys.path.insert(0, str(ROOT))
    import bench
    base = json.loads((ROOT / "BASELINE.json").read_text())
    assert "2^17" in base["configs"][2] and "tile 64" in base["configs"][2] and "seed 42" in base["configs"][2]
    assert bench.WORKLOAD == dict(L=1 << 17, tile=64, p=1.0, q=0.0, seed=42)
    assert bench.CONFIGS[3]["mcs_per_step"] * bench.CONFIGS[3]["steps"] == 100          # "100 MCS timed"
    L = bench.WORKLOAD["L"]
    updates_per_launch = L * L // 4
    assert updates_per_launch == 2 ** 32
    assert bench.ALG_BYTES_PER_UPDATE * updates_per_launch == L * L / 8                  # 2 bits in + 2 bits out per site and MCS, / 4 launches
    assert 4 * bench.ALG_BYTES_PER_UPDATE * updates_per_launch == 2 * (L * L * 2 / 8)    # = the packed lattice read and written once per MCS
    assert bench.ALG_SMEM_BYTES_PER_UPDATE == (5 + 1) * 4
    assert bench.ALG_BYTES_PER_SITE_MEASURE * 8 == 1
    for n, c in bench.CONFIGS.items():                                                   # every config is a valid handle
        assert c["L"] % (2 * c["tile"]) == 0 and c["L"] % 32 == 0 and 0 <= c["q"] <= c["p"] <= 1
    assert bench.CONFIGS[4]["replicas"] == 1024 and bench.CONFIGS[5]["L"] == 1 << 19
