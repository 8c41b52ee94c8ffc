"""CPU-side checks of bench.py's bookkeeping (no GPU, no timing): both arms print the same `config` object, the recorded DRAM
traffic is only reported for the configuration it was captured on, and the reference arm (the oracle on a tiny sample) prints the
keys the contract asks for."""
import importlib.util
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench():
    spec = importlib.util.spec_from_file_location("bench", os.path.join(ROOT, "bench.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_recorded_traffic_only_for_the_captured_configuration():
    b = _bench()
    rec = json.load(open(os.path.join(ROOT, "profiles", "r02_force_fast_traffic.json")))
    want = rec["dram_bytes_read"] + rec["dram_bytes_write"]
    assert b.recorded_traffic(rec["n_j"], rec["n_i"], rec["jsplits"]) == want > 0
    assert b.recorded_traffic(rec["n_j"], rec["n_i"], rec["jsplits"] // 2) is None       # another split count: another traffic
    assert b.recorded_traffic(rec["n_j"] // 2, rec["n_i"] // 2, rec["jsplits"]) is None


def test_both_arms_print_the_same_config_and_the_reference_arm_has_the_contract_keys():
    b = _bench()
    from paper_0902_4463_b200 import inputs
    n = 4096
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--n", str(n), "--steps", "1", "--warmup", "0",
                          "--ref-seconds", "0.2"], capture_output=True, text=True, cwd=ROOT, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == b.METRIC and line["unit"] == "interactions/s" and line["higher_is_better"] is True
    assert line["config"] == b.bench_config(inputs, n, inputs.config(b.WORKLOAD, n=n)[3], 1, 1)
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1 and line["cpu_baseline"]["value"] == line["value"] > 0
    assert line["e2e"] == {"value": line["value"], "unit": "interactions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
