"""CPU-side checks of bench.py's contract: the reference arm (the oracle, as it stands) prints one JSON line with the keys the
driver reads; the ncu side file parses; the CUDA arm refuses to run without a GPU instead of falling back."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--batch", "1", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "decode_tokens_per_s_128k" and line["unit"] == "tok/s"
    assert line["value"] > 0 and line["higher_is_better"] is True and line["data"] == "synthetic"
    assert line["config"]["workload"] == "cfg3_128k_pipeline" and line["config"]["context"] == 131072
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"] == {"value": line["value"], "unit": "tok/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_ncu_side_file_parses_and_names_its_source():
    sys.path.insert(0, ROOT)
    import bench
    m, src = bench.load_ncu_metrics()
    assert src and src.startswith("profiles/r2_ncu_metrics.csv@")
    for key in ("gather_b4", "select_b32", "attn_b32", "prefill_one", "prefill_chunked_pass"):
        assert m[key]["gpu__time_duration.sum"] > 0 and "dram__bytes_read.sum" in m[key]
    # the summary that names the commands behind the numbers is committed beside it
    assert os.path.exists(os.path.join(ROOT, "profiles", "r2_ncu_summary.md"))


def test_cuda_arm_has_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "3", "--warmup", "3"], capture_output=True, text=True,
                         timeout=300, cwd=ROOT)
    assert out.returncode != 0 and "no CUDA device" in (out.stderr + out.stdout)
