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


def test_flat_scalars_puts_the_per_kernel_figures_directly_under_roofline():
    """A record that keeps only the scalar keys of `roofline` must still carry the select / attention / pair figures, isolated
    (one launch, no PDL) beside the back-to-back period, the prefill times, the cached-step floor and the gather rate under load."""
    sys.path.insert(0, ROOT)
    import bench
    kern = lambda name, shape, **kw: {"kernel": name, "shape": shape, **kw}
    roof = {"kernels": [kern("forecast_select_kernel<128,false>", "batch 32: R=64", us=7.3, frac=0.71, us_isolated=9.2, frac_isolated=0.56),
                        kern("sparse_decode_kernel<128>", "batch 32: R=64", us=24.1, frac=0.87, us_isolated=26.0, frac_isolated=0.80),
                        kern("pair: forecast_select + sparse_decode", "batch 32: one layer", us_isolated=32.6, frac_isolated=0.8, frac_of_8tbs=0.64),
                        kern("sparse_decode_tc5_kernel (experiment)", "batch 32: same shape", us=37.9, frac=0.55),
                        kern("forecast_select_kernel<128,grid>", "f3 (reading q19)", us=23.2, frac=0.9),
                        kern("forecast_select_kernel<128,false>", "batch 4: R=8", us=3.6, frac=0.18, us_isolated=5.5, frac_isolated=0.12),
                        kern("sparse_decode_kernel<128>", "batch 4: R=8", us=7.6, frac=0.34, us_isolated=9.0, frac_isolated=0.29),
                        kern("pair: forecast_select + sparse_decode", "batch 4: one layer", us_isolated=11.8, frac_isolated=0.28, frac_of_8tbs=0.22)],
            "prefill_select": {"forecast_us_chunked": 152.5, "forecast_us_one_launch": 76.8},
            "reuse_cache": {"compute_floor_ms_per_step": 0.39},
            "gather_sweep": {"sweep": [{"batch": 4, "rows": [{"engine": "tma", "ctas": 4, "gbs_under_hbm_load": 33.4},
                                                              {"engine": "tma", "ctas": 8, "gbs_under_hbm_load": 49.5}]},
                                       {"batch": 32, "rows": [{"engine": "tma", "ctas": 8}]}]}}
    flat = bench.flat_scalars(roof, 8, "tma")
    assert flat["select_b32_us_isolated"] == 9.2 and flat["select_b32_us_period"] == 7.3 and flat["select_b32_frac_isolated"] == 0.56
    assert flat["attn_b32_frac_isolated"] == 0.80 and flat["attn_b4_us_isolated"] == 9.0 and flat["select_b4_frac_period"] == 0.18
    assert flat["pair_b32_us"] == 32.6 and flat["pair_b32_frac"] == 0.8 and flat["pair_b4_us"] == 11.8
    assert flat["prefill_chunked_us"] == 152.5 and flat["prefill_one_us"] == 76.8 and flat["floor_cached_step_ms"] == 0.39
    assert flat["gather_gbs_under_hbm_load"] == 49.5
    assert all(not isinstance(v, (dict, list)) for v in flat.values())
    assert bench.flat_scalars({}, 8, "tma") == {}
