"""bench.py's LAST stdout line is what the driver parses: one compact JSON object with the contract keys, well under
4 KB whatever the side phases hold (round 2's single 21.7 KB line was cut by the driver and the round went unmeasured).
No GPU here: the line is built from a canned result of the shape run_ours() produces."""
import json
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import bench  # noqa: E402


def canned(big: int = 400) -> dict:
    blob = {f"key_{i}": {"ms": {"mean": 1.2345678, "median": 1.2, "best": 1.1, "n": 20}, "note": "x" * 60} for i in range(big)}
    return {
        "metric": bench.METRIC, "value": 28412.123456789, "unit": bench.UNIT, "n_gpus": 1, "steps": 40, "warmup": 5,
        "ms_per_step": 1.1263, "ms_per_step_stats_rank0": {"mean": 1.1, "median": 1.1, "best": 1.0, "n": 40},
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u16 mod q (u8 x u8 -> s32 tensor, u32/u64 integer)", "data": "synthetic",
        "config": {"workload": bench.WORKLOAD, "instances_per_step_per_gpu": 32, "parallelism": "instances x1 (no collective)",
                   "l2": "inputs larger than L2 (A 256 MiB read twice + U 128 MiB written and read per step); no flush",
                   "regime": "burst (K steps back to back, tens of ms; see `sustained` for the power-capped regime)",
                   "all_bits_recovered": True},
        "clocks": {"sm_mhz": 1875.0, "sm_max_mhz": 1965, "reasons": ["sw_power_cap"], "samples": 23},
        "e2e": {"value": 12270.5, "unit": bench.UNIT, "h2d_bytes_per_step": 18350080, "d2h_bytes_per_step": 135283712,
                "ms_per_step": 2.607, "ms_per_step_stats_rank0": {"mean": 2.6}, "api": "lwe_kem_host (pinned host buffers; "
                "ciphertext U,v and b copied back)", "d2h_GBps": 51.9,
                "without_reading_U_back": {"value": 24480.1, "ms_per_step": 1.307, "note": "y" * 100}},
        "gpu_launches": 160,
        "roofline": {"kernel": "encaps_tc2_kernel (tcgen05 cta_group::2 kind::i8, B operand expanded from bits in-kernel)",
                     "bound": "tensor", "achieved": 4359.1, "peak": 3316.8, "unit": "TOP/s", "frac": 1.3142, "traffic": 415e6,
                     "peak_kind": "z" * 220, "ms_per_launch": 1.0089, "frac_of_measured_int8_pipe": 0.93,
                     "measured_int8_pipe_TOPs": 4690.0, "frac_of_nominal_4500": 0.97, "library_int8_gemm": blob,
                     "int8_pipe_probe": blob},
        "dominant_kernel_share_of_step": 0.895,
        "sustained": {"value_settled": 25500.0, "gemm": {"int8_TOPs": 3900.0, "frac_of_measured_int8_pipe": 0.95}, "clocks": blob},
        "cpu_baseline": {"value": 0.0318, "unit": bench.UNIT, "cores": 16, "kind": "oracle", "sample": "s" * 200,
                         "host_cpus": 16, "configs": blob},
        "modular_GOPs": 123456.7, "kernels": blob, "kernels_note": "n" * 100,
        "phases": {"keygen_stored_B1": {"frac_hbm": 0.91, "back_to_back": {"frac_hbm": 0.99}},
                   "keygen_stored_B32": {"back_to_back": {"frac_hbm": 0.87}}, "decaps_B32": {"back_to_back": {"frac_hbm": 0.85}},
                   "rng_fill_1GiB": {"GBps": 813.0}, "pipelined_B32": {"step": {"kem_per_s": 29300.0}}, "paper_table1_all_rows": blob},
        "peaks": {"hbm_gbs": 6556.2}, "details": "gpurun_out/bench_details.json",
    }


def test_final_line_is_compact_and_carries_the_contract_keys():
    line = bench.dumps_compact(canned())
    assert "\n" not in line and len(line) < bench.MAX_LINE_BYTES < 4097
    d = json.loads(line)
    for key in bench.COMPACT_KEYS:
        assert key in d, key
    assert d["value"] > 0 and d["e2e"]["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    for key in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert key in d["roofline"], key
    for key in ("value", "unit", "cores", "kind", "sample"):
        assert key in d["cpu_baseline"], key
    for key in ("sm_mhz", "sm_max_mhz", "reasons"):
        assert key in d["clocks"], key
    assert d["config"]["workload"] == bench.WORKLOAD
    assert "phases" not in d and "kernels" not in d and "configs" not in d["cpu_baseline"]
    assert d["sustained_value"] == 25500.0 and d["keygen_gemv_frac_hbm"] == 0.99 and d["decaps_frac_hbm"] == 0.85


def test_final_line_stays_small_however_large_the_details_grow():
    full = canned(big=5000)
    full["config"]["regime"] = "r" * 3000                    # even a contract field grown absurdly must not break the line
    full["cpu_baseline"]["sample"] = "s" * 3000
    try:
        line = bench.dumps_compact(full)
    except AssertionError:
        line = None
    assert line is None or len(line) < bench.MAX_LINE_BYTES  # never a long line: it either fits or refuses loudly


def test_both_arms_name_the_same_workload():
    src = (ROOT / "bench.py").read_text()
    assert src.count('"workload": WORKLOAD') == 2            # run_ours and run_reference
