"""The line the driver reads from bench.py: built here from canned numbers through the same function
run_ours uses (build_headline), then checked as the driver would read it -- strict JSON, one line, at
most 4 KB, every key of the contract present.  (Round 2's line carried every extra and did not parse.)"""
import argparse
import json
import math

import pytest

import bench

REQUIRED = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
            "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline")


def _canned():
    args = argparse.Namespace(instances=4096, requests=1000, lam=4.0)
    return {
        "metric": bench.METRIC, "value": 753123456789.123456, "unit": bench.UNIT, "n_gpus": 8, "steps": 20, "warmup": 5,
        "ms_per_step": 5.351234567891234, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int32/int64", "data": "synthetic", "config": bench.workload_config(args),
        "decisions_per_sec": 3712345678.987654321, "requests_per_sec": 3061234567.123,
        "step_ms": [5.35 + 1e-7 * k for k in range(200)],                       # must NOT reach the headline
        "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "samples": 7,
                   "reasons": ["sw_power_cap", "hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"]},
        "e2e": {"value": 653123456789.12345, "unit": bench.UNIT, "h2d_bytes_per_step": 53280832, "d2h_bytes_per_step": 131858432,
                "ms_per_step": 6.171234567, "chunks": 8},
        "gpu_launches": 40,
        "roofline": {"kernel": "k_sim_slots (persistent simulator, phase B)", "bound": "alu", "achieved": 6.0912345678,
                     "peak": 37.2234567, "unit": "Tlane-op/s", "frac": 0.163712345, "traffic": 390592256.0,
                     "traffic_source": "x" * 300, "peak_source": "y" * 300, "kernel_ms": 5.16123456,
                     "algorithmic_ops_per_launch": 31433562508, "share_of_step": {"phase_a_keys_sort_rank": 0.035,
                                                                                  "phase_b_simulator": 0.9612345, "phase_c_p99": 0.0},
                     "hbm": {"algorithmic_bytes_per_launch": 524288000, "achieved_gbs": 101.6, "peak_gbs": 6544.0,
                             "frac": float("nan"), "peak_source": "z" * 200},
                     "note": "n" * 500},
        "fingerprint_fnv1a64": "0123456789abcdef",
        "cpu_baseline": {"value": 2761234567.891, "unit": bench.UNIT, "cores": 16, "kind": "oracle", "nproc": 16,
                         "sample": "all 4096 instances x 1000 requests x 4 policies (rank 0's batch), 9 repetitions, 12.9 s, "
                                   "instance-parallel over 16 host threads"},
        "kernels": [{"kernel": "k" * 80, "ms": 1.0}] * 50, "admit_sweep": [{"note": "w" * 400}] * 9,   # extras: never in the headline
        "stochastic_regime": {"points": [{"rho": float("inf")}] * 13},
    }


def test_headline_is_one_short_line_of_strict_json_with_every_contract_key():
    text = bench.build_headline(_canned(), bench.EXTRAS_FILE)
    assert "\n" not in text and len(text.encode()) <= 4096 and bench.HEADLINE_MAX_BYTES == 4096

    def no_constants(name):          # json.loads accepts NaN / Infinity unless told otherwise
        raise AssertionError(f"non-strict JSON constant {name}")
    line = json.loads(text, parse_constant=no_constants)
    for k in REQUIRED:
        assert k in line, k
    assert line["value"] > 0 and math.isclose(line["value"], 753123456789.123456, rel_tol=1e-6)
    assert math.isclose(line["ms_per_step"], 5.351234567891234, rel_tol=1e-6)
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in line["roofline"], k
    assert all(not isinstance(v, (list, dict)) for v in line["roofline"].values())      # scalar fields only
    assert line["roofline"]["hbm_frac"] is None                                         # NaN -> null
    assert math.isclose(line["roofline"]["share_of_step"], 0.9612345, rel_tol=1e-6)
    for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"):
        assert k in line["e2e"], k
    for k in ("value", "unit", "cores", "kind", "sample"):
        assert k in line["cpu_baseline"], k
    assert line["extras_file"] == bench.EXTRAS_FILE
    for k in ("step_ms", "kernels", "admit_sweep", "stochastic_regime"):
        assert k not in line


def test_headline_refuses_a_missing_key_and_an_oversized_line():
    full = _canned()
    del full["e2e"]
    with pytest.raises(KeyError):
        bench.build_headline(full)
    full = _canned()
    full["config"]["workload"] = "w" * 5000
    with pytest.raises(ValueError):
        bench.build_headline(full)


def test_committed_traffic_file_is_read():
    """... and only while the simulator sources are the ones that were profiled (SHA-256 stamped in the file)."""
    total, src = bench.profiled_dram_traffic()
    rec = json.load(open(bench.os.path.join(bench.ROOT, bench.SIM_PROFILE)))
    if bench._sources_sha256(rec["source_files"]) == rec["source_sha256"]:
        assert total == rec["dram__bytes_read.sum"] + rec["dram__bytes_write.sum"] and bench.SIM_PROFILE in src
    else:
        assert total is None and "capture again" in src


def test_reference_arm_prints_one_short_strict_json_line_on_a_cpu_box():
    """`bench.py --impl reference` is the driver's other arm: the oracle on the host cores, no GPU.  Run it
    on a small batch as the driver would (a subprocess), and read its last stdout line the same way."""
    import os
    import subprocess
    import sys
    r = subprocess.run([sys.executable, os.path.join(bench.ROOT, "bench.py"), "--impl", "reference", "--instances", "8",
                        "--requests", "60", "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    last = r.stdout.strip().splitlines()[-1]
    assert len(last.encode()) <= 4096

    def no_constants(name):
        raise AssertionError(f"non-strict JSON constant {name}")
    line = json.loads(last, parse_constant=no_constants)
    assert line["impl"] == "reference" and line["metric"] == bench.METRIC and line["unit"] == bench.UNIT
    assert line["value"] > 0 and line["steps"] == 2 and line["gpu_launches"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"] == {"value": line["value"], "unit": bench.UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    # under torchrun every rank but 0 exits 0 without work and without output
    r1 = subprocess.run([sys.executable, os.path.join(bench.ROOT, "bench.py"), "--impl", "reference", "--instances", "8",
                         "--requests", "60", "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=300,
                        env=dict(os.environ, RANK="1", WORLD_SIZE="2"))
    assert r1.returncode == 0 and r1.stdout.strip() == ""
