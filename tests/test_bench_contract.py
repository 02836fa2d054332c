"""The reference arm of bench.py (the CPU oracle timed on the host cores) runs without a GPU:
its JSON line must carry the keys the driver reads."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args):
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                         timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, "exactly ONE JSON line on stdout"
    return json.loads(lines[0])


def test_reference_arm_prints_one_json_line_with_the_contract_keys():
    d = _run("--impl", "reference", "--steps", "1", "--warmup", "0")
    assert d["impl"] == "reference" and d["n_gpus"] == 1 and d["steps"] == 1 and d["warmup"] == 0
    assert d["metric"].startswith("Gnum/s") and d["unit"] == "Gnum/s" and d["higher_is_better"] is True
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["vs_baseline"] is None
    assert d["config"]["workload"] == "C2_u32" and "sample" in d["config"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and cb["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["data"].startswith("synthetic")


def test_reference_arm_other_workloads():
    for w, unit in (("C5b_xorwow", "flips/ns"), ("T1_xorwow_k100", "flips/ns"), ("N4_lfib521_draw", "Gnum/s")):
        d = _run("--impl", "reference", "--steps", "1", "--warmup", "0", "--workload", w)
        assert d["unit"] == unit and d["value"] > 0 and d["config"]["workload"] == w


# ---- the b200 arm's line, built from stub results on the CPU (no kernel runs here) ----------------------------
def _stub_result(bench, workload, long_name, bound, unit="Gnum/s"):
    r = {"name": long_name, "value": 1234.5678901234567, "unit": unit, "steps": 20, "warmup": 5,
         "ms_per_step": 0.67890123456789, "gpu_launches": 20, "dtype": "u32", "workload": workload,
         "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "reasons": ["sw_power_cap"], "samples": 4000}}
    r["roofline"] = bench.roofline(workload, bound, 4.3e9 if bound == "hbm" else 5e10, 6.8e-4, 7300.123)
    r["cpu"] = {"value": 0.0123456789012, "unit": unit, "cores": 16, "kind": "oracle", "sample": "a sample", "seconds": 2.01}
    return r


def test_b200_line_is_one_compact_parseable_line_for_every_suite():
    """round 1's line was 31 KB and the driver could not parse it (Missing #1): whatever the suite,
    the stdout line stays under 4 KB, is a single line, round-trips through json and carries the contract keys"""
    import types
    sys.path.insert(0, ROOT)
    import bench
    args = types.SimpleNamespace(workload="C2_u32")
    res = _stub_result(bench, "C2_u32", "C2_philox_2^20x1024_u32", "hbm")
    e2e = {"value": 13.512312312312312, "unit": "Gnum/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 1 << 32,
           "steps": 3, "ms_per_step": 79.712312312312, "api": "rng_fill_u32_host",
           "note": "inputs are scalars (kind, n_streams, seed); the result crosses the bus every step"}
    sample = "streams [0,1048576) of 1048576, 1024 draws each (fill_u32)"
    cpu = {"value": 0.5506378113756993, "unit": "Gnum/s", "cores": 16, "kind": "oracle", "sample": sample, "seconds": 7.81,
           "single_thread": {"value": 0.0412345678901, "unit": "Gnum/s", "cores": 1, "sample": sample, "seconds": 6.02}}
    ceil = {"memset_write_gbs": 7301.123456, "copy_rw_gbs": 6533.123456}
    info = {"desc": bench.SHORT_DESC["C2_u32"], "streams_per_gpu": 1 << 20, "l2": "4 GiB output per step > 126 MB L2, no flush needed"}
    for suite in ([], bench.BASELINE_SUITE, bench.SUITE):
        cfgs = [_stub_result(bench, n, n + "_some_long_name_2^22x4096", "alu" if ("draw" in n or n[0] in "T") else "hbm",
                             "flips/ns" if n[0] in "TC5" and "5b" in n or n[0] == "T" else "Gnum/s") for n, _, _ in suite]
        sustained = {"value": 1432.12, "unit": "Gnum/s", "steps": 3196, "ms_per_step": 0.74912, "seconds": 2.39,
                     "roofline_frac": 0.8912, "frac_vs_store_ceiling": 0.7801,
                     "clocks": {"sm_mhz": 1755.0, "sm_min_mhz": 1687.0, "sm_max_mhz": 1965.0, "reasons": ["sw_power_cap"],
                                "samples": 2390, "sample_period_ms": 1.0}}
        line = json.dumps(bench.build_line(res, args, 1, info, e2e, cpu, ceil, cfgs, sustained))
        assert "\n" not in line and len(line) < 4096, len(line)
        d = json.loads(line)
        for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                  "vs_baseline", "dtype", "data", "config", "clocks", "gpu_launches", "roofline", "e2e", "cpu_baseline"):
            assert k in d, k
        assert d["value"] > 0 and d["ms_per_step"] > 0 and d["gpu_launches"] > 0 and d["higher_is_better"] is True
        assert d["config"]["workload"] == "C2_u32"          # the same name the reference arm prints
        rl = d["roofline"]
        for k in ("bound", "achieved", "peak", "unit", "frac", "traffic", "algorithmic_bytes", "store_ceiling",
                  "frac_vs_store_ceiling", "ncu"):
            assert k in rl, k
        assert rl["bound"] == "hbm" and abs(rl["frac"] - rl["achieved"] / rl["peak"]) < 1e-3
        assert rl["ncu"] is None or rl["ncu"]["measured_in_this_run"] is False
        for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "api"):
            assert k in d["e2e"], k
        for k in ("value", "unit", "cores", "kind", "sample", "single_thread"):
            assert k in d["cpu_baseline"], k
        assert d["cpu_baseline"]["single_thread"]["cores"] == 1
        assert d["sustained"]["seconds"] >= 2.0 and d["sustained"]["clocks"]["samples"] > 1000
        if suite:
            assert d["configs_cols"][-2:] == ["frac_vs_store", "cpu_oracle"]
            assert all(row[-1] is not None and row[-1] > 0 for row in d["configs"])  # every BASELINE config has its CPU figure
            assert {"N2_seed_xs1024_random", "N2_seed_xs1024_skip", "C1big_u32"} <= {row[0] for row in d["configs"]}  # row a1
            assert len(d["configs"]) <= 11 and all(len(row) == len(d["configs_cols"]) for row in d["configs"])
            own = {n for n, _, _ in bench.BASELINE_SUITE}
            assert {row[0] for row in d["configs"]} == own


def test_alu_roofline_leads_with_the_ncu_figures():
    sys.path.insert(0, ROOT)
    import bench
    rl = bench.roofline("C3_draw", "alu", 1.07e10, 3.5e-4)
    assert rl["bound"] == "alu" and rl["basis"].startswith("frac = ncu smsp__issue_active")
    assert rl["ncu"]["measured_in_this_run"] is False and rl["ncu_issue_active_pct"] > 0 and rl["ncu_binding_pipe"]
    # north_star: the ncu-measured fraction of the issue peak leads; the hand count is kept beside it
    assert abs(rl["frac"] - rl["ncu_issue_active_pct"] / 100.0) < 1e-3
    assert abs(rl["frac_algorithmic"] - rl["achieved"] / rl["peak"]) < 1e-3
    # a workload without a committed capture falls back to the hand count and says so
    rl2 = bench.roofline("no_such_workload", "alu", 1.07e10, 3.5e-4)
    assert rl2["frac"] == rl2["frac_algorithmic"] and rl2["basis"] == "algorithmic instruction count"


def test_both_arms_name_the_workload_alike():
    """the reference arm's config.workload is args.workload; so is the b200 arm's (build_line)"""
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert src.count('"workload": args.workload') == 2
