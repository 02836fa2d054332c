"""-m "not gpu": the committed profile summaries are what the committed tools make of the committed raw pages
(host logic only; nothing here runs a kernel)."""
import csv
import json
import os

import ncu_summary  # tests/ncu_summary.py (conftest puts tests/ on sys.path)

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PROF = os.path.join(ROOT, "profiles")


def test_launch_summary_is_reproducible_from_the_raw_launch_list(tmp_path):
    for rnd in ("r02", "r03"):
        raw = os.path.join(PROF, f"{rnd}_launches_bench_primary.csv")
        out = tmp_path / f"{rnd}_summary.csv"
        n = ncu_summary.summarise_launches(raw, str(out))
        got = list(csv.reader(open(out)))
        exp = list(csv.reader(open(os.path.join(PROF, f"{rnd}_launches_bench_primary_summary.csv"))))
        assert n == len(got) - 1 and got == exp
        # the headline kernel is every launch of the library in the primary step
        lib = [r for r in got[1:] if "rngb200::" in r[0]]
        assert len(lib) == 1 and "philox_fill_warp_kernel" in lib[0][0] and int(lib[0][3]) == 23  # 20 steps + 3 warm-up


def test_traffic_json_and_the_text_page_are_rederived_from_the_committed_raw_pages(tmp_path):
    """profiles/traffic.json (what bench.py quotes as roofline.traffic / roofline.ncu) and the text page are
    exactly what tests/ncu_summary.py makes of profiles/r03_raw/ -- number by number, not just by kernel name"""
    text, js = tmp_path / "page.txt", tmp_path / "traffic.json"
    src = "profiles/r03_ncu_full_all_workloads.txt"
    made = ncu_summary.summarise(os.path.join(PROF, "r03_raw"), str(text), str(js), src, fresh=True)
    committed = json.load(open(os.path.join(PROF, "traffic.json")))
    again = json.load(open(js))
    assert set(again) == set(committed)
    for name in committed:
        assert again[name] == committed[name], name
    assert len(made) == len([k for k in committed if not k.startswith("_")]) >= 31
    assert open(text).read() == open(os.path.join(ROOT, src)).read()


def test_traffic_json_entries_cite_existing_captures_and_carry_the_bench_keys():
    d = json.load(open(os.path.join(PROF, "traffic.json")))
    entries = {k: v for k, v in d.items() if not k.startswith("_")}
    assert {"C2_u32", "C2_f32", "C1_u32", "C1big_u32", "C3_draw", "C4_fill", "C4_draw", "C5b_philox", "C5b_xorwow",
            "N2_seed_xs1024_random", "N2_seed_xs1024_skip"} <= set(entries)  # every row of bench.py's baseline suite
    for name, e in entries.items():
        assert os.path.exists(os.path.join(ROOT, e["source"])), (name, e["source"])
        assert os.path.exists(os.path.join(PROF, "r03_raw", f"raw_{name}.csv")), name
        text = open(os.path.join(ROOT, e["source"])).read()
        kernel = e["kernel"].replace("void ", "").split("(")[0]
        assert kernel in text, (name, kernel)  # the capture the entry cites holds this kernel
        for key in ("kernel", "dram_bytes_per_launch", "ncu_time_us", "issue_active_pct"):
            assert key in e, (name, key)
    # algorithmic bytes of the headline (4 B x 2^30 draws) against the measured DRAM traffic: no wasted re-reads
    assert 0.95 < entries["C2_u32"]["dram_bytes_per_launch"] / (4 * 2 ** 30) < 1.02
    # the seeding captures are of the kernels as they stand (byte tables; round 1's xs_skip_level_kernel capture is gone)
    assert "xs_skip_level_table_kernel" in entries["N2_seed_xs1024_skip"]["kernel"]
    assert "seed_xs1024_kernel" in entries["N2_seed_xs1024_random"]["kernel"]
