"""CPU tests of the host-side harness: sharding, max-over-ranks over gloo with world_size 2,
clock-record parsing, roofline byte counts."""
import os
import subprocess
import sys
import textwrap

import numpy as np

from paper_2110_13693_b200 import harness, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_ranges_partition():
    for n, world in [(16384, 1), (16384, 8), (65536, 3), (10, 4), (3, 8)]:
        covered = []
        for r in range(world):
            lo, hi = harness.shard_range(n, r, world)
            covered.extend(range(lo, hi))
        assert covered == list(range(n))
    assert harness.weak_rows(16384, 3) == (3 * 16384, 4 * 16384)


def test_weak_rows_give_distinct_plans():
    a = W.perm_rows(0, 50, np.arange(*harness.weak_rows(4, 0)))
    b = W.perm_rows(0, 50, np.arange(*harness.weak_rows(4, 1)))
    assert not any((x == y).all() for x in a for y in b)
    assert all(sorted(r.tolist()) == list(range(50)) for r in np.concatenate([a, b]))


def test_perms_torch_equals_numpy():
    import torch
    for n, lo, hi in [(20, 0, 64), (500, 1000, 1016), (4000, 16380, 16384)]:
        t = W.perms_torch(0, n, lo, hi, "cpu").numpy()
        assert np.array_equal(t, W.perm_rows(0, n, np.arange(lo, hi)))


def test_two_rank_gloo_max_and_sharding(tmp_path):
    """world_size 2 on CPU (gloo): each rank owns a disjoint candidate range and the reported
    time is the max over ranks."""
    script = tmp_path / "rank.py"
    script.write_text(textwrap.dedent(f"""
        import sys
        sys.path.insert(0, {ROOT!r})
        from paper_2110_13693_b200 import harness
        rank, local_rank, world = harness.init_dist("gloo")
        lo, hi = harness.weak_rows(100, rank)
        harness.barrier(world)
        t = harness.max_over_ranks(1.0 + rank, world)
        tot = harness.sum_over_ranks(hi - lo, world)
        print(f"RESULT {{rank}} {{lo}} {{hi}} {{t}} {{tot}}")
    """))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29533", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r), LOCAL_RANK=str(r)),
                              stdout=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=120)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs)
    rows = sorted(l.split()[1:] for o in outs for l in o.splitlines() if l.startswith("RESULT"))
    assert rows == [["0", "0", "100", "2.0", "200.0"], ["1", "100", "200", "2.0", "200.0"]]


def test_clock_parsing_and_rejection():
    lines = ["0, 1905, 1965, 612.1, 0x0000000000000004, Not Active, Not Active, Not Active, Active",
             "0, 1890, 1965, 640.0, 0x0000000000000000, Not Active, Not Active, Not Active, Not Active",
             "0, 1920, 1965, 598.3, 0x0000000000000000, Not Active, Not Active, Not Active, Not Active"]
    c = harness.parse_clock_lines(lines)
    assert c["sm_mhz"] == 1905 and c["sm_max_mhz"] == 1965 and c["reasons"] == ["sw_power_cap"]
    assert not harness.clocks_rejected(c)
    hot = ["0, 900, 1965, 300, 0x8, Not Active, Active, Not Active, Not Active"]
    assert harness.clocks_rejected(harness.parse_clock_lines(hot))
    locked = ["0, 600, 1965, 200, 0x0, Not Active, Not Active, Not Active, Not Active"]
    assert harness.clocks_rejected(harness.parse_clock_lines(locked))
    assert harness.parse_clock_lines([])["sm_mhz"] is None


def test_algorithmic_bytes_match_survey_table():
    b = harness.algorithmic_bytes_per_candidate(4000, 9919)
    assert b["survey"] == 4 * 4000 + 8 * 4000 + 4 * 9919 + 36  # ~87.7 KB, SURVEY.md 8(d)
    assert b["hbm_compulsory"] == 16036 and b["packed"] < b["survey"]


def test_bench_reference_arm_prints_one_json_line():
    import json
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                          "--steps", "1", "--warmup", "1"], capture_output=True, text=True,
                         timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["value"] > 0 and line["e2e"]["h2d_bytes_per_step"] == 0


def test_ncu_counters_are_quoted_only_for_the_sources_they_were_captured_on(tmp_path):
    """bench.py prints roofline.traffic / binding_resource from profiles/ncu_counters.csv only while
    the evaluation-path sources hash to the fingerprint stored beside the counters."""
    import shutil
    root = tmp_path / "repo"
    csrc = root / "paper_2110_13693_b200" / "csrc"
    csrc.mkdir(parents=True)
    (root / "profiles").mkdir()
    for name in harness.EVAL_PATH_SOURCES:
        shutil.copy(os.path.join(ROOT, "paper_2110_13693_b200", "csrc", name), csrc / name)
    sha = harness.csrc_sha16(str(root))
    assert sha == harness.csrc_sha16(ROOT) and len(sha) == 16
    (root / "profiles" / "ncu_counters.csv").write_text(
        "csrc_sha16,workload,counter,value,source\n# comment\n"
        f"{sha},paper,dram_bytes,521.0e6,profiles/x.md\n{sha},paper,warp_inst,2.5e8,profiles/x.md\n"
        "0123456789abcdef,paper,dram_bytes,1.0,profiles/old.md\n")
    c = harness.ncu_counters(str(root))
    assert c["paper"]["dram_bytes"] == 521.0e6 and c["paper"]["warp_inst"] == 2.5e8
    assert c["paper"]["source"] == "profiles/x.md" and not c["stale"]
    with open(csrc / "whp_fast.cu", "a") as f:
        f.write("// edited\n")
    c2 = harness.ncu_counters(str(root))
    assert "paper" not in c2 and c2["stale"] and c2["csrc_sha16"] != sha
    os.remove(root / "profiles" / "ncu_counters.csv")
    c3 = harness.ncu_counters(str(root))
    assert "paper" not in c3 and not c3["stale"]


def test_binding_constants_match_the_header():
    """whp.py mirrors the enums of include/whp.h by value."""
    import re
    from paper_2110_13693_b200 import whp
    text = open(os.path.join(ROOT, "include", "whp.h")).read()
    enums = dict((k, int(v)) for k, v in re.findall(r"\b(WHP_[A-Z0-9_]+)\s*=\s*(\d+)", text))
    for name, value in enums.items():
        if name.startswith("WHP_DEBUG_"):
            assert getattr(whp, name[4:]) == value, name
        elif name.startswith("WHP_ROUTE_"):
            assert getattr(whp, name[4:]) == value, name
        elif name.startswith("WHP_ERR_") or name == "WHP_OK":
            assert getattr(whp, name[4:]) == value, name
    assert enums["WHP_DEBUG_K1_WARPS"] == 4 and enums["WHP_ROUTE_LARGEST_GAP"] == 2
