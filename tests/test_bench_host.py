"""Host-side pieces of bench.py (no GPU): the algorithmic-work model of DESIGN.md 6 and the committed ncu summaries it reads."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench  # noqa: E402
from paper_1704_04381_b200 import workloads  # noqa: E402


def test_algorithmic_model_matches_design():
    assert bench.lattice_site_tests(64) == 930 and bench.lattice_site_tests(16) == 42
    assert bench.algorithmic_thread_instr(workloads.CONFIG_2) == 6 * 930 + 70 * 16 + 20 * 63 == 7960
    assert abs(bench.algorithmic_thread_instr(workloads.CONFIG_3) - 118780.2) < 1e-6
    assert abs(bench.algorithmic_thread_instr(workloads.CONFIG_5) - 1905513.0) < 1e-6


def test_every_listed_profile_is_committed_and_parses():
    for name, fname in bench.PROFILE_OF.items():
        assert name in workloads.CONFIGS, name
        assert os.path.exists(os.path.join(ROOT, "profiles", fname)), fname
        m = bench.profile_metrics(workloads.CONFIGS[name])
        assert m["traffic"] is not None and m["warp_inst_executed"] > 0 and 1.0 <= m["active_lane_ratio"] <= 32.0
        assert 0.0 < m["issue_active_pct"] <= 100.0
    # the dump workload's capture shows the 3.2 GB of conformations on their way to HBM
    assert bench.profile_metrics(workloads.CONFIG_5)["traffic"] > 3.0e9


def test_workload_table_and_perm_thresholds():
    assert workloads.CONFIGS[bench.DEFAULT_WORKLOAD] is workloads.CONFIG_2
    lo, hi, ref = workloads.perm_thresholds(32, 0.5, 2.0)
    assert len(lo) == len(hi) == 33 and all(a < b for a, b in zip(lo[2:], hi[2:])) and lo[2] < ref
    off = [workloads.shard(1000, r, 3) for r in range(3)]
    assert off[0][0] == 0 and sum(c for _, c in off) == 1000 and off[1][0] == off[0][1]


def test_model_and_perm_workloads_have_a_roofline_model_and_a_committed_summary():
    """Round 3 (VERDICT r2 missing 2): every model / PERM bench workload has an algorithmic-work model and an
    ncu summary under profiles/ that bench.py can read."""
    import bench
    from paper_1704_04381_b200 import workloads
    want = {"lattice_z26_N64_2p20": (30082.5, "per chain"), "lattice_z6_contact0.3_N64_2p20": (22774.5, "per chain"),
            "lattice_perm_N256_2p20": (478.0, "per attempted step")}
    for w in workloads.MODELS:
        per, unit = bench.model_thread_instr(w)
        assert per > 0 and unit in ("per chain", "per attempted step")
        if w.name in want:
            assert (per, unit) == want[w.name], (w.name, per, unit)
        alg, text = bench.alg_warp_inst(w, 1e6)
        assert alg > 0 and "thread-instr" in text
        m = bench.profile_metrics(w)
        assert m.get("file", "").startswith("profiles/r03_") and m["warp_inst_executed"] > 0 and 1.0 <= m["active_lane_ratio"] <= 32.0
    well = next(w for w in workloads.MODELS if w.lam)
    per, _ = bench.model_thread_instr(well)
    assert abs(per - 149600) < 200          # 6.25 candidates per trial: DESIGN.md 6
