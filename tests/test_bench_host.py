"""Host-side logic of bench.py and the build (no GPU): the roofline's `traffic` is READ from the
tracked ncu summaries (profiles/), golden digests are found and ordered, the N > 1 launch builds
the library under a lock, and the ALU-op model follows the PT cadence."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
from ea_inputs import CONFIGS  # noqa: E402


def test_traffic_comes_from_the_tracked_ncu_summaries():
    for cid, (fname, kernel) in bench.NCU_PROFILES.items():
        path = os.path.join(ROOT, "profiles", fname)
        assert os.path.exists(path), f"{fname}: bench.py names a profile that is not committed"
        text = open(path).read()
        assert kernel in text, f"{fname} is not a capture of {kernel}"
        p = bench.ncu_profile_numbers(cid)
        assert p is not None and p["file"] == "profiles/" + fname
        # the state is read at least once per launch and nothing like a second copy of it is moved
        cfg = CONFIGS[cid]
        state = 4 * cfg.n_temps * cfg.W * cfg.N + 4 * 3 * cfg.W * cfg.N
        assert 0.9 * state < p["dram_bytes"] < 2.5 * state, (p, state)
        assert 0 < p["alu_pipe_max_pct"] <= 100
    assert bench.ncu_profile_numbers(1) is None          # no capture for the tiny configs: traffic = null


def test_golden_checkpoints_cover_the_configs_full_length():
    for cid in (1, 2, 3, 4, 5):
        gold = bench.golden_checkpoints(cid)
        assert gold, f"no oracle digests for config {cid}"
        longest = max(max(cps) for cps in gold.values())
        assert longest == CONFIGS[cid].sweeps, (cid, longest)      # north_star: all five configs, full length
    assert len(bench.golden_checkpoints(4)) >= 4 and len(bench.golden_checkpoints(5)) >= 2


def test_alu_model_follows_the_pt_cadence():
    cfg = CONFIGS[4]
    assert bench.alu_ops_per_update(cfg, 5000) == bench.ALU_OPS_PER_WORD_UPDATE == 38.0
    import dataclasses
    assert bench.alu_ops_per_update(dataclasses.replace(cfg, swap_interval=10), 5000) == pytest.approx(30.8)
    assert bench.alu_ops_per_update(dataclasses.replace(cfg, swap_interval=0), 1000) == pytest.approx(30.008)


def test_shard_offsets():
    assert bench.shard_first_realization(0, 2048) == 0
    assert bench.shard_first_realization(3, 2048) == 3 * 2048
    assert bench.shard_first_realization(2, 40) == 2 * 64         # ragged shards start at a word boundary


def test_concurrent_builds_serialise_on_the_lock():
    """Two processes asking for the library at once (what N ranks do at start-up): both return the
    same, complete file."""
    code = ("import sys; sys.path.insert(0, %r); from paper_1311_5582_b200.build import build_library; "
            "p = build_library(); import os; print(os.path.getsize(p))" % ROOT)
    procs = [subprocess.Popen([sys.executable, "-c", code], stdout=subprocess.PIPE, text=True) for _ in range(2)]
    sizes = [p.communicate(timeout=600)[0].strip() for p in procs]
    assert all(p.returncode == 0 for p in procs) and sizes[0] == sizes[1] and int(sizes[0]) > 100000
