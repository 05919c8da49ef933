"""Host-side logic of bench.py (CPU): the timed schedule, the schedule mean, and the ncu-summary reader."""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402


def test_schedule_has_search_steps_whatever_k_is():
    for nstlist, k in [(100, 20), (100, 200), (100, 1), (40, 20), (2, 7), (100, 0)]:
        pos = bench.Replica.schedule(nstlist, k)
        searches = [i for i, t in enumerate(pos) if t == 0]
        assert len(searches) >= 3                                 # the driver's --steps 20 still times (a2)-(a5)
        assert sum(1 for t in pos if t != 0) == k                 # exactly K inner steps
        assert pos[0] == 0                                        # a list exists before the first inner step
        assert all(0 < t < nstlist for t in pos if t != 0)        # inner positions stay inside one list lifetime
        # inside one lifetime the inner positions run 1, 2, 3, ... (the rolling parts alternate as in a real run)
        for a, b in zip(searches, searches[1:] + [len(pos)]):
            run = pos[a + 1:b]
            assert run == [1 + (j % max(nstlist - 1, 1)) for j in range(len(run))]


def test_schedule_mean_weights():
    pop = {"search": [3 * 0.6, 3, 3 * 1000, 3 * 10], "inner": [20 * 0.1, 20, 20 * 900, 20 * 8]}
    ms, pairs, slots = bench.schedule_mean(pop, 100)
    assert abs(ms - (0.6 + 99 * 0.1) / 100) < 1e-12
    assert abs(pairs - (1000 + 99 * 900) / 100) < 1e-9
    assert abs(slots - (10 + 99 * 8) / 100) < 1e-9
    ms1, _, _ = bench.schedule_mean({"search": [1.5, 3, 0, 0], "inner": [0.0, 0, 0, 0]}, 100)   # no inner steps timed
    assert abs(ms1 - 0.5) < 1e-12


def test_ncu_traffic_reads_the_newest_committed_summary(tmp_path, monkeypatch):
    prof = tmp_path / "profiles"
    prof.mkdir()
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    assert bench.ncu_traffic("force", 2, "ewald")[0] is None      # nothing committed: null, with the reason
    (prof / "r1c_force_full_cfg2.md").write_text("| `dram__bytes_read.sum` | Mbyte | 10.0 | 11.0 |\n| `dram__bytes_write.sum` | byte | 0 | 0 |\n")
    (prof / "r2b_force_full_cfg2.md").write_text("| `dram__bytes_read.sum` | Mbyte | 14.5 | 14.6 |\n| `dram__bytes_write.sum` | Kbyte | 2 | 3 |\n")
    (prof / "r2b_force_full_cfg2_rf.md").write_text("| `dram__bytes_read.sum` | Mbyte | 20 | 20 |\n| `dram__bytes_write.sum` | byte | 0 | 0 |\n")
    v, src = bench.ncu_traffic("force", 2, "ewald")
    assert abs(v - (14.5e6 + 2e3)) < 1 and src.endswith("r2b_force_full_cfg2.md")
    assert abs(bench.ncu_traffic("force", 2, "rf")[0] - 20e6) < 1
    assert bench.ncu_traffic("prune", 2, "ewald")[0] is None
