"""Host-side pieces of bench.py that need no GPU: the algorithmic byte count and the rule that ncu counters
are only used with the sources they were taken with."""
import csv
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_algorithmic_bytes_formula():
    import bench

    ab = bench.algorithmic_bytes(n_events=10, n_layers=26, raw_bytes=1000, n_clusters=300, n_tracks=20, n_track_hits=150)
    assert ab["raw"] == 1000 + 4 * 11
    assert ab["clusters"] == 30 * 300 + 4 * (10 * 26 + 1) + 4 * 11 + 4 * 10
    assert ab["tracks"] == 4 * 11 + 4 * 21 + 2 * 150 + 16 * 20
    assert ab["total"] == ab["raw"] + ab["clusters"] + ab["tracks"]
    # every compulsory byte is charged to exactly one kernel segment (tracks to follow + compact: counted once in `total`)
    assert ab["velo_cluster"] == ab["raw"] and ab["velo_seed"] == ab["clusters"] and ab["velo_follow"] == ab["tracks"]


def test_ncu_counters_are_tied_to_the_sources(tmp_path, monkeypatch):
    import bench

    h = bench.source_hash()
    assert len(h) == 16 and h == bench.source_hash()
    prof = tmp_path / "profiles"
    prof.mkdir()
    with open(prof / "x_counters.csv", "w") as f:
        w = csv.writer(f)
        w.writerow(["workload", "kernel", "dram_read_bytes", "dram_write_bytes", "warp_instructions",
                    "active_lanes_per_instruction", "source_hash"])
        w.writerow(["config2_10000", "velo_seed", 10, 20, 1000, 24.0, h])
        w.writerow(["config2_10000", "velo_cluster", 1, 2, 3, 18.0, "0123456789abcdef"])  # other sources: ignored
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    monkeypatch.setattr(bench, "source_hash", lambda: h)
    got = bench.ncu_counters("config2_10000")
    assert got["velo_seed"] == dict(dram_bytes=30, warp_instructions=1000, lanes=24.0) and "velo_cluster" not in got
    assert bench.ncu_counters("config3_10000") == {}


def test_committed_counters_name_their_sources():
    import glob

    files = glob.glob(os.path.join(ROOT, "profiles", "r02_counters.csv"))
    assert files
    with open(files[0]) as f:
        rows = list(csv.DictReader(f))
    assert rows and all(len(r["source_hash"]) == 16 for r in rows)
    assert {r["kernel"] for r in rows} >= {"velo_cluster", "velo_seed", "velo_follow", "compact_tracks"}
