"""Writes tests/golden/oracle_regression.json from the oracle alone (never from the CUDA path).

Run: python tests/golden/make_golden.py
"""
import hashlib
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1912_09161_b200 import workload  # noqa: E402

CASES = [(0, None), (1, 24), (2, 24), (3, 8)]


def digest(res):
    h = hashlib.sha256()
    c, t = res.clusters, res.tracks
    for a in (c.event_offsets, c.layer_offsets, c.key, c.n_pixels, c.sum_col, c.sum_row, c.x, c.y, c.z, c.phi16,
              c.checksum, c.status, t.event_offsets, t.hit_offsets, t.hits, t.x0, t.y0, t.tx, t.ty):
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()


def compute():
    out = {}
    for config, n in CASES:
        b = workload.generate(config, n_events=n)
        res = oracle.reconstruct(b.geometry, b.raw, b.event_offsets)
        out[f"config{config}"] = dict(n_events=b.n_events, input_sha=b.sha(), n_clusters=int(res.clusters.event_offsets[-1]),
                                      n_tracks=int(res.tracks.event_offsets[-1]), n_track_hits=int(len(res.tracks.hits)),
                                      output_sha256=digest(res))
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.json")
    with open(path, "w") as f:
        json.dump(compute(), f, indent=1, sort_keys=True)
    print("wrote", path)
