"""The parity comparator itself (tests/helpers.py): the near-cut excuse of BASELINE.json's tolerance clause must apply
only where the oracle logged a near-cut decision that touches (or precedes) the differing hits (R7)."""
import copy

import numpy as np

from tests.helpers import compare_tracks


def _drop_last_hit_of_first_long_track(tracks, e):
    """A copy of `tracks` in which the first track of event e with > 3 hits loses its last hit."""
    t = copy.deepcopy(tracks)
    for i in range(int(t.event_offsets[e]), int(t.event_offsets[e + 1])):
        h0, h1 = int(t.hit_offsets[i]), int(t.hit_offsets[i + 1])
        if h1 - h0 > 3:
            dropped = int(t.hits[h1 - 1])
            t.hits = np.delete(t.hits, h1 - 1)
            t.hit_offsets = t.hit_offsets.copy()
            t.hit_offsets[i + 1:] -= 1
            return t, dropped, [int(h) for h in tracks.hits[h0:h1]]
    raise AssertionError("no long track")


def test_identical_results_compare_clean(oracle_of):
    _, ref = oracle_of(1, 64)
    rep = compare_tracks(ref.tracks, ref.tracks, ref)
    assert rep["mismatched_tracks"] == 0 and rep["bad_fits"] == 0 and rep["n_got"] == rep["n_ref"] > 0
    assert rep["near_cut_decisions"] == int(ref.near_cut_per_event.sum())


def test_a_mismatch_is_near_cut_only_if_a_logged_decision_touches_it(oracle_of):
    _, ref = oracle_of(1, 64)
    e = 5
    got, dropped, hits = _drop_last_hit_of_first_long_track(ref.tracks, e)
    fake = copy.deepcopy(ref)
    # no logged decision in this event: hard failure (two differing hit sets: the shortened and the original track)
    keep = fake.near_cut_hit_event != e
    fake.near_cut_hit_event, fake.near_cut_hit_index = fake.near_cut_hit_event[keep], fake.near_cut_hit_index[keep]
    rep = compare_tracks(got, ref.tracks, fake)
    assert rep["mismatched_tracks"] == 2 and rep["hard_mismatched_tracks"] == 2 and rep["near_cut_mismatched_tracks"] == 0
    # a logged decision on a hit BELOW every differing hit (a later iteration) does not excuse it
    lowest = min(hits)
    if lowest > 0:
        fake.near_cut_hit_event = np.append(fake.near_cut_hit_event, e).astype(np.uint32)
        fake.near_cut_hit_index = np.append(fake.near_cut_hit_index, 0).astype(np.uint32)
        rep = compare_tracks(got, ref.tracks, fake)
        assert rep["hard_mismatched_tracks"] == 2
    # a logged decision on the dropped hit itself does
    fake.near_cut_hit_event = np.append(fake.near_cut_hit_event, e).astype(np.uint32)
    fake.near_cut_hit_index = np.append(fake.near_cut_hit_index, dropped).astype(np.uint32)
    rep = compare_tracks(got, ref.tracks, fake)
    assert rep["near_cut_mismatched_tracks"] == 2 and rep["hard_mismatched_tracks"] == 0
    # and so does one on a hit of an earlier iteration (a higher index than the lowest differing hit)
    fake.near_cut_hit_index[-1] = max(hits) + 1
    rep = compare_tracks(got, ref.tracks, fake)
    assert rep["near_cut_mismatched_tracks"] == 2
    # a decision logged in ANOTHER event never excuses it
    fake.near_cut_hit_event[-1] = e + 1
    rep = compare_tracks(got, ref.tracks, fake)
    assert rep["hard_mismatched_tracks"] == 2
