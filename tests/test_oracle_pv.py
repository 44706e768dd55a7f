"""Pins for O8, primary-vertex finding (R10): hand-made histograms with closed-form seeds, tracks
from an exact point, the fixed point of the weighted fit solved with numpy's least squares, and generator truth."""
import numpy as np
import pytest

PITCH = 0.055


def toy_tracks(points, n_per, rng, sigma=0.0, z_state=50.0):
    """Straight tracks through the given points; returns the O6 parameters and O7-like states with a fixed covariance."""
    x0, y0, tx, ty, kal = [], [], [], [], []
    for (px, py, pz), n in zip(points, n_per):
        for _ in range(n):
            th, ph = rng.uniform(0.02, 0.25), rng.uniform(0, 2 * np.pi)
            sx, sy = np.tan(th) * np.cos(ph), np.tan(th) * np.sin(ph)
            ox, oy = rng.normal(0, sigma, 2) if sigma else (0.0, 0.0)
            x0.append(px + ox - sx * pz); y0.append(py + oy - sy * pz); tx.append(sx); ty.append(sy)
            zs = pz + z_state
            kal.append([px + ox + sx * z_state, py + oy + sy * z_state, sx, sy, zs, 0.0,
                        4e-4, 0.0, 1e-8, 4e-4, 0.0, 1e-8])
    f = lambda a: np.array(a, np.float32)
    return f(x0), f(y0), f(tx), f(ty), np.array(kal, np.float64)


def run(x0, y0, tx, ty, kal):
    import oracle

    v, c, cand = oracle.find_pvs([0, len(x0)], x0, y0, tx, ty, kal)
    return v[0, :c[0]], int(cand[0])


def test_tracks_from_exact_points_give_those_points():
    rng = np.random.default_rng(1)
    pts = [(0.03, -0.02, -35.25), (-0.05, 0.01, 12.5), (0.0, 0.04, 80.75)]
    v, cand = run(*toy_tracks(pts, [12, 7, 20], rng))
    assert cand == 3 and len(v) == 3
    for got, (px, py, pz), n in zip(v, pts, [12, 7, 20]):
        assert got[:3] == pytest.approx([px, py, pz], abs=2e-4)   # fp32 track parameters in, fp64 fit
        assert got[3] == pytest.approx(n, rel=1e-4) and got[4] == n and got[5] < 1e-3


def poca_tracks(zps):
    """Tracks whose z of closest approach to the beam line is exactly zp (they cross the beam line there)."""
    n = len(zps)
    phi = 2.4 * np.arange(n) + 0.3                      # different directions: the vertex fit is well conditioned
    tx, ty = (0.0625 * np.cos(phi)).astype(np.float32), (0.0625 * np.sin(phi)).astype(np.float32)
    zps = np.asarray(zps, np.float64)
    x0, y0 = (-tx * zps).astype(np.float32), (-ty * zps).astype(np.float32)
    kal = np.zeros((n, 12))
    kal[:, 2], kal[:, 3], kal[:, 4] = tx, ty, zps
    kal[:, 6], kal[:, 9], kal[:, 8], kal[:, 11] = 4e-4, 4e-4, 1e-8, 1e-8
    return x0, y0, tx, ty, kal


def test_histogram_seeds_closed_forms():
    # five tracks in one bin: one candidate at the bin centre
    v, cand = run(*poca_tracks([10.25] * 5))
    assert cand == 1 and v[0, 6] == pytest.approx(10.5)
    # 3 + 3 in adjacent bins: one candidate (tie rule), seed exactly between the bin centres
    v, cand = run(*poca_tracks([10.25] * 3 + [11.25] * 3))
    assert cand == 1 and v[0, 6] == pytest.approx(11.0)
    # 3 tracks only: below the threshold of 4; 4 spread 2+0+2 over three bins: one candidate in the middle
    assert run(*poca_tracks([10.25] * 3))[1] == 0
    v, cand = run(*poca_tracks([10.25, 10.5, 12.25, 12.5]))
    assert cand == 1 and len(v) == 0   # a candidate, but tracks 2 mm apart along z do not make a vertex (sum w < 3)
    # two well separated groups: two candidates; range limits: outside [-300, 300) ignored
    assert run(*poca_tracks([-100.5] * 4 + [100.5] * 6))[1] == 2
    assert run(*poca_tracks([-300.5] * 6 + [300.5] * 6 + [299.5] * 4))[1] == 1
    # asymmetric neighbours pull the seed: h = 2, 4, 0 -> centre - 2/6
    v, cand = run(*poca_tracks([9.5] * 2 + [10.5] * 4))
    assert cand == 1 and v[0, 6] == pytest.approx(10.5 - 2 / 6)


def test_one_more_iteration_is_the_weighted_least_squares_step(oracle_of):
    """The vertex after n+1 passes equals numpy's lstsq over the stacked residual equations (x and y of every track,
    unknowns vx, vy, vz) weighted with the Tukey weights at the vertex after n passes: pins weights, normal equations
    and their solution without assuming convergence.  The sums reported after n passes are checked on the way."""
    import oracle

    batch, ref = oracle_of(2, 200)
    kal = oracle.kalman_of(ref, PITCH)
    t = ref.tracks
    args = (t.event_offsets, t.x0, t.y0, t.tx, t.ty, kal)
    checked = 0
    for n_it in (1, 3, 8):
        v, c, cand = oracle.find_pvs(*args, iterations=n_it)
        v1, c1, cand1 = oracle.find_pvs(*args, iterations=n_it + 1)
        assert np.array_equal(cand, cand1)
        for e in range(0, 200, 7):
            k = kal[t.event_offsets[e]:t.event_offsets[e + 1]]
            nxt = {round(r[6], 9): r for r in v1[e, :c1[e]]}   # match by seed
            for vx, vy, vz, sw, nw, chi2, seed, _ in v[e, :c[e]]:
                d = vz - k[:, 4]
                px, py = k[:, 0] + k[:, 2] * d, k[:, 1] + k[:, 3] * d
                var_x = k[:, 6] + 2 * d * k[:, 7] + d * d * k[:, 8]
                var_y = k[:, 9] + 2 * d * k[:, 10] + d * d * k[:, 11]
                c2 = (px - vx) ** 2 / var_x + (py - vy) ** 2 / var_y
                w = np.where(c2 < 12, (1 - c2 / 12) ** 2, 0.0)
                assert w.sum() == pytest.approx(sw, rel=1e-6) and (w > 0).sum() == nw
                assert (w * c2).sum() == pytest.approx(chi2, rel=1e-6, abs=1e-9)
                if round(seed, 9) not in nxt:
                    continue  # dropped after the extra pass (sum w fell below 3, or a duplicate)
                sx, sy = np.sqrt(w / var_x), np.sqrt(w / var_y)
                A = np.vstack([np.c_[-sx, 0 * sx, sx * k[:, 2]], np.c_[0 * sy, -sy, sy * k[:, 3]]])
                rhs = np.r_[-sx * (px - k[:, 2] * vz), -sy * (py - k[:, 3] * vz)]
                sol = np.linalg.lstsq(A, rhs, rcond=None)[0]
                assert sol == pytest.approx(nxt[round(seed, 9)][:3], abs=1e-7)
                checked += 1
    assert checked > 150


def test_finds_the_generated_collisions(batch_of):
    import oracle

    batch = batch_of(1, 300)
    ref = oracle.reconstruct(batch.geometry, batch.raw, batch.event_offsets, n_threads=8)
    v, c, _ = oracle.pvs_of(ref, PITCH)
    pv, part = batch.pvs, batch.particles
    n_part = np.zeros(len(pv["z"]), int)
    first = np.searchsorted(pv["event"], np.arange(batch.n_events))
    np.add.at(n_part, first[part["event"]] + part["pv"], 1)
    n_good = n_found = n_reco = n_fake = 0
    for e in range(batch.n_events):
        m = pv["event"] == e
        zt, nt = pv["z"][m], n_part[m]
        zf = v[e, :c[e], 2]
        n_reco += len(zf)
        n_fake += sum(1 for z in zf if not len(zt) or np.min(np.abs(zt - z)) > 1.0)
        for i, z in enumerate(zt):
            others = np.delete(zt, i)
            if nt[i] >= 15 and (not len(others) or np.min(np.abs(others - z)) > 5.0):
                n_good += 1
                n_found += bool(len(zf)) and np.min(np.abs(zf - z)) < 0.5
    assert n_good > 500
    assert n_found / n_good > 0.97, (n_found, n_good)
    assert n_fake / n_reco < 0.03, (n_fake, n_reco)
    # resolution in x, y: found vertices sit on the beam line within the generated spread and the fit error
    assert np.abs(v[..., 0][v[..., 3] > 0]).max() < 0.5


# ------------------------------------------------------------------------------------------------
# Step 4 of R10 (acceptance and duplicate removal).  Hand-made events; every expectation below follows from the
# written rule ("accepted iff sum w >= 3; dropped if another accepted vertex lies within 1 mm in z with a sum w more
# than 0.1 % larger; within 0.1 % the earlier candidate wins"), not from running the oracle.
# ------------------------------------------------------------------------------------------------
def one_vertex_seen_from_two_peaks(sign=1.0, var=4e-3):
    """Ten tracks of slope 0.02 from the point (0, 0, 0), shifted sideways along their own slope direction by
    +-0.021 mm: their points of closest approach to the beam line fall at z = -+1.05 mm, i.e. into the histogram bins
    [-2, -1) and [1, 2) with two empty bins between them -> two candidates (seeds -1.5 and +1.5).  With a position
    variance of 4e-3 mm^2 every track is compatible with one vertex at z ~ 0 (chi2_t ~ 0.1), so both fits converge to it.
    `sign` mirrors the event in z (the physical groups swap roles)."""
    n = 10
    phi = 2.4 * np.arange(n) + 0.3
    tx, ty = 0.02 * np.cos(phi), 0.02 * np.sin(phi)
    shift = np.where(np.arange(n) % 2 == 0, 0.021, -0.021) * sign
    ox, oy = shift * np.cos(phi), shift * np.sin(phi)   # along the slope direction: moves the POCA by -shift / 0.02 in z
    f = lambda a: np.asarray(a, np.float32)
    x0, y0, tx, ty = f(ox), f(oy), f(tx), f(ty)
    kal = np.zeros((n, 12))
    zs = 64.0
    kal[:, 0], kal[:, 1] = x0.astype(np.float64) + tx.astype(np.float64) * zs, y0.astype(np.float64) + ty.astype(np.float64) * zs
    kal[:, 2], kal[:, 3], kal[:, 4] = tx, ty, zs
    kal[:, 6], kal[:, 9], kal[:, 8], kal[:, 11] = var, var, 1e-10, 1e-10
    return x0, y0, tx, ty, kal


@pytest.mark.parametrize("sign", [1.0, -1.0])
def test_two_peaks_that_converge_to_one_vertex_leave_the_earlier_candidate(sign):
    import oracle

    v, cand = oracle.pv_candidates(*one_vertex_seen_from_two_peaks(sign))
    assert len(cand) == 2 and cand[:, 0].tolist() == [-1.5, 1.5]          # closed-form seeds, in histogram order
    assert np.all(cand[:, 5] == 1) and np.abs(cand[0, 3] - cand[1, 3]) < 1e-3   # both converged, to the same z
    # the two fits describe the same vertex: their sum w agree to rounding / residual-convergence level, far inside
    # the 0.1 % band ...
    assert abs(cand[0, 4] - cand[1, 4]) < 1e-4 * cand[0, 4]
    # ... so exactly one survives, and it is the EARLIER candidate whichever physical group it came from (the event and
    # its mirror image keep the seed -1.5): the survivor is not decided by the last bits of sum w
    assert len(v) == 1 and v[0, 6] == -1.5
    assert v[0, 3] == cand[0, 4] and v[0, 2] == cand[0, 3]


def test_exact_comparison_of_sum_w_would_be_decided_by_rounding():
    """Why the band exists (fp64 behaviour alone, no GPU involved): the two candidates that converged to one vertex have
    sums of weights that differ by at most a few units in the last place, and the sign of that difference changes
    between an event and its mirror image and with the track covariance: an exact "larger sum w wins" rule would
    let the last bit of an 8-pass iteration pick the surviving seed."""
    import oracle

    signs = set()
    for var in (4e-3, 5e-3, 6e-3, 8e-3):
        for sign in (1.0, -1.0):
            _, cand = oracle.pv_candidates(*one_vertex_seen_from_two_peaks(sign, var))
            assert len(cand) == 2 and abs(cand[0, 4] - cand[1, 4]) <= 8 * np.spacing(cand[0, 4])
            signs.add(float(np.sign(cand[0, 4] - cand[1, 4])))
    assert len(signs) >= 2, signs


@pytest.mark.parametrize("n_first,n_second,survivor", [(12, 7, 0), (5, 14, 1)])
def test_duplicate_rule_on_hand_made_candidates(n_first, n_second, survivor):
    """Two accepted candidates whose fitted z differ by 1.1 mm (both stay) or 0.9 mm (only the one with the larger sum of
    weights stays, whether it is the earlier or the later candidate).  Construction: the straight-line parameters (which
    only feed the histogram) put the groups into bins 3 mm apart, so they are seeded separately; the Kalman states (which
    only feed the fit) let the first group cross the beam line at z = 10.5 and the second at 10.5 + dz with slopes of 0.2.
    The second group has a large slope variance, so it is compatible with its candidate's seed 1.9 mm away and the fit
    walks to the crossing point, where its position variance is 4e-4 mm^2 again and the first group (0.2 mm away
    sideways, chi2_t ~ 100) has weight 0: candidate 2 ends exactly at 10.5 + dz with sum w = n_second.  Candidate 1 sits
    at ~10.5 and also collects part of the second group's weight.  The preconditions of the rule (distance, sums) are
    asserted on the candidates before step 4; the expectation is the written rule."""
    import oracle

    for dz, both in ((1.1, True), (0.9, False)):
        n = n_first + n_second
        phi = 2.4 * np.arange(n) + 0.3
        tx, ty = (0.2 * np.cos(phi)).astype(np.float32), (0.2 * np.sin(phi)).astype(np.float32)
        first = np.arange(n) < n_first
        zp = np.where(first, 10.5, 13.5)                      # POCA z of the straight-line parameters (histogram)
        x0, y0 = (-tx * zp).astype(np.float32), (-ty * zp).astype(np.float32)
        kal = np.zeros((n, 12))
        kal[:, 2], kal[:, 3], kal[:, 4] = tx, ty, np.where(first, 10.5, 10.5 + dz)   # states on the beam line (fit)
        kal[:, 6], kal[:, 9] = 4e-4, 4e-4
        kal[:, 8] = kal[:, 11] = np.where(first, 1e-10, 1e-2)
        v, cand = oracle.pv_candidates(x0, y0, tx, ty, kal)
        assert len(cand) == 2 and cand[:, 0].tolist() == [10.5, 13.5] and np.all(cand[:, 5] == 1)
        assert cand[1, 3] == pytest.approx(10.5 + dz, abs=1e-9) and cand[1, 4] == pytest.approx(n_second, rel=1e-9)
        assert abs(cand[0, 3] - 10.5) < 0.09 and cand[0, 4] > n_first
        gap = abs(cand[1, 3] - cand[0, 3])
        larger = int(cand[1, 4] > cand[0, 4])
        assert larger == survivor and max(cand[:, 4]) > 1.001 * min(cand[:, 4])   # clearly outside the tie band
        if both:
            assert gap > 1.0 and len(v) == 2 and v[:, 6].tolist() == [10.5, 13.5]
        else:
            assert gap < 1.0 and len(v) == 1 and v[0, 6] == cand[survivor, 0] and v[0, 3] == cand[survivor, 4]


def test_acceptance_threshold_of_three_is_inclusive():
    """Three tracks exactly through (0, 0, 0) (state at z = 64, exactly representable products) give chi2_t = 0, w = 1 and
    sum w = 3.0 after the fit has reached the point; a fourth track whose POCA is in the same bin but which passes 5 mm
    from the beam line has weight 0 (it only lifts the histogram to the candidate threshold of 4).  sum w = 3 is
    accepted; the same event with one of the three tracks 0.03 mm off (w < 1, sum w < 3) is not."""
    import oracle

    def event(offset):
        phi = np.array([0.3, 2.7, 5.1, 1.0])
        t = np.array([0.125, 0.125, 0.125, 0.125])
        tx, ty = (t * np.cos(phi)).astype(np.float32), (t * np.sin(phi)).astype(np.float32)
        x0, y0 = np.zeros(4, np.float32), np.zeros(4, np.float32)
        # track 3: displaced by 5 mm perpendicular to its slope -> POCA z = 0 (same bin), far from the beam line
        x0[3], y0[3] = -5.0 * np.sin(phi[3]), 5.0 * np.cos(phi[3])
        x0[0], y0[0] = -offset * np.sin(phi[0]), offset * np.cos(phi[0])
        kal = np.zeros((4, 12))
        zs = 64.0
        kal[:, 0] = x0.astype(np.float64) + tx.astype(np.float64) * zs
        kal[:, 1] = y0.astype(np.float64) + ty.astype(np.float64) * zs
        kal[:, 2], kal[:, 3], kal[:, 4] = tx, ty, zs
        kal[:, 6], kal[:, 9] = 4e-4, 4e-4
        return x0, y0, tx, ty, kal

    v, cand = oracle.pv_candidates(*event(0.0))
    assert len(cand) == 1 and cand[0, 0] == 0.5
    assert cand[0, 4] == 3.0 and cand[0, 5] == 1 and len(v) == 1 and v[0, 4] == 3
    v, cand = oracle.pv_candidates(*event(0.03))
    assert len(cand) == 1 and 2.5 < cand[0, 4] < 3.0 and cand[0, 5] == 0 and len(v) == 0
