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
