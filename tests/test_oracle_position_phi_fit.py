"""Pins for oracle steps O3 (centroid -> global, phi16), the scatter helper of O5 and O6 (line fit)."""
import math

import numpy as np
import pytest

import oracle
from paper_1912_09161_b200 import workload

N_COLS = 768
PITCH = 0.055


def run_pixels(geometry, events):
    raw, off = workload.pack_events(geometry, events)
    return oracle.reconstruct(geometry, raw, off)


# ---------------------------------------------------------------- O3: phi16
def test_phi16_within_one_lsb_of_exact_rounding():
    rng = np.random.default_rng(3)
    r = rng.uniform(4.0, 60.0, 20000)
    a = rng.uniform(-math.pi, math.pi, 20000)
    worst = 0
    for x, y in zip((r * np.cos(a)).astype(np.float32), (r * np.sin(a)).astype(np.float32)):
        want = round(math.atan2(float(y), float(x)) * 32768.0 / math.pi)
        d = (oracle.phi16(x, y) - want + 32768) % 65536 - 32768
        worst = max(worst, abs(d))
    assert worst <= 1


def test_atan2_poly_error_bound():
    # Abramowitz & Stegun 4.4.49 quotes |eps| <= 2e-8 for the polynomial on [0,1]; in fp32 with the range
    # reduction used here the total error stays below 1e-6 rad (R3 measured 3.1e-7).
    rng = np.random.default_rng(4)
    xs = rng.normal(size=20000).astype(np.float32) * 30
    ys = rng.normal(size=20000).astype(np.float32) * 30
    err = max(abs(oracle.atan2_poly(x, y) - math.atan2(float(y), float(x))) for x, y in zip(xs, ys))
    assert err < 1e-6


@pytest.mark.parametrize("x,y,want", [
    (1.0, 0.0, 0), (0.0, 1.0, 16384), (-1.0, 0.0, -32768), (0.0, -1.0, -16384),
    (1.0, 1.0, 8192), (-1.0, 1.0, 24576), (-1.0, -1.0, -24576), (1.0, -1.0, -8192),
    (-1.0, -0.0, -32768),  # y = -0: "y < 0" is false, pi scales to +32768 which wraps to -32768
    (0.0, 0.0, 0),  # degenerate: t := 0
    (5.0, 1e-30, 0), (-5.0, -1e-30, -32768),
])
def test_phi16_quadrants_and_axes(x, y, want):
    assert oracle.phi16(np.float32(x), np.float32(y)) == want


def test_phi16_is_odd_in_y_and_monotone_around_the_circle():
    xs = [np.float32(10 * math.cos(a)) for a in np.linspace(-3.1, 3.1, 500)]
    ys = [np.float32(10 * math.sin(a)) for a in np.linspace(-3.1, 3.1, 500)]
    ph = [oracle.phi16(x, y) for x, y in zip(xs, ys)]
    assert all(b >= a for a, b in zip(ph, ph[1:]))
    for x, y in zip(xs, ys):
        if y != 0:
            assert oracle.phi16(x, -y) == -oracle.phi16(x, y)


# ---------------------------------------------------------------- O3: centroid and local -> global
def test_single_pixel_closed_form(geometry):
    # single pixel (c, r) on every sensor of station 0: x = ox + (c+.5)p*ecx + (r+.5)p*erx etc. (G0 frames)
    cases = [(0, 10, 20), (1, 700, 3), (2, 0, 255), (3, 767, 0), (50, 123, 45)]
    res = run_pixels(geometry, [[(s, c, r)] for s, c, r in cases])
    for e, (s, c, r) in enumerate(cases):
        ox, oy, ecx, ecy, erx, ery, z = geometry.sensor_frame[s]
        u, v = (c + 0.5) * PITCH, (r + 0.5) * PITCH
        assert res.clusters.x[e] == pytest.approx(ox + u * ecx + v * erx, abs=2e-5)
        assert res.clusters.y[e] == pytest.approx(oy + u * ecy + v * ery, abs=2e-5)
        assert res.clusters.z[e] == np.float32(z)
        assert (res.clusters.n_pixels[e], res.clusters.sum_col[e], res.clusters.sum_row[e]) == (1, c, r)


def test_centroid_of_multi_pixel_cluster(geometry):
    # 2x1 and 3-pixel L clusters on sensor 0 (col -> +x, row -> +y, origin (-4, 4))
    res = run_pixels(geometry, [[(0, 100, 50), (0, 101, 50)], [(0, 100, 50), (0, 101, 50), (0, 100, 51)]])
    assert res.clusters.x[0] == pytest.approx(-4 + (100.5 + 0.5) * PITCH, abs=2e-5)
    assert res.clusters.y[0] == pytest.approx(4 + 50.5 * PITCH, abs=2e-5)
    assert res.clusters.x[1] == pytest.approx(-4 + (301 / 3 + 0.5) * PITCH, abs=2e-5)
    assert res.clusters.y[1] == pytest.approx(4 + (151 / 3 + 0.5) * PITCH, abs=2e-5)


def test_g0_fourfold_symmetry(geometry):
    # the same local pixel pattern on the four sensors of a station gives positions rotated by 90 degrees
    # (R0 -> R1 -> L0 -> L1 is a rotation by -90 degrees each: (x, y) -> (y, -x)); z differs for the left module.
    pat = [(200, 100), (201, 100), (201, 101)]
    res = run_pixels(geometry, [[(40 + k, c, r) for c, r in pat] for k in range(4)])
    x, y = res.clusters.x.astype(np.float64), res.clusters.y.astype(np.float64)
    for k in range(3):
        assert x[k + 1] == pytest.approx(y[k], abs=2e-5)
        assert y[k + 1] == pytest.approx(-x[k], abs=2e-5)
    d = [(int(res.clusters.phi16[k]) - int(res.clusters.phi16[k + 1])) % 65536 for k in range(3)]
    assert all(abs(v - 16384) <= 1 for v in d)


def test_cluster_position_residual_to_generator_truth(oracle_of):
    # Every cluster made only of one particle's pixels lies within a pixel diagonal (plus the one-pixel
    # charge-sharing shift) of that particle's true crossing point.
    batch, res = oracle_of(1, 40)
    geo = batch.geometry
    px, pt = batch.pixels, batch.particles
    key = (px["sensor"].astype(np.uint32) << 18) | (px["row"].astype(np.uint32) * N_COLS + px["col"])
    owner = {}
    for e, k, p in zip(px["event"], key, px["particle"]):
        owner.setdefault((int(e), int(k)), set()).add(int(p))
    members = {}
    for e, k, c in zip(res.pix_event, res.pix_key, res.pix_cluster):
        members.setdefault((int(e), int(c)), []).append(int(k))
    checked = 0
    for (e, c), keys in members.items():
        owners = set().union(*(owner[(e, k)] for k in keys))
        if len(owners) != 1 or -1 in owners:
            continue
        p = owners.pop()
        g = int(res.clusters.event_offsets[e]) + c
        z = float(res.clusters.z[g])
        if batch.config >= 2:
            continue
        tx, ty = pt["tx"][p], pt["ty"][p]
        xt = pt["ox"][p] + tx * (z - pt["oz"][p])
        yt = pt["oy"][p] + ty * (z - pt["oz"][p])
        d = math.hypot(float(res.clusters.x[g]) - xt, float(res.clusters.y[g]) - yt)
        assert d <= PITCH * math.sqrt(2) / 2 + PITCH * 0.75, (e, c, d)
        checked += 1
    assert checked > 5000


# ---------------------------------------------------------------- O5 helper: scatter
def test_scatter_closed_form():
    # S = squared distance, in the plane z = z_c, between c and the straight line through a and b (fp64 closed form)
    rng = np.random.default_rng(9)
    for _ in range(2000):
        a = np.array([rng.normal() * 20, rng.normal() * 20, 300.0], np.float32)
        b = np.array([a[0] + rng.normal() * 3, a[1] + rng.normal() * 3, 275.0 + 12.5 * rng.integers(0, 2)], np.float32)
        c = np.array([b[0] + rng.normal() * 3, b[1] + rng.normal() * 3, 250.0], np.float32)
        A, B, C = a.astype(np.float64), b.astype(np.float64), c.astype(np.float64)
        t = (C[2] - A[2]) / (B[2] - A[2])
        ext = A[:2] + t * (B[:2] - A[:2])
        want = float(np.sum((ext - C[:2]) ** 2))
        got = oracle.scatter(a, b, c)
        assert got == pytest.approx(want, rel=2e-4, abs=1e-9)
        assert got >= 0.0


def test_scatter_zero_on_exact_line_and_order_of_arguments():
    a, b, c = [0.0, 0.0, 100.0], [1.0, 2.0, 75.0], [2.0, 4.0, 50.0]  # exactly collinear, representable
    assert oracle.scatter(a, b, c) == 0.0
    # moving c by (0.5, 0) gives S = 0.25 exactly
    assert oracle.scatter(a, b, [2.5, 4.0, 50.0]) == 0.25
    # the extrapolation runs from b with the slope of a->b over the lever arm z_c - z_b: with unequal spacing,
    # swapping the roles of a and c changes S (0.5 mm off over a 50 mm arm vs 0.25 mm over a 25 mm arm)
    a2, b2, c2 = [0.0, 0.0, 100.0], [1.0, 0.0, 75.0], [3.5, 0.0, 25.0]
    assert oracle.scatter(a2, b2, c2) == 0.25
    assert oracle.scatter(c2, b2, a2) == pytest.approx(0.0625, rel=1e-6)
    # dz_ab = 0 -> division by zero -> NaN or inf, which no cut accepts
    s = oracle.scatter([0, 0, 10.0], [1.0, 0, 10.0], [2.0, 0, 0.0])
    assert not (s <= 1e30)


# ---------------------------------------------------------------- O6: straight-line fit
def test_fit_recovers_exact_line():
    z = np.array([700.0, 600.0, 450.0, 350.0, 275.0], np.float32)
    x = (0.25 + 0.03125 * z).astype(np.float32)  # exactly representable
    y = (-1.5 - 0.0625 * z).astype(np.float32)
    x0, y0, tx, ty = oracle.fit(x, y, z)
    assert (x0, y0, tx, ty) == (0.25, -1.5, 0.03125, -0.0625)


def test_fit_agrees_with_polyfit_and_normal_equations():
    rng = np.random.default_rng(21)
    for n in (3, 4, 7, 12, 26):
        for _ in range(50):
            z = np.sort(rng.uniform(-290, 750, n)).astype(np.float32)[::-1].copy()
            tx_t, ty_t = rng.uniform(-0.3, 0.3, 2)
            x = (rng.normal() * 0.1 + tx_t * z + rng.normal(size=n) * 0.02).astype(np.float32)
            y = (rng.normal() * 0.1 + ty_t * z + rng.normal(size=n) * 0.02).astype(np.float32)
            got = oracle.fit(x, y, z).astype(np.float64)
            Z, X, Y = z.astype(np.float64), x.astype(np.float64), y.astype(np.float64)
            px, py = np.polyfit(Z, X, 1), np.polyfit(Z, Y, 1)
            assert got[2] == pytest.approx(px[0], rel=1e-6, abs=1e-9) and got[0] == pytest.approx(px[1], rel=1e-6, abs=1e-6)
            assert got[3] == pytest.approx(py[0], rel=1e-6, abs=1e-9) and got[1] == pytest.approx(py[1], rel=1e-6, abs=1e-6)
            # normal equations [n, Sz; Sz, Szz] [x0; tx] = [Sx; Szx]
            M = np.array([[n, Z.sum()], [Z.sum(), (Z * Z).sum()]])
            sol = np.linalg.solve(M, np.array([X.sum(), (Z * X).sum()]))
            assert got[0] == pytest.approx(sol[0], rel=1e-6, abs=1e-6) and got[2] == pytest.approx(sol[1], rel=1e-6, abs=1e-9)


def test_fit_residual_to_generator_truth(oracle_of):
    # config 0: straight noiseless tracks -> fitted slopes agree with the generated ones to pixel resolution
    from tests.helpers import physics_report

    batch, res = oracle_of(0)
    rep = physics_report(batch, res)
    mp = rep["matched_particle"]
    assert (mp >= 0).all()
    tx, ty = batch.particles["tx"][mp], batch.particles["ty"][mp]
    # pixel resolution 0.055/sqrt(12) mm over lever arms of 50 mm (3-hit tracks) .. 1 m
    assert np.max(np.abs(res.tracks.tx - tx)) < 2e-3 and np.median(np.abs(res.tracks.tx - tx)) < 1e-4
    assert np.max(np.abs(res.tracks.ty - ty)) < 2e-3 and np.median(np.abs(res.tracks.ty - ty)) < 1e-4
    x0 = batch.particles["ox"][mp] - tx * batch.particles["oz"][mp]
    assert np.max(np.abs(res.tracks.x0 - x0)) < 1.0 and np.median(np.abs(res.tracks.x0 - x0)) < 0.03
