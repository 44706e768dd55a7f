"""Pins for O7, the simple Kalman fit (R9), against formulations that share nothing with the
recursion: the posterior of the equivalent linear-Gaussian model solved in one go, closed forms and symmetries."""
import numpy as np
import pytest

PITCH = 0.055
VAR_M = PITCH ** 2 / 12


def noise(x, y, z):
    """q_x, q_y of R9 from the first two hits (retyped from the text of R9, not from the oracle)."""
    tx, ty = (x[1] - x[0]) / (z[1] - z[0]), (y[1] - y[0]) / (z[1] - z[0])
    t2 = tx * tx + ty * ty
    th = (13.6 / 400.0) ** 2 * 0.02 * t2 / (1 + t2)
    return th * (1 + tx * tx) * (1 + t2), th * (1 + ty * ty) * (1 + t2)


def posterior_in_one_go(m, z, q):
    """Unknowns u = (pos at hit 0, slope at hit 0, kink after hit 0 .. kink after hit n-2).  Measurement k sees
    pos0 + slope0 (z_k - z_0) + sum_{j<k} kink_j (z_k - z_j), variance VAR_M; prior: slope0 ~ N(0, 1), kinks ~ N(0, q),
    pos0 flat.  Returns mean and covariance of (pos, slope) at the last hit, and the chi2 of the innovations."""
    n = len(m)
    A = np.zeros((n, n + 1))
    A[:, 0] = 1
    A[:, 1] = z - z[0]
    for j in range(n - 1):
        A[j + 1:, 2 + j] = z[j + 1:] - z[j]
    prec = np.diag([0.0, 1.0] + [1.0 / q] * (n - 1))
    cov_u = np.linalg.inv(A.T @ A / VAR_M + prec)
    u = cov_u @ (A.T @ m) / VAR_M
    B = np.zeros((2, n + 1))
    B[0] = A[-1]
    B[1, 1:] = 1
    # innovations: measurements 1.. given hit 0 (pos0 ~ N(m0, VAR_M), slope0 ~ N(0,1), kinks ~ N(0,q))
    P = np.diag([VAR_M, 1.0] + [q] * (n - 1))
    mu = A[1:, 0] * m[0]
    V = A[1:] @ P @ A[1:].T + VAR_M * np.eye(n - 1)
    r = m[1:] - mu
    return B @ u, B @ cov_u @ B.T, float(r @ np.linalg.solve(V, r))


@pytest.fixture(scope="module")
def tracks(oracle_of):
    batch, ref = oracle_of(2, 200)
    t, c = ref.tracks, ref.clusters
    import oracle

    kf = oracle.kalman_of(ref, PITCH)
    ev = np.repeat(np.arange(len(t.event_offsets) - 1), np.diff(t.event_offsets.astype(np.int64)))
    return t, c, ev, kf


def test_equals_the_posterior_of_the_linear_gaussian_model(tracks):
    t, c, ev, kf = tracks
    rng = np.random.default_rng(5)
    for i in rng.choice(len(kf), 300, replace=False):
        h = c.event_offsets[ev[i]].astype(np.int64) + t.hits[t.hit_offsets[i]:t.hit_offsets[i + 1]]
        x, y, z = (a[h].astype(np.float64) for a in (c.x, c.y, c.z))
        qx, qy = noise(x, y, z)
        chi2 = 0
        for pr, (m, q) in enumerate(((x, qx), (y, qy))):
            mean, cov, c2 = posterior_in_one_go(m, z, q)
            chi2 += c2
            assert kf[i, pr] == pytest.approx(mean[0], rel=1e-9, abs=1e-9)
            assert kf[i, 2 + pr] == pytest.approx(mean[1], rel=1e-7, abs=1e-11)
            got = kf[i, 6 + 3 * pr:9 + 3 * pr]
            assert got == pytest.approx([cov[0, 0], cov[0, 1], cov[1, 1]], rel=1e-6)
        assert kf[i, 4] == z[-1]
        assert kf[i, 5] == pytest.approx(chi2, rel=1e-6, abs=1e-9)


def test_exact_line_is_recovered_and_chi2_is_the_prior_term():
    import oracle

    z = np.array([600.0, 450.0, 350.0, 275.0, 250.0], np.float32)
    x = (1.5 + 0.03125 * z).astype(np.float32)   # exactly representable
    y = (-2.0 - 0.0625 * z).astype(np.float32)
    kf = oracle.kalman([0, 5], np.arange(5), x, y, z, PITCH)[0]
    # the prior pulls the slope towards 0 by var/(var + 1) ~ 1e-9 relative: far below the tolerances here
    assert kf[:5] == pytest.approx([1.5 + 0.03125 * 250, -2.0 - 0.0625 * 250, 0.03125, -0.0625, 250.0], rel=1e-7)
    # on a perfect line only the slope prior N(0, 1) contributes to chi2: tx^2 + ty^2 (closed form)
    assert kf[5] == pytest.approx(0.03125 ** 2 + 0.0625 ** 2, rel=1e-5)


def test_projections_are_independent_and_symmetric(tracks):
    import oracle

    t, c, ev, kf = tracks
    i = 7
    h = c.event_offsets[ev[i]].astype(np.int64) + t.hits[t.hit_offsets[i]:t.hit_offsets[i + 1]]
    x, y, z = c.x[h], c.y[h], c.z[h]
    a = oracle.kalman([0, len(h)], np.arange(len(h)), x, y, z, PITCH)[0]
    b = oracle.kalman([0, len(h)], np.arange(len(h)), y, x, z, PITCH)[0]   # swap the projections
    assert np.array_equal(a[[0, 2, 6, 7, 8]], b[[1, 3, 9, 10, 11]]) and a[5] == pytest.approx(b[5], rel=1e-12)
    # moving one x measurement changes the x state only through x; y changes only through the common noise term,
    # which depends on the first two hits: move the last hit
    x2 = x.copy()
    x2[-1] += 0.01
    d = oracle.kalman([0, len(h)], np.arange(len(h)), x2, y, z, PITCH)[0]
    assert np.array_equal(d[[1, 3, 9, 10, 11]], a[[1, 3, 9, 10, 11]]) and d[0] != a[0]
    assert np.array_equal(d[6:9], a[6:9])  # covariances do not depend on the measured values


def test_agrees_with_the_straight_line_fit_within_its_errors(tracks):
    """Physics sanity: slopes of O7 and O6 agree within a few sigma of O7's own covariance."""
    t, c, ev, kf = tracks
    pull = (kf[:, 2] - t.tx) / np.sqrt(kf[:, 8])
    assert np.abs(np.median(pull)) < 0.2 and np.percentile(np.abs(pull), 99) < 6
