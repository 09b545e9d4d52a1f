"""Pins of the oracle's geometry and Kalman arithmetic (R0, R5) against closed forms.

Nothing here re-types the oracle's formulas: the references are the analytic circle/helix in
double (asin / cos), central finite differences of that analytic map, the closed-form
Bayesian straight-line fit, and the statistical unit-width of the pulls.
"""
import math

import numpy as np
import pytest

import oracle
from paper_2601_20569_b200 import datagen as dg

CB = 0.00299792458 * 0.5  # (GeV/c)/cm at 0.5 T


def test_geometry_closed_forms():
    # BASELINE.json config 1: radii 85-245 cm linear over 152 rows; PAPER.md:25 trapezoidal
    # sectors of 20 degrees; R[cm] = pT / (0.3 B).
    x, ymax, dx, cfield = oracle.geom_tables()
    assert x[0] == np.float32(85.0) and x[151] == np.float32(245.0)
    assert abs(dx - 160.0 / 151.0) < 1e-7
    assert np.allclose(np.diff(x.astype(np.float64)), 160.0 / 151.0, atol=2e-5)
    assert np.allclose(ymax, x.astype(np.float64) * math.tan(math.radians(10.0)), rtol=1e-6)
    assert abs(ymax[0] - 14.9878) < 1e-3 and abs(ymax[151] - 43.2001) < 1e-3
    # curvature per q/pT: radius of a 1 GeV/c track at 0.5 T is 667.128 cm, and a positive
    # charge bends towards -y (negative curvature) when moving along +x with B along +z
    assert abs(1.0 / abs(cfield) - 667.128) < 0.01
    assert cfield < 0


def exact_helix(y, z, s, t, q, dx, cfield):
    """Analytic propagation on the circle (double): sin(phi) is linear in x."""
    k = cfield * q
    s1 = s + k * dx
    c0, c1 = math.sqrt(1 - s * s), math.sqrt(1 - s1 * s1)
    if abs(k) < 1e-14:
        dy = dx * s / c0
        arc = dx / c0
    else:
        dy = (c0 - c1) / k
        arc = (math.asin(s1) - math.asin(s)) / k
    return y + dy, z + t * arc, s1


@pytest.mark.parametrize("pt,charge,s0,tanl", [(0.15, 1, 0.1, 0.8), (0.3, -1, -0.2, -1.0),
                                                (1.0, 1, 0.3, 0.5), (5.0, -1, 0.0, 0.2),
                                                (0.12, -1, 0.05, 1.02)])
def test_propagation_state_follows_exact_helix(pt, charge, s0, tanl):
    """fp32 propagation row by row over the whole TPC vs the analytic helix in double."""
    x, _, dx, cfield = oracle.geom_tables()
    q = charge / pt
    st = np.zeros(20, dtype=np.float32)
    st[:5] = [1.0, 7000.0 if pt > 0.2 else -3.0, s0, tanl, q]
    y_e, z_e, s_e = float(st[0]), float(st[1]), float(st[2])
    n_steps = 0
    for r in range(1, 152):
        ok, st, _ = oracle.propagate(st, dx, cfield)
        s_next = s_e + cfield * q * float(dx)
        if abs(s_next) > 0.95:
            assert not ok
            break
        assert ok
        y_e, z_e, s_e = exact_helix(y_e, z_e, s_e, tanl, q, float(dx), float(cfield))
        n_steps += 1
        assert abs(float(st[0]) - y_e) < 1e-3
        # z carries an offset of up to 7000 cm: fp32 ulp there is 4.9e-4
        assert abs(float(st[1]) - z_e) < 1e-3 + 152 * 2.5e-4 * (abs(z_e) > 1000)
        assert abs(float(st[2]) - s_e) < 2e-6 * (r + 1)
    assert n_steps > 20
    # and back again (inward steps, signed chord): returns to the start
    for _ in range(n_steps):
        ok, st, _ = oracle.propagate(st, -dx, cfield)
        assert ok
    assert abs(float(st[0]) - 1.0) < 2e-3
    assert abs(float(st[2]) - s0) < 1e-4


def test_propagation_double_matches_exact_helix_tightly():
    """Same statements in double: the asin series is exact to < 1e-11 at one-row steps."""
    _, _, dx, cfield = oracle.geom_tables()
    rng = np.random.default_rng(7)
    for _ in range(200):
        s0 = rng.uniform(-0.8, 0.8)
        q = rng.uniform(-8, 8)
        t = rng.uniform(-1.1, 1.1)
        sign = rng.choice([-1.0, 1.0])
        if abs(s0 + cfield * q * dx * sign) > 0.9:
            continue
        st = np.zeros(20)
        st[:5] = [0.3, -2.0, s0, t, q]
        ok, st1, _ = oracle.propagate(st, sign * dx, float(cfield))
        assert ok
        y_e, z_e, s_e = exact_helix(0.3, -2.0, s0, t, q, sign * dx, float(cfield))
        assert abs(st1[0] - y_e) < 1e-11
        assert abs(st1[1] - z_e) < 1e-10
        assert abs(st1[2] - s_e) < 1e-14


def test_jacobian_matches_finite_differences():
    """F of the oracle vs central finite differences of the ANALYTIC map (double)."""
    _, _, dx, cfield = oracle.geom_tables()
    cfield = float(cfield)
    rng = np.random.default_rng(11)

    def amap(v, d):
        y, z, s1 = exact_helix(v[0], v[1], v[2], v[3], v[4], d, cfield)
        return np.array([y, z, s1, v[3], v[4]])

    for _ in range(100):
        v = np.array([rng.uniform(-5, 5), rng.uniform(-100, 100), rng.uniform(-0.7, 0.7),
                      rng.uniform(-1, 1), rng.uniform(-6, 6)])
        d = float(dx) * rng.choice([-1.0, 1.0])
        st = np.zeros(20)
        st[:5] = v
        ok, _, jac = oracle.propagate(st, d, cfield)
        assert ok
        F = np.eye(5)
        for j in range(5):
            h = 1e-6 * max(1.0, abs(v[j]))
            e = np.zeros(5)
            e[j] = h
            F[:, j] = (amap(v + e, d) - amap(v - e, d)) / (2 * h)
        f02, f04, f12, f13, f14, f24 = jac
        assert abs(f02 - F[0, 2]) < 1e-5 * max(1, abs(F[0, 2]))
        assert abs(f04 - F[0, 4]) < 1e-5
        assert abs(f12 - F[1, 2]) < 1e-5 * max(1, abs(F[1, 2]))
        assert abs(f13 - F[1, 3]) < 1e-6
        assert abs(f24 - F[2, 4]) < 1e-9
        # F14 is the documented small-step approximation: within 2 % (or 2e-6 absolute)
        assert abs(f14 - F[1, 4]) < 0.02 * abs(F[1, 4]) + 2e-6
        # entries the oracle treats as exactly 0 / 1
        for (i, j) in [(0, 1), (0, 3), (1, 0), (2, 0), (2, 1), (2, 3), (3, 4), (4, 0)]:
            assert abs(F[i, j]) < 1e-8
        assert abs(F[0, 0] - 1) < 1e-9 and abs(F[1, 1] - 1) < 1e-9 and abs(F[2, 2] - 1) < 1e-9


def test_covariance_transport_is_F_C_Ft():
    """C' produced by the oracle equals F C F^T built from its own Jacobian entries with a
    dense numpy product (catches index slips in the packed lower-triangular code)."""
    _, _, dx, cfield = oracle.geom_tables()
    rng = np.random.default_rng(3)
    tri = [(i, j) for i in range(5) for j in range(i + 1)]
    for _ in range(50):
        A = rng.normal(size=(5, 5))
        Cm = A @ A.T + 0.1 * np.eye(5)
        st = np.zeros(20)
        st[:5] = [0.5, 3.0, rng.uniform(-0.6, 0.6), rng.uniform(-1, 1), rng.uniform(-5, 5)]
        st[5:] = [Cm[i, j] for (i, j) in tri]
        ok, st1, jac = oracle.propagate(st, float(dx), float(cfield))
        assert ok
        F = np.eye(5)
        F[0, 2], F[0, 4], F[1, 2], F[1, 3], F[1, 4], F[2, 4] = jac
        C1 = F @ Cm @ F.T
        got = np.array(st1[5:])
        want = np.array([C1[i, j] for (i, j) in tri])
        assert np.allclose(got, want, rtol=1e-11, atol=1e-12)


def test_update_is_the_textbook_kalman_update():
    """Update vs dense numpy K = C H^T (H C H^T + V)^-1 in double."""
    rng = np.random.default_rng(5)
    tri = [(i, j) for i in range(5) for j in range(i + 1)]
    H = np.zeros((2, 5))
    H[0, 0] = H[1, 1] = 1
    for _ in range(50):
        A = rng.normal(size=(5, 5)) * 0.1
        Cm = A @ A.T + 0.01 * np.eye(5)
        p = np.array([0.2, -1.0, 0.1, 0.4, 1.5])
        st = np.concatenate([p, [Cm[i, j] for (i, j) in tri]])
        m = p[:2] + rng.normal(size=2) * 0.1
        V = np.diag([0.01, 0.04])
        chi2, stop, st1 = oracle.update(st, m[0], m[1], V[0, 0], V[1, 1], 0.95, 20.0)
        S = H @ Cm @ H.T + V
        K = Cm @ H.T @ np.linalg.inv(S)
        r = m - H @ p
        p1 = p + K @ r
        C1 = Cm - K @ H @ Cm
        assert not stop
        assert abs(chi2 - r @ np.linalg.inv(S) @ r) < 1e-10
        assert np.allclose(st1[:5], p1, atol=1e-12)
        assert np.allclose(st1[5:], [C1[i, j] for (i, j) in tri], atol=1e-13)


def test_filter_equals_weighted_least_squares_straight_line():
    """kappa = 0, hits exactly on y = 0: the (z, tan lambda) filter over n rows equals the
    closed-form Bayesian straight-line fit z = a + t*(x - x0) with prior var(a) = sigma^2 from
    the first hit and var(t) = init_var_tanl."""
    _, _, dx, _ = oracle.geom_tables()
    dx = float(dx)
    rng = np.random.default_rng(9)
    n, sig, var_t = 30, 0.1, 4.0
    zt = 5.0 + 0.7 * dx * np.arange(n) + rng.normal(size=n) * sig
    st = np.zeros(20)
    st[:5] = [0.0, zt[0], 0.0, 0.0, 0.0]
    st[5 + 0], st[5 + 2], st[5 + 5], st[5 + 9], st[5 + 14] = sig ** 2, sig ** 2, 0.25, var_t, 100.0
    for i in range(1, n):
        ok, st, _ = oracle.propagate(st, dx, 0.0)
        assert ok
        _, stop, st = oracle.update(st, 0.0, zt[i], sig ** 2, sig ** 2, 0.95, 20.0)
        assert not stop
    # closed form at the LAST row: parameters (z_last, t); z_i = z_last - t*(n-1-i)*dx
    A = np.stack([np.ones(n), -(n - 1 - np.arange(n)) * dx], axis=1)
    # first hit enters as a measurement too (prior on a = first hit with variance sig^2)
    prec = A.T @ A / sig ** 2 + np.diag([0.0, 0.0])
    # the prior on t (variance var_t around 0)
    prec[1, 1] += 1.0 / var_t
    rhs = A.T @ zt / sig ** 2
    cov = np.linalg.inv(prec)
    sol = cov @ rhs
    assert abs(st[1] - sol[0]) < 1e-9 and abs(st[3] - sol[1]) < 1e-9
    assert abs(st[5 + 2] - cov[0, 0]) < 1e-12      # C11
    assert abs(st[5 + 9] - cov[1, 1]) < 1e-12      # C33
    assert abs(st[5 + 7] - cov[1, 0]) < 1e-12      # C31
    assert abs(st[0]) < 1e-15 and abs(st[2]) < 1e-15


def _true_state_at(x, phi_loc, pt, charge, tanl):
    """Analytic state (y, z, sin phi, tan lambda, q/pT) of a track from the origin at local x
    (first outgoing leg), for the pulls."""
    R = pt / CB
    sphi = math.sin(phi_loc) - charge * x / R
    cphi = math.sqrt(1 - sphi * sphi)
    y = charge * R * (cphi - math.cos(phi_loc))
    psi = charge * (phi_loc - math.asin(sphi))
    return np.array([y, tanl * R * psi, sphi, tanl, charge / pt])


def test_kalman_fit_pulls_have_unit_width():
    """>= 5000 generated tracks, truth cluster association, err = smearing: pulls of all five
    parameters at the innermost hit have |mean| <= 0.06 and width in [0.95, 1.10]
    (north star: "Kalman fit recovering the generating parameters with pulls of unit width")."""
    cfg = dg.preset("C1", tracks_per_event=12000, noise_frac=0.0, seed=77, pt_lo=0.3, p_hit=0.9)
    clusters, labels, truth = dg.generate(cfg)
    x_rows, _, _, _ = oracle.geom_tables()
    alpha = math.radians(10.0)  # centre azimuth of sector 0
    order = np.argsort(labels, kind="stable")
    lab_s = labels[order]
    starts = np.flatnonzero(np.r_[True, lab_s[1:] != lab_s[:-1]])
    ends = np.r_[starts[1:], len(lab_s)]
    pulls = []
    for a, b in zip(starts, ends):
        lab = lab_s[a]
        if lab < 0 or lab % 8 != 0 or b - a < 50:
            continue
        idx = order[a:b]
        rows = clusters["row"][idx].astype(np.int32)
        o = np.argsort(rows, kind="stable")
        rows, idx = rows[o], idx[o]
        if len(np.unique(rows)) != len(rows):
            continue
        k = 0
        while k + 1 < len(rows) and rows[k + 1] != rows[k] + 1:
            k += 1
        rows, idx = rows[k:], idx[k:]
        if len(rows) < 50:
            continue
        fit = oracle.fit_hits(rows, clusters["y"][idx], clusters["z"][idx])
        if fit is None:
            continue
        chi2, x, p, c, n_hits, row_first = fit
        if n_hits < 50 or row_first != rows[0]:
            continue
        tr = truth[lab // 8]
        want = _true_state_at(float(x_rows[row_first]), float(tr["phi0"]) - alpha, float(tr["pt"]),
                              int(tr["charge"]), float(tr["tanl"]))
        diag = np.array([c[0], c[2], c[5], c[9], c[14]], dtype=np.float64)
        pulls.append((p.astype(np.float64) - want) / np.sqrt(diag))
    pulls = np.array(pulls)
    assert len(pulls) >= 5000, len(pulls)
    mean, width = pulls.mean(axis=0), pulls.std(axis=0)
    # y, sin(phi), q/pT: |mean| <= 0.06.  z and tan(lambda): the single-sector sample has
    # tan(lambda) > 0 only, which exposes the extended-Kalman second-order bias (+0.08 sigma on
    # tan(lambda), growing with tan(lambda); it vanishes with zero smearing, see the next test)
    # instead of averaging it away -> bound 0.10 (R5 note).
    assert np.all(np.abs(mean[[0, 2, 4]]) <= 0.06), mean
    assert np.all(np.abs(mean[[1, 3]]) <= 0.10), mean
    assert np.all((width >= 0.95) & (width <= 1.10)), width


def test_noise_free_fit_recovers_generating_parameters():
    """Zero smearing: the fit returns the generating helix (closed form) at the innermost hit
    to fp32 accuracy — the track model has no systematic error."""
    cfg = dg.preset("C1", tracks_per_event=600, noise_frac=0.0, seed=78, pt_lo=0.3, p_hit=0.9,
                    smear_y=0.0, smear_z=0.0)
    clusters, labels, truth = dg.generate(cfg)
    x_rows, _, _, _ = oracle.geom_tables()
    alpha = math.radians(10.0)
    n_checked = 0
    for lab in np.unique(labels):
        if lab < 0 or lab % 8 != 0:
            continue
        idx = np.flatnonzero(labels == lab)
        rows = clusters["row"][idx].astype(np.int32)
        o = np.argsort(rows, kind="stable")
        rows, idx = rows[o], idx[o]
        if len(rows) < 50 or len(np.unique(rows)) != len(rows) or rows[1] != rows[0] + 1:
            continue
        fit = oracle.fit_hits(rows, clusters["y"][idx], clusters["z"][idx])
        assert fit is not None
        chi2, x, p, c, n_hits, row_first = fit
        assert n_hits == len(rows) and row_first == rows[0]
        tr = truth[lab // 8]
        want = _true_state_at(float(x_rows[row_first]), float(tr["phi0"]) - alpha, float(tr["pt"]),
                              int(tr["charge"]), float(tr["tanl"]))
        assert abs(p[0] - want[0]) < 1e-4 and abs(p[1] - want[1]) < 5e-4
        assert abs(p[2] - want[2]) < 5e-6 and abs(p[3] - want[3]) < 1e-5
        assert abs(p[4] - want[4]) < 1e-4
        assert chi2 < 1e-3
        n_checked += 1
    assert n_checked > 100


# ------------------------------------------------------------------ R8 sector-track refit
def _track_hit_lists(cfg, min_hits, keep_holes):
    clusters, labels, truth = dg.generate(cfg)
    order = np.argsort(labels, kind="stable")
    lab_s = labels[order]
    starts = np.flatnonzero(np.r_[True, lab_s[1:] != lab_s[:-1]])
    ends = np.r_[starts[1:], len(lab_s)]
    for a, b in zip(starts, ends):
        lab = lab_s[a]
        if lab < 0 or lab % 8 != 0 or b - a < min_hits:
            continue
        idx = order[a:b]
        rows = clusters["row"][idx].astype(np.int32)
        o = np.argsort(rows, kind="stable")
        rows, idx = rows[o], idx[o]
        if len(np.unique(rows)) != len(rows):
            continue
        if not keep_holes and not (np.diff(rows) == 1).all():
            continue
        yield rows, clusters["y"][idx], clusters["z"][idx], truth[lab // 8]


def test_refit_equals_the_follower_fit_on_hole_free_lists():
    """On a cluster list without holes the refit (R8) performs the statements of the follower's
    chain fit, turn and inward refit (R5.1, R5.2, R5.4, R5.5), which are pinned above: same bits."""
    cfg = dg.preset("C1", tracks_per_event=400, noise_frac=0.0, seed=5, pt_lo=0.4, p_hit=1.0)
    n = 0
    for rows, y, z, _ in _track_hit_lists(cfg, 30, keep_holes=False):
        a = oracle.fit_hits(rows, y, z)
        b = oracle.refit_hits(rows, y, z)
        if a is None or a[4] != len(rows) or a[5] != rows[0]:
            continue            # the follower stopped early or picked something up: not the same hit list
        assert b is not None
        assert np.float32(a[0]).tobytes() == np.float32(b[0]).tobytes()
        assert a[2].tobytes() == b[2].tobytes() and a[3].tobytes() == b[3].tobytes() and a[1] == b[1]
        n += 1
    assert n >= 100


def test_refit_pulls_have_unit_width_with_holes():
    """Lists with holes (hit probability 0.8): pulls of the refit parameters at the innermost cluster."""
    cfg = dg.preset("C1", tracks_per_event=5000, noise_frac=0.0, seed=78, pt_lo=0.3, p_hit=0.8)
    x_rows, _, _, _ = oracle.geom_tables()
    alpha = math.radians(10.0)
    pulls = []
    for rows, y, z, tr in _track_hit_lists(cfg, 50, keep_holes=True):
        fit = oracle.refit_hits(rows, y, z)
        if fit is None:
            continue
        chi2, x, p, c, n = fit
        assert x == x_rows[rows[0]] and n == len(rows)
        want = _true_state_at(float(x), float(tr["phi0"]) - alpha, float(tr["pt"]), int(tr["charge"]), float(tr["tanl"]))
        diag = np.array([c[0], c[2], c[5], c[9], c[14]], dtype=np.float64)
        pulls.append((p.astype(np.float64) - want) / np.sqrt(diag))
    pulls = np.array(pulls)
    assert len(pulls) >= 1500, len(pulls)
    mean, width = pulls.mean(axis=0), pulls.std(axis=0)
    assert np.all(np.abs(mean[[0, 2, 4]]) <= 0.08), mean
    assert np.all(np.abs(mean[[1, 3]]) <= 0.12), mean
    assert np.all((width >= 0.93) & (width <= 1.12)), width
