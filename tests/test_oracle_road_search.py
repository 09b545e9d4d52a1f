"""Pins of the follower's ROAD SEARCH (R5.3 / R5.5 / R5.6) and of the selector key for
negative weights (R6.1).  PAPER.md:27 (section 2): the follower propagates every seed "picking up
more clusters of the track"; PAPER.md:57 (section 3): chi2 gets priority in the selection weight.

Every expectation below is worked out BY HAND in the docstring from the readings, on inputs built
so that the hand computation is exact or has wide margins:

* a RADIAL STRAIGHT track (y = 0, z = z0 on every row): every residual of its own hits is exactly
  0, the state stays exactly (0, z0, 0, 0, 0), the (y,s,q) and (z,t) blocks of C never mix, so the
  prediction on every row is exactly (0, z0) with C10 = 0, and
  chi2(candidate) = dy^2/(C00+Vy) + dz^2/(C11+Vz) with Vy = Vz = 0.01;
* prediction variances from the textbook weighted-least-squares formulas (numpy, float64), which
  share nothing with the oracle.

The last test is a brute force: every road search the oracle performed on a dense frame is redone
with a numpy linear scan of the whole pad row.
"""
import numpy as np

import oracle
from paper_2601_20569_b200 import datagen as dg

R = 152
Z0 = np.float32(100.0)
VY = 0.1 * 0.1


def frame(recs):
    """recs: list of (row, y, z) in INPUT ORDER (= original ids)."""
    c = np.zeros(len(recs), dtype=oracle.CLUSTER_DTYPE)
    c["row"] = [r[0] for r in recs]
    c["y"] = np.float32([r[1] for r in recs])
    c["z"] = np.float32([r[2] for r in recs])
    return c


def radial(rows):
    return [(int(r), 0.0, float(Z0)) for r in rows]


def test_own_hit_beats_decoy_on_every_row():
    """(a) Radial track on rows 10..80 with the hits of rows 20,30,...,70 removed (so the link chains
    are short and most rows are reached by the road search), plus, on every row that holds a track
    hit, a decoy at (+-0.2, z0+0.2) listed BEFORE the track hits (lower original ids).
    By hand: the track's own hit has chi2 = 0 exactly; the decoy has
    chi2 = 0.04/(C00+Vy) + 0.04/(C11+Vz) > 0 and lies inside the road (0.2 < road_min = 0.3).
    The decoys get no reciprocal link (their best pair is (track hit, track hit), whose own partners
    are track hits), so every seed is a piece of the track.
    => every tracklet holds exactly the track's hits, no decoy, on all 65 rows."""
    keep = [r for r in range(10, 81) if r % 10 != 0 or r in (10, 80)]
    decoys = [(r, 0.2 if r % 2 == 0 else -0.2, float(Z0) + 0.2) for r in keep]
    cl = frame(decoys + radial(keep))
    own = {r: len(decoys) + i for i, r in enumerate(keep)}
    o = oracle.run(cl, want=("seeds", "tracklets", "trace"))
    assert o.n_seeds >= 6 and o.n_tracklets == o.n_seeds
    for k in range(o.n_seeds):
        h = o.row_hit[k]
        assert {r: int(h[r]) for r in keep} == own
        assert np.all(h[[r for r in range(R) if r not in own]] == -1)
        assert o.tracklets[k]["n_hits"] == len(keep)
    # the searches really had two candidates to choose from, and the prediction is exact
    t = o.trace[(o.trace["searched"] == 1) & (o.trace["picked_id"] >= 0)]
    assert len(t) > 300
    assert np.all(t["y"] == 0.0) and np.all(t["z"] == Z0) and np.all(t["c10"] == 0.0) and np.all(t["chi2"] == 0.0)


def test_exact_chi2_tie_goes_to_the_lower_original_id():
    """(b) Rule D2.  Radial track on rows 10..50; row 51 holds no track hit but two candidates at
    mirrored positions (-0.2, z0) and (+0.2, z0): dy^2 is the same fp32 number and C10 = 0, so both
    have exactly the same chi2 = 0.04/(C00+Vy) (< 12, inside the road).  With 0.25 cm bins they sit
    in different bins, the one at -0.2 is visited first.  Expected: the one with the LOWER original
    id, whichever side it is on; same in z with (0, z0 -+ 0.2)."""
    p = oracle.default_params(grid_dy=0.25, grid_dz=0.25)
    for a, b in (((-0.2, 0.0), (0.2, 0.0)), ((0.0, -0.2), (0.0, 0.2))):
        for low_first in (False, True):
            first, second = (a, b) if low_first else (b, a)
            # ids 0 and 1 are the two candidates, in this order
            cl = frame([(51, first[0], float(Z0) + first[1]), (51, second[0], float(Z0) + second[1])]
                       + radial(range(10, 51)))
            o = oracle.run(cl, params=p, want=("seeds", "tracklets", "trace"))
            assert o.n_seeds == 1 and o.n_tracklets == 1
            assert o.row_hit[0][51] == 0, (a, b, low_first)
            t = o.trace[(o.trace["row"] == 51) & (o.trace["dir"] == 1)][0]
            assert t["c10"] == 0.0 and t["y"] == 0.0 and t["z"] == Z0 and t["accepted"] == 1


def wls_prediction_variance(hit_rows, row_pred, dx, cf, p):
    """Textbook weighted least squares, float64: y(x) = y0 + s*x + cf*q*x^2/2 (small angles) with
    priors var(s) = init_var_sinphi, var(q) = init_var_qpt and none on y0; z(x) = z0 + t*x with prior
    var(t) = init_var_tanl.  Returns (var_y, var_z) of the prediction on row_pred."""
    x = (np.asarray(hit_rows, dtype=np.float64) - row_pred) * dx
    A = np.stack([np.ones_like(x), x, 0.5 * cf * x * x], axis=1)
    info = A.T @ A / VY + np.diag([0.0, 1.0 / p.init_var_sinphi, 1.0 / p.init_var_qpt])
    B = np.stack([np.ones_like(x), x], axis=1)
    info_z = B.T @ B / VY + np.diag([0.0, 1.0 / p.init_var_tanl])
    return np.linalg.inv(info)[0, 0], np.linalg.inv(info_z)[0, 0]


def test_chi2_cut_decides_between_taken_and_missing():
    """(c) Radial track on rows 10..60 and 64..68; rows 61 and 63 are empty and row 62 holds only a
    decoy (with empty neighbour rows it cannot enter a link chain; rows 64..68 are too few for a
    seed of their own), so there is ONE seed (chain 11..59) whose outward search meets the decoy.
    Prediction variance on row 62 from the 50 hits of rows 11..60 (WLS, wls_prediction_variance):
    C00 ~ 0.0020, C11 ~ 0.0009, so S00 = C00+Vy, S11 = C11+Vz lie in [0.0105, 0.0125].
      decoy at (0.20, z0+0.20): chi2 = 0.04/S00 + 0.04/S11 in [6.4, 7.7]  <= 12  => TAKEN;
      decoy at (0.32, z0+0.32): chi2 = 0.1024/S00 + 0.1024/S11 in [16, 19.6] > 12 => row MISSING
        although it is inside the road (0.32 < 3.5*sqrt(S) >= 0.35), and the follower goes on to
        rows 64..68 across the three-row gap."""
    x, _, dx, cf = oracle.geom_tables()
    p = oracle.default_params()
    vy, vz = wls_prediction_variance(range(11, 61), 62, dx, cf, p)
    assert 0.0105 < VY + vy < 0.0125 and 0.0105 < VY + vz < 0.0125
    for d, taken in ((0.20, True), (0.32, False)):
        rows = list(range(10, 61)) + list(range(64, 69))
        cl = frame([(62, d, float(Z0) + d)] + radial(rows))
        o = oracle.run(cl, want=("seeds", "tracklets", "trace"))
        assert o.n_seeds == 1 and o.seeds[0]["len"] == 49 and o.n_tracklets == 1
        h = o.row_hit[0]
        assert h[62] == (0 if taken else -1), d
        assert np.all(h[64:69] >= 1) and o.tracklets[0]["row_last"] == 68
        t = o.trace[(o.trace["row"] == 62) & (o.trace["dir"] == 1)][0]
        # the oracle's covariance on that row against the closed form (1 %)
        assert abs(t["c00"] - vy) < 0.01 * vy + 1e-7 and abs(t["c11"] - vz) < 0.01 * vz + 1e-7 and t["c10"] == 0
        chi2 = d * d / (VY + vy) + d * d / (VY + vz)
        assert t["picked_id"] == 0 and abs(t["chi2"] - chi2) < 0.01 * chi2
        assert bool(t["accepted"]) == taken == (chi2 <= 12.0)


def test_z_road_width_comes_from_c11():
    """(d) Short seed, then a hole: radial track on rows 10..15 (chain 11..14, seed length 4; row 15
    is picked up with chi2 = 0), nothing on rows 16, 17, one cluster on row 18 at (0, z0+0.55).
    z-line through the 5 fitted hits (rows 11..15) extrapolated 3 rows: var = Vz*(1/5 + 5^2*12/(5*24))
    = 2.7 Vz = 0.027 (the tan-lambda prior, var 4, is negligible) => rz = 3.5*sqrt(0.037) = 0.673 > 0.55
    and chi2 = 0.3025/0.037 = 8.2 <= 12  => TAKEN.  (A road built from anything but C11 -- e.g. the
    off-diagonal C10, which is exactly 0 here -- would be 0.35 wide and miss it.)
    The same cluster at z0+0.75 is outside the z road (0.75 > 0.673) => not taken."""
    x, _, dx, cf = oracle.geom_tables()
    p = oracle.default_params(min_hits_tracklet=5)
    _, vz = wls_prediction_variance(range(11, 16), 18, dx, cf, p)
    assert abs(vz - 0.027) < 2e-4
    for dz, taken in ((0.55, True), (0.75, False)):
        cl = frame([(18, 0.0, float(Z0) + dz)] + radial(range(10, 16)))
        o = oracle.run(cl, params=p, want=("seeds", "tracklets", "trace"))
        assert o.n_seeds == 1 and o.seeds[0]["len"] == 4 and o.n_tracklets == 1
        assert o.row_hit[0][18] == (0 if taken else -1)
        assert o.tracklets[0]["n_hits"] == (7 if taken else 6)
        t = o.trace[(o.trace["row"] == 18) & (o.trace["dir"] == 1)][0]
        assert abs(t["c11"] - vz) < 0.01 * vz and t["c10"] == 0.0
        assert t["picked_id"] == (0 if taken else -1)


def test_rows_beyond_the_acceptance_are_missing_rows():
    """(e) R5.3: if |y_pred| > ylim_r = ymax_r + 2 cm the row is missing, whatever lies nearby.
    Straight track of slope dy/dx = 0.5 at constant z, hits on rows 60..99, aimed so that on row 100
    it is 0.10 cm BEYOND ylim_100 (on row 99 it is 0.24 cm inside: the acceptance edge has slope
    tan 10 deg = 0.176).  A decoy sits on row 100 at ylim_100 - 0.05, i.e. 0.15 cm from the prediction:
    chi2 ~ 0.0225/0.011 ~ 2, well inside road and cut.  Expected: NOT taken, row 100 is not searched,
    the tracklet ends on row 99."""
    x, ymax, dx, _ = oracle.geom_tables()
    re_ = 100
    ylim = float(ymax[re_]) + 2.0
    line = lambda r: ylim + 0.10 - 0.5 * (float(x[re_]) - float(x[r]))
    assert line(99) < float(ymax[99]) + 2.0 - 0.2 and line(60) > 0
    cl = frame([(re_, ylim - 0.05, 50.0)] + [(r, line(r), 50.0) for r in range(60, re_)])
    o = oracle.run(cl, want=("seeds", "tracklets", "trace"))
    assert o.n_dropped == 0 and o.n_seeds == 1 and o.n_tracklets == 1
    assert o.row_hit[0][re_] == -1 and not np.any(o.row_hit == 0)
    assert o.tracklets[0]["row_last"] == 99 and o.tracklets[0]["n_hits"] == 40
    t = o.trace[(o.trace["row"] == re_) & (o.trace["dir"] == 1)][0]
    assert t["searched"] == 0 and abs(t["y"] - (ylim + 0.10)) < 0.01
    # control: the same decoy 0.2 cm further in, track aimed 0.1 cm INSIDE the edge => taken
    line2 = lambda r: ylim - 0.10 - 0.5 * (float(x[re_]) - float(x[r]))
    cl = frame([(re_, ylim - 0.25, 50.0)] + [(r, line2(r), 50.0) for r in range(60, re_)])
    o = oracle.run(cl, want=("tracklets",))
    assert o.row_hit[0][re_] == 0 and o.tracklets[0]["row_last"] == re_


def test_hits_below_the_row_where_the_inward_refit_stops_are_dropped():
    """(f) DESIGN.md R5.5 Delta: if the leg ends inside the refit (|sin phi| would leave max_sinphi),
    the recorded hits below the stopping row are NOT part of the tracklet.
    Hand-built with max_sinphi = 0.30: an exact circle of radius 66.7 cm (pT = 0.1 GeV/c), z constant,
    hits on rows 49..85, sin phi = 0.305 on row 50 falling by dx/R = 0.0159 per row (-0.25 on row 85).
      chain = rows 50..84, start hit on row 50;
      outward: the initial sin phi is the chord direction rows 50->51 = 0.297 <= 0.30, then it
        falls: the whole chain is fitted, row 85 is picked up, row_last = 85;
      inward refit: on row 51 sin phi = 0.289; the step to row 50 would give 0.305 > 0.30
        => the leg ends on row 51.
    Expected tracklet: rows 51..85, n_hits = 35, row_first = 51, and NO hit on row 50 although it is
    the seed's own start hit (and none on row 49: the inward search never starts)."""
    x, _, dx, _ = oracle.geom_tables()
    Rc, s50 = 66.7, 0.305
    rows = np.arange(49, 86)
    sphi = s50 - (x[rows].astype(np.float64) - float(x[50])) / Rc
    y = Rc * (np.sqrt(1 - sphi ** 2) - np.sqrt(1 - s50 ** 2))
    cl = frame([(int(r), float(v), 20.0) for r, v in zip(rows, y)])
    p = oracle.default_params(max_sinphi=0.30)
    o = oracle.run(cl, params=p, want=("seeds", "tracklets"))
    assert o.n_seeds == 1 and o.seeds[0]["row"] == 50 and o.seeds[0]["len"] == 35
    t = o.tracklets[0]
    assert (t["n_hits"], t["row_first"], t["row_last"]) == (35, 51, 85)
    h = o.row_hit[0]
    assert h[50] == -1 and h[49] == -1 and np.array_equal(h[51:86], np.arange(2, 37))
    assert 0.28 < t["p"][2] < 0.30                      # sin phi on row 51
    # control: with the default limit nothing stops, rows 49..85 all belong to the tracklet
    o = oracle.run(cl, want=("tracklets",))
    assert (o.tracklets[0]["n_hits"], o.tracklets[0]["row_first"]) == (37, 49)


def test_tracklet_counts_agree_with_row_hit():
    """Invariant of every tracklet (dense low-pT frame): n_hits = number of rows holding a hit,
    row_first / row_last = first / last such row; rejected tracklets hold no hit."""
    cl, _, _ = dg.generate(dg.preset("C5", tracks_per_event=3000, seed=31))
    p = oracle.default_params(err_y=0.15, err_z=0.15, nf_max_d2=1.6)
    o = oracle.run(cl, params=p, want=("seeds", "tracklets"))
    ok = o.tracklets["n_hits"] > 0
    assert ok.sum() > 300
    has = o.row_hit >= 0
    assert np.array_equal(has.sum(axis=1)[ok], o.tracklets["n_hits"][ok])
    assert np.all(has.sum(axis=1)[~ok] == 0)
    assert np.array_equal(has.argmax(axis=1)[ok], o.tracklets["row_first"][ok])
    assert np.array_equal((R - 1 - has[:, ::-1].argmax(axis=1))[ok], o.tracklets["row_last"][ok])


def test_selector_orders_negative_weights():
    """(g) R6.1: Q = nHits - 2*chi2/ndf can be negative; the key order must still be the order of
    Q.  Two tracklets over the same 60 clusters (ndf = 115): chi2 = 100*115 -> Q = 60 - 200 = -140;
    chi2 = 50*115 -> Q = 60 - 100 = -40.  The LESS negative one (-40) owns all clusters and is the
    only track; a third case mixes signs: Q = -40 loses against Q = +10 (chi2 = 25*115)."""
    h = np.full(R, -1, np.int32)
    h[20:80] = np.arange(60)
    o = oracle.select_only(np.stack([h, h]), [60, 60], [100.0 * 115, 50.0 * 115], [1, 2], n_clusters=60)
    assert o.n_tracks == 1 and o.tracks[0]["seed_id"] == 2 and o.tracks[0]["n_shared"] == 0
    o = oracle.select_only(np.stack([h, h]), [60, 60], [50.0 * 115, 100.0 * 115], [1, 2], n_clusters=60)
    assert o.n_tracks == 1 and o.tracks[0]["seed_id"] == 1
    o = oracle.select_only(np.stack([h, h, h]), [60, 60, 60], [50.0 * 115, 25.0 * 115, 100.0 * 115], [1, 2, 3],
                           n_clusters=60)
    assert o.n_tracks == 1 and o.tracks[0]["seed_id"] == 2


def test_road_search_brute_force_on_a_dense_frame():
    """Every road search of the oracle on a dense low-pT frame (C5-like, ~1 cluster/cm^2, several
    candidates per road) redone with a numpy LINEAR SCAN of the whole pad row, in float64:
      searched  <=> |y_pred| <= ymax_r + 2;
      road      ry = clamp(3.5*sqrt(C00+Vy), 0.3, 2.0), rz likewise from C11   (R5.3);
      candidate <=> |y_c - y| <= ry and |z_c - z| <= rz;
      chi2      = r^T (H C H^T + V)^-1 r  (numpy solve);
      picked    = the minimum of (chi2, original id); accepted <=> chi2 <= 12.
    Decisions closer than 1e-4 (relative) to a threshold or to the runner-up are skipped (fp32 vs
    fp64 rounding) and must stay below 1 % of all searches."""
    cl, _, _ = dg.generate(dg.preset("C5", tracks_per_event=4000, seed=15))
    p = oracle.default_params(err_y=0.15, err_z=0.15, nf_max_d2=1.6)
    o = oracle.run(cl, params=p, want=("trace",))
    x, ymax, _, _ = oracle.geom_tables()
    V = 0.15 * 0.15
    t = o.trace
    assert len(t) > 20000
    by_row = {}
    for r in range(R):      # rows 63.. are empty in this frame; the follower still steps onto them
        m = np.flatnonzero((cl["row"] == r) & np.isfinite(cl["y"]) & (np.abs(cl["y"]) <= np.float32(ymax[r] + 2.0)))
        by_row[r] = (m, cl["y"][m].astype(np.float64), cl["z"][m].astype(np.float64))
    n_multi = n_skip = n_acc = n_rej = 0
    for rec in t:
        r = int(rec["row"])
        y, z = float(rec["y"]), float(rec["z"])
        inside = abs(y) <= float(np.float32(ymax[r] + 2.0))
        assert bool(rec["searched"]) == inside
        if not inside:
            assert rec["picked_id"] == -1 and rec["accepted"] == 0
            continue
        S = np.array([[float(rec["c00"]) + V, float(rec["c10"])], [float(rec["c10"]), float(rec["c11"]) + V]])
        ry = min(max(3.5 * np.sqrt(S[0, 0]), 0.3), 2.0)
        rz = min(max(3.5 * np.sqrt(S[1, 1]), 0.3), 2.0)
        ids, ys, zs = by_row[r]
        dy, dz = ys - y, zs - z
        edge = (np.abs(np.abs(dy) - ry) < 1e-4) | (np.abs(np.abs(dz) - rz) < 1e-4)
        m = (np.abs(dy) <= ry) & (np.abs(dz) <= rz)
        if np.any(edge & (np.abs(dy) <= ry + 1e-4) & (np.abs(dz) <= rz + 1e-4)):
            n_skip += 1
            continue
        if not m.any():
            assert rec["picked_id"] == -1 and rec["accepted"] == 0
            continue
        res = np.stack([dy[m], dz[m]], axis=0)
        chi2 = np.einsum("ik,ik->k", res, np.linalg.solve(S, res))
        order = np.lexsort((ids[m], chi2))
        best = order[0]
        n_multi += len(order) > 1
        if len(order) > 1 and chi2[order[1]] - chi2[best] < 1e-4 * max(chi2[best], 1.0):
            n_skip += 1
            continue
        assert rec["picked_id"] == ids[m][best]
        assert abs(rec["chi2"] - chi2[best]) <= 1e-3 * max(chi2[best], 1.0)
        if abs(chi2[best] - 12.0) < 1e-3:
            n_skip += 1
            continue
        assert bool(rec["accepted"]) == (chi2[best] <= 12.0)
        n_acc += int(rec["accepted"])
        n_rej += 1 - int(rec["accepted"])
    assert n_multi > 2000 and n_acc > 5000 and n_rej > 500      # the frame exercises choice and cut
    assert n_skip < 0.01 * len(t)


def test_shared_budget_at_the_exact_boundary():
    """R6.3, running fraction from the outermost row: a foreign cluster is accepted as shared iff
    (n_shared+1)*1000 <= shared_permille*(n_accepted+1).  Tracklet A = rows 0..29 (30 clusters);
    a better tracklet B (rows 60..119, chi2 0) also holds ONE of A's clusters.
      foreign cluster on row 20: A has accepted rows 29..21 = 9 clusters: 1*1000 <= 100*(9+1) holds
        with equality => accepted as shared: A keeps 30 clusters, 1 shared;
      foreign cluster on row 21: 8 accepted: 1000 <= 100*9 fails => refused: 29 clusters, 0 shared."""
    a = np.full(R, -1, np.int32)
    a[0:30] = np.arange(30)
    for row, expect in ((20, (30, 1)), (21, (29, 0))):
        b = np.full(R, -1, np.int32)
        b[60:120] = 100 + np.arange(60)
        b[row] = a[row]
        o = oracle.select_only(np.stack([a, b]), [30, 61], [30.0, 0.0], [1, 2], n_clusters=200)
        t = o.tracks[o.tracks["seed_id"] == 1][0]
        assert (t["n_clusters"], t["n_shared"]) == expect, row
