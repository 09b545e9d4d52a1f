"""Pins of the oracle's path steps R1..R6: invariants, brute force on tiny inputs,
constructed cases, and the behaviours PAPER.md states.  None of the references below uses
the oracle's grid or its code: they are numpy linear scans / hand-built examples.
"""
import numpy as np
import pytest

import oracle
from paper_2601_20569_b200 import datagen as dg
from paper_2601_20569_b200.metrics import track_quality

R = 152


def mk_clusters(rows, y, z, sector=0):
    c = np.zeros(len(rows), dtype=oracle.CLUSTER_DTYPE)
    c["row"], c["y"], c["z"], c["sector"] = rows, y, z, sector
    return c


# ------------------------------------------------------------------ R1 grid
def test_grid_invariants_and_rebinning(c1, c1_oracle):
    cl, o = c1[0], c1_oracle
    assert o.n_sorted + o.n_dropped + o.n_ignored == len(cl)
    bs = o.bin_start.astype(np.int64)
    assert np.all(np.diff(bs) >= 0) and bs[0] == 0 and bs[-1] == o.n_sorted
    assert sorted(o.sorted_ids.tolist()) == list(range(len(cl)))  # a permutation (nothing dropped in C1)
    x, ymax, _, _ = oracle.geom_tables()
    for r in range(R):
        d = o.row_desc[r]
        ids = o.sorted_ids[d["clu_ofs"]:d["clu_ofs"] + d["count"]]
        assert np.all(cl["row"][ids] == r)
        if d["count"] == 0:
            continue
        # closed-form grid descriptor: y0 = -(ymax+2), ny = ceil(2(ymax+2)/2), z0 = min z
        assert abs(d["y0"] + (ymax[r] + 2.0)) < 1e-5
        assert d["ny"] == int(np.ceil((float(ymax[r]) + 2.0)))
        assert d["z0"] == cl["z"][ids].min()
        assert d["nz"] == int(np.floor((cl["z"][ids].max() - d["z0"]) / np.float32(2.0))) + 1
        # every cluster sits in the bin its coordinates give; ids ascending inside a bin
        for b in range(d["ny"] * d["nz"]):
            lo, hi = bs[d["bin_ofs"] + b], bs[d["bin_ofs"] + b + 1]
            if hi == lo:
                continue
            m = o.sorted_ids[lo:hi]
            by = np.clip(np.floor((cl["y"][m] - d["y0"]) * np.float32(0.5)), 0, d["ny"] - 1)
            bz = np.clip(np.floor((cl["z"][m] - d["z0"]) * np.float32(0.5)), 0, d["nz"] - 1)
            assert np.all(bz * d["ny"] + by == b)
            assert np.all(np.diff(m.astype(np.int64)) > 0)


def test_grid_drops_and_ignores():
    x, ymax, _, _ = oracle.geom_tables()
    rows = np.array([10, 10, 10, 10, 11])
    y = np.array([0.0, ymax[10] + 1.9, ymax[10] + 2.5, np.nan, 0.0], dtype=np.float32)
    z = np.array([1.0, 2.0, 3.0, 4.0, np.inf], dtype=np.float32)
    o = oracle.run(mk_clusters(rows, y, z), sector_hi=1)
    assert (o.n_sorted, o.n_dropped, o.n_ignored) == (2, 1, 2)
    assert sorted(o.sorted_ids.tolist()) == [0, 1]


# ------------------------------------------------------------------ R2 neighbour finder
def brute_force_links(cl, dx, x, wy_slope=1.0, wz_slope=1.6, max_d2=0.70):
    """O(N^2) reference without any grid: all (j,k) on rows r+-1, fp32 arithmetic in the
    order DESIGN.md R2 states, lexicographic (d2, j, k) minimum."""
    f = np.float32
    n = len(cl)
    up = np.full(n, -1, np.int32)
    dn = np.full(n, -1, np.int32)
    wy, wz = f(wy_slope) * f(dx), f(wz_slope) * f(dx)
    by_row = {r: np.flatnonzero(cl["row"] == r) for r in range(R)}
    for i in range(n):
        r = int(cl["row"][i])
        if r < 1 or r > R - 2:
            continue
        yi, zi = f(cl["y"][i]), f(cl["z"][i])
        ty = f(yi / f(x[r])) * f(dx)
        U = [j for j in by_row[r + 1]
             if abs(f(f(cl["y"][j] - yi) - ty)) <= wy and abs(f(cl["z"][j] - zi)) <= wz]
        D = [k for k in by_row[r - 1]
             if abs(f(f(yi - cl["y"][k]) - ty)) <= wy and abs(f(zi - cl["z"][k])) <= wz]
        best = None
        for j in U:
            for k in D:
                dy = f(f(cl["y"][j] - yi) + f(cl["y"][k] - yi))
                dz = f(f(cl["z"][j] - zi) + f(cl["z"][k] - zi))
                d2 = f(f(dy * dy) + f(dz * dz))
                if d2 <= f(max_d2) and (best is None or (d2, j, k) < best):
                    best = (d2, j, k)
        if best:
            up[i], dn[i] = best[1], best[2]
    return up, dn


def test_neighbours_match_brute_force_on_small_frame():
    cl, _, _ = dg.generate(dg.preset("C1", tracks_per_event=40, noise_frac=0.3, seed=5))
    assert 500 < len(cl) <= 2500
    x, _, dx, _ = oracle.geom_tables()
    o = oracle.run(cl)
    up, dn = brute_force_links(cl, dx, x)
    assert np.array_equal(o.link_up, up) and np.array_equal(o.link_dn, dn)
    assert (up >= 0).sum() > 200


def test_neighbours_dense_blob_brute_force():
    """Dense random blob (many candidates per window, C5-like) on 5 rows."""
    rng = np.random.default_rng(3)
    n = 1500
    rows = rng.integers(40, 45, n)
    y = rng.uniform(-4, 4, n).astype(np.float32)
    z = rng.uniform(100, 108, n).astype(np.float32)
    cl = mk_clusters(rows, y, z)
    x, _, dx, _ = oracle.geom_tables()
    o = oracle.run(cl)
    up, dn = brute_force_links(cl, dx, x)
    assert np.array_equal(o.link_up, up) and np.array_equal(o.link_dn, dn)
    assert (up >= 0).mean() > 0.4


def test_neighbours_hand_built_best_pair_and_ties():
    x, _, dx, _ = oracle.geom_tables()
    # centre cluster 0 on row 50 at y=0: straight candidates and an exact tie
    rows = [50, 51, 51, 49, 49, 51]
    y = [0.0, 0.35, 0.10, -0.10, -0.30, 0.10]
    z = [10.0, 10.5, 10.5, 9.5, 9.5, 10.5]
    o = oracle.run(mk_clusters(rows, np.float32(y), np.float32(z)))
    # pairs: (2,3): dy=0,dz=0 -> d2=0 ; (5,3) identical coordinates to (2,3): tie -> lower id 2
    assert o.link_up[0] == 2 and o.link_dn[0] == 3
    # one-sided: remove the down candidates -> no link at all
    o = oracle.run(mk_clusters(rows[:3], np.float32(y[:3]), np.float32(z[:3])))
    assert o.link_up[0] == -1 and o.link_dn[0] == -1
    # beyond the straightness cut (dy = 0.9 -> d2 = 0.81 > 0.70)
    o = oracle.run(mk_clusters([50, 51, 49], np.float32([0, 0.45, 0.45]), np.float32([0, 0, 0])))
    assert o.link_up[0] == -1
    o = oracle.run(mk_clusters([50, 51, 49], np.float32([0, 0.40, 0.40]), np.float32([0, 0, 0])))
    assert o.link_up[0] == 1 and o.link_dn[0] == 2
    # rows 0 and 151 get no links of their own
    o = oracle.run(mk_clusters([0, 1, 2], np.float32([0, 0, 0]), np.float32([0, 0, 0])))
    assert o.link_up.tolist() == [-1, 2, -1] and o.link_dn.tolist() == [-1, 0, -1]


@pytest.mark.parametrize("dy,dz", [(1.0, 1.0), (4.0, 4.0), (1.0, 8.0), (0.5, 3.0)])
def test_results_do_not_depend_on_bin_size(c1, c1_oracle, dy, dz):
    """Rule D3: the grid is a performance device; links, seeds, tracks are defined by the
    window inequalities alone."""
    o = oracle.run(c1[0], params=oracle.default_params(grid_dy=dy, grid_dz=dz))
    ref = c1_oracle
    for name in ("link_up", "link_dn", "link_up2", "link_dn2", "row_hit", "cluster_ids", "cluster_shared"):
        assert np.array_equal(getattr(o, name), getattr(ref, name)), name
    assert np.array_equal(o.seeds, ref.seeds)
    assert o.tracks.tobytes() == ref.tracks.tobytes()
    assert o.tracklets.tobytes() == ref.tracklets.tobytes()


# ------------------------------------------------------------------ R3 / R4
def test_cleanup_invariants(c1, c1_oracle):
    cl, o = c1[0], c1_oracle
    up2, dn2 = o.link_up2, o.link_dn2
    i = np.flatnonzero(up2 >= 0)
    assert np.array_equal(dn2[up2[i]], i)
    k = np.flatnonzero(dn2 >= 0)
    assert np.array_equal(up2[dn2[k]], k)
    assert np.all(cl["row"][up2[i]].astype(int) == cl["row"][i].astype(int) + 1)
    assert np.all(cl["sector"][up2[i]] == cl["sector"][i])
    # a subset of the raw links
    assert np.all((up2 == o.link_up) | (up2 == -1))
    # idempotent
    up3 = np.where((up2 >= 0) & (dn2[np.maximum(up2, 0)] == np.arange(len(up2))), up2, -1)
    assert np.array_equal(up3, up2)
    # removed links were indeed not reciprocal
    removed = np.flatnonzero((o.link_up >= 0) & (up2 < 0))
    assert np.all(o.link_dn[o.link_up[removed]] != removed)


def test_seed_invariants_no_chain_breaks(c1, c1_oracle):
    """North star invariant: no seed whose link chain breaks; chains vertex-disjoint."""
    o = c1_oracle
    seen = set()
    assert o.n_seeds > 100
    assert np.all(np.diff(o.seeds["start_id"].astype(np.int64)) > 0)  # rule D4 (single sector)
    for s in o.seeds:
        c, n = int(s["start_id"]), 0
        assert o.link_dn2[c] == -1
        while c >= 0:
            assert c not in seen
            seen.add(c)
            n += 1
            c = int(o.link_up2[c])
        assert n == s["len"] and n >= 4
    # every chain of >= 4 is a seed
    starts = np.flatnonzero((o.link_dn2 < 0) & (o.link_up2 >= 0))
    n_long = 0
    for c in starts:
        n, k = 0, int(c)
        while k >= 0:
            n, k = n + 1, int(o.link_up2[k])
        n_long += n >= 4
    assert n_long == o.n_seeds


def noise_free_track(seed=11, pt=1.0):
    cfg = dg.preset("C1", tracks_per_event=1, noise_frac=0.0, seed=seed, smear_y=0.0, smear_z=0.0,
                    p_hit=1.0, pt_lo=pt, pt_hi=pt * 1.0001, pt_uniform=1)
    return dg.generate(cfg)


def test_noise_free_single_track_one_seed_one_track():
    for seed in range(11, 40):
        cl, lab, tr = noise_free_track(seed)
        if len(cl) >= 100 and len(np.unique(cl["row"])) == len(cl):
            break
    o = oracle.run(cl)
    rows = np.sort(cl["row"])
    assert np.all(np.diff(rows) == 1)
    # one seed; its chain spans every row except the two end clusters, which have no
    # (up, down) PAIR of their own and therefore no reciprocal link (R2: both links or none)
    assert o.n_seeds == 1 and o.seeds[0]["len"] == len(cl) - 2
    assert o.seeds[0]["row"] == rows[0] + 1
    assert o.n_tracklets == 1 and o.tracklets[0]["n_hits"] == len(cl)
    assert sorted(o.row_hit[0][o.row_hit[0] >= 0].tolist()) == list(range(len(cl)))
    assert o.n_tracks == 1 and o.tracks[0]["n_clusters"] == len(cl) and o.tracks[0]["n_shared"] == 0
    assert np.array_equal(cl["row"][o.cluster_ids], rows)     # ascending in row


def test_follower_bridges_gaps_and_picks_up():
    """Remove rows from a noise-free track: the seed covers one chain, the follower picks up
    the rest across gaps <= max_gap_follow and stops at a larger hole."""
    for seed in range(11, 40):
        cl, _, _ = noise_free_track(seed)
        if len(cl) >= 140 and len(np.unique(cl["row"])) == len(cl) and cl["row"].min() == 0:
            break
    keep = np.ones(len(cl), bool)
    r = cl["row"]
    keep[(r == 30) | (r == 31) | (r == 60) | ((r >= 90) & (r < 94))] = False  # gaps of 2, 1, 4
    keep[(r >= 120) & (r < 126)] = False                                       # hole of 6 > max gap
    sub = cl[keep]
    o = oracle.run(sub)
    assert o.n_seeds >= 4
    best = o.tracklets[np.argmax(o.tracklets["n_hits"])]
    assert best["row_first"] == 0 and best["row_last"] == 119
    assert best["n_hits"] == 120 - 2 - 1 - 4
    # the part above the hole is its own tracklet
    assert np.any((o.tracklets["row_first"] == 126) & (o.tracklets["n_hits"] == r.max() - 125))


def test_follower_efficiency_on_c1(c1, c1_oracle):
    """With smearing: >= 95 % of findable tracks have a tracklet holding >= 90 % of their
    in-sector clusters (SURVEY 8(c) pin; prototype 98.6 %)."""
    cl, lab, _ = c1
    o = c1_oracle
    labs, cnt = np.unique(lab[lab >= 0], return_counts=True)
    findable = labs[cnt >= 70]
    ok = 0
    hit_lab = np.where(o.row_hit >= 0, lab[np.maximum(o.row_hit, 0)], -2)
    for m, n in zip(labs[cnt >= 70], cnt[cnt >= 70]):
        per_tracklet = (hit_lab == m).sum(axis=1)
        ok += per_tracklet.max() >= 0.9 * n
    assert ok >= 0.95 * len(findable)


# ------------------------------------------------------------------ R6 selector
def check_selector_invariants(o, params, row_of):
    own_count = np.zeros(o.n_clusters, dtype=np.int64)
    tot_count = np.zeros(o.n_clusters, dtype=np.int64)
    for t in o.tracks:
        ids = o.cluster_ids[t["cluster_ofs"]:t["cluster_ofs"] + t["n_clusters"]]
        sh = o.cluster_shared[t["cluster_ofs"]:t["cluster_ofs"] + t["n_clusters"]]
        assert t["n_clusters"] >= params.min_hits_track
        assert sh.sum() == t["n_shared"]
        rows = row_of[ids].astype(int)
        assert np.all(np.diff(rows) > 0)
        assert rows[0] == t["row_first"] and rows[-1] == t["row_last"]
        assert np.all(np.diff(rows) <= params.max_gap_select + 1)
        # running rule from the OUTERMOST row inward at every prefix
        n_sh = np.cumsum(sh[::-1])
        n_acc = np.arange(1, len(sh) + 1)
        assert np.all(n_sh * 1000 <= params.shared_permille * n_acc)
        own_count[ids[sh == 0]] += 1
        tot_count[ids] += 1
    assert own_count.max(initial=0) <= 1          # every cluster owned by at most one track
    multi = tot_count > 1
    assert np.all(tot_count[multi] - own_count[multi] >= tot_count[multi] - 1)


def test_selector_invariants_on_c1(c1, c1_oracle):
    check_selector_invariants(c1_oracle, oracle.default_params(), c1[0]["row"])
    assert c1_oracle.n_tracks > 50


def test_selector_invariants_dense(c1):
    cfg = dg.preset("C5", tracks_per_event=4000, seed=15)
    cl, _, _ = dg.generate(cfg)
    p = oracle.default_params(err_y=0.15, err_z=0.15, nf_max_d2=1.6, shared_permille=200)
    o = oracle.run(cl, params=p)
    assert o.n_tracks > 20 and o.cluster_shared.sum() > 0
    check_selector_invariants(o, p, cl["row"])


def straight_tracklet(rows, base):
    h = np.full(R, -1, np.int32)
    h[rows] = base + np.arange(len(rows))
    return h


def test_selector_identical_tracklets_one_survives():
    rows = np.arange(20, 80)
    h = straight_tracklet(rows, 0)
    o = oracle.select_only(np.stack([h, h]), [60, 60], [50.0, 50.0], [7, 3], n_clusters=60)
    assert o.n_tracks == 1 and o.tracks[0]["seed_id"] == 3      # tie in weight -> lower seed id
    assert o.tracks[0]["n_clusters"] == 60 and o.tracks[0]["n_shared"] == 0
    # smaller chi2 wins over equal length
    o = oracle.select_only(np.stack([h, h]), [60, 60], [80.0, 40.0], [3, 7], n_clusters=60)
    assert o.n_tracks == 1 and o.tracks[0]["seed_id"] == 7


def test_selector_chi2_priority_over_length():
    """more priority to smaller global chi2, less to length: a 58-hit tracklet
    with chi2/ndf 1 beats a 60-hit one with chi2/ndf 3 (weight = n - 2*chi2/ndf)."""
    a = straight_tracklet(np.arange(20, 80), 0)            # 60 hits
    b = a.copy()
    b[[20, 21]] = -1                                       # 58 hits, same clusters otherwise
    o = oracle.select_only(np.stack([a, b]), [60, 58], [3.0 * 115, 1.0 * 111], [1, 2], n_clusters=60)
    assert o.n_tracks == 1 and o.tracks[0]["seed_id"] == 2 and o.tracks[0]["n_clusters"] == 58


def test_selector_crossing_tracks_share_three():
    rows = np.arange(10, 70)
    a = straight_tracklet(rows, 0)          # clusters 0..59
    b = straight_tracklet(rows, 100)        # clusters 100..159
    b[[38, 39, 40]] = a[[38, 39, 40]]       # crossing: 3 common clusters in the middle
    o = oracle.select_only(np.stack([a, b]), [60, 60], [40.0, 60.0], [1, 2], n_clusters=200)
    assert o.n_tracks == 2
    t = {int(x["seed_id"]): x for x in o.tracks}
    assert t[1]["n_shared"] == 0 and t[2]["n_shared"] == 3 and t[2]["n_clusters"] == 60
    ids = o.cluster_ids[t[2]["cluster_ofs"]:t[2]["cluster_ofs"] + 60]
    sh = o.cluster_shared[t[2]["cluster_ofs"]:t[2]["cluster_ofs"] + 60]
    assert sorted(ids[sh == 1].tolist()) == sorted(a[[38, 39, 40]].tolist())


def test_selector_running_fraction_counts_from_outermost_row():
    """counting from the outermost row "allows for a larger number of shared
    clusters in the inner pad rows for long tracks": foreign clusters at the OUTER end are
    refused (no budget yet), the same number at the INNER end of a long track is accepted."""
    rows = np.arange(10, 110)                       # 100 rows
    owner = straight_tracklet(rows, 0)
    inner = straight_tracklet(rows, 1000)
    inner[10:18] = owner[10:18]                     # 8 foreign clusters on the innermost rows
    outer = straight_tracklet(rows, 2000)
    outer[102:110] = owner[102:110]                 # 8 foreign clusters on the outermost rows
    o = oracle.select_only(np.stack([owner, inner, outer]), [100, 100, 100], [50.0, 100.0, 100.0],
                           [1, 2, 3], n_clusters=3000)
    t = {int(x["seed_id"]): x for x in o.tracks}
    assert t[2]["n_shared"] == 8 and t[2]["n_clusters"] == 100      # budget accumulated
    assert t[3]["n_shared"] == 0 and t[3]["n_clusters"] == 92       # refused at the outer end
    assert t[3]["row_last"] == 101


def test_selector_gap_split_and_min_length():
    rows = np.arange(0, 120)
    owner = straight_tracklet(rows, 0)
    v = straight_tracklet(rows, 500)
    v[50:60] = owner[50:60]          # 10 foreign rows in the middle: budget allows only a few
    o = oracle.select_only(np.stack([owner, v]), [120, 120], [10.0, 300.0], [1, 2], n_clusters=1000)
    segs = sorted([(int(t["segment"]), int(t["row_first"]), int(t["row_last"]), int(t["flags"]))
                   for t in o.tracks if t["seed_id"] == 2])
    # outer part 60..119 (60 own) accepts floor(.1*(n+1)) shared going inward: rows 59..54 -> 6
    # shared (7*1000 <= 100*67 fails), then rows 53..50 missing = gap 4 (not > 4), continues
    assert len(segs) == 1 and segs[0][1] == 0 and segs[0][2] == 119
    p = oracle.default_params(max_gap_select=2)
    o = oracle.select_only(np.stack([owner, v]), [120, 120], [10.0, 300.0], [1, 2], n_clusters=1000, params=p)
    segs = sorted([(int(t["segment"]), int(t["row_first"]), int(t["row_last"]), int(t["flags"]))
                   for t in o.tracks if t["seed_id"] == 2])
    assert segs == [(0, 54, 119, 1), (1, 0, 49, 0)]   # outer segment: PARAMS_STALE
    # a remainder shorter than min_hits_track is dropped
    short = straight_tracklet(np.arange(0, 25), 800)
    short[0:10] = owner[0:10]
    o = oracle.select_only(np.stack([owner, short]), [120, 25], [10.0, 100.0], [1, 2], n_clusters=1000)
    assert [int(t["seed_id"]) for t in o.tracks] == [1]


def test_selector_monotonic_in_shared_fraction():
    """raising the shared fraction 10 % -> 20 % lets more (inner) segments
    survive."""
    cl, _, _ = dg.generate(dg.preset("C5", tracks_per_event=6000, seed=21))
    n = []
    inner = []
    for pm in (0, 100, 200):
        p = oracle.default_params(err_y=0.15, err_z=0.15, nf_max_d2=1.6, shared_permille=pm)
        o = oracle.run(cl, params=p, want=("tracks",))
        n.append(o.n_tracks)
        inner.append(int((o.tracks["row_first"] < 20).sum()))
    assert n[0] <= n[1] <= n[2] and n[0] < n[2]
    assert inner[0] <= inner[1] <= inner[2]


# ------------------------------------------------------------------ paper behaviours
def test_paper_behaviours_on_c1(c1, c1_oracle):
    cl, lab, _ = c1
    o = c1_oracle
    labs, cnt = np.unique(lab[lab >= 0], return_counts=True)
    findable = set(labs[cnt >= 70].tolist())
    seed_labels = lab[o.seeds["start_id"]]
    per_track = [int((seed_labels == m).sum()) for m in findable]
    assert np.mean(per_track) > 1.5            # "usually find multiple seeds for the same track"
    assert o.n_tracklets > o.n_tracks          # "tracks are found multiple times" ... clones removed
    assert o.tracks["n_clusters"].min() >= 20  # "cannot find very short track segments"
    q = track_quality(o.tracks["n_clusters"], o.tracks["cluster_ofs"], o.cluster_ids, o.tracks["sector"], lab)
    # sanity floors (parity unpinned: the paper's Fig. 2 values are not available)
    assert q["efficiency"] >= 0.95 and q["clone_rate"] <= 0.10 and q["fake_rate"] <= 0.02


def test_sectors_are_independent():
    """sector tracking works per sector; running a sector alone gives the
    same tracks as running it inside the full frame (the basis of sharding)."""
    cl, _, _ = dg.generate(dg.preset("C2", tracks_per_event=600, seed=9))
    full = oracle.run(cl, n_threads=4)
    one = oracle.run(cl, sector_lo=7, sector_hi=8)
    m = full.tracks["sector"] == 7
    assert m.sum() == one.n_tracks > 0
    a, b = full.tracks[m].copy(), one.tracks.copy()
    a["cluster_ofs"] = 0
    b["cluster_ofs"] = 0
    assert a.tobytes() == b.tobytes()
    single = oracle.run(cl, n_threads=1)
    assert single.tracks.tobytes() == full.tracks.tobytes()
    assert np.array_equal(single.cluster_ids, full.cluster_ids)


def test_selector_fixed_cap_variant_spends_the_budget_on_the_outer_rows():
    """SURVEY.md 8(f) variant (the rule before Phase I): with a fixed cap floor(f*nHits) the shared
    budget is spent where the walk starts, on the OUTER rows, and nothing is left for the inner
    ones; the Phase-I running fraction does the opposite.  Hand-computed expectation:
    tracklet A (rows 0..99) loses rows 90..99 and 0..9 to a better, short tracklet B."""
    rows = np.arange(0, 100)
    a = straight_tracklet(rows, 0)
    b = np.full(152, -1, dtype=np.int32)
    b[0:10] = a[0:10]
    b[90:100] = a[90:100]
    args = (np.stack([a, b]), [100, 20], [45.0 * 195, 0.0], [1, 2])      # Q_A = 100 - 2*45 = 10 < Q_B = 20
    running = oracle.select_only(*args, n_clusters=3000)
    t = running.tracks[running.tracks["seed_id"] == 1][0]
    # outer foreign rows refused (no budget yet); own rows 10..89; inner: (k)*1000 <= 100*(80+k) -> k <= 8
    assert (t["n_clusters"], t["n_shared"], t["row_first"], t["row_last"]) == (88, 8, 2, 89)
    fixed = oracle.select_only(*args, n_clusters=3000, params=oracle.default_params(shared_fixed_cap=1))
    t = fixed.tracks[fixed.tracks["seed_id"] == 1][0]
    # cap = floor(0.1*100) = 10, spent on rows 99..90; rows 9..0 refused
    assert (t["n_clusters"], t["n_shared"], t["row_first"], t["row_last"]) == (90, 10, 10, 99)
    assert running.n_tracks == fixed.n_tracks == 1                        # B: two 10-hit segments, below min_hits_track
