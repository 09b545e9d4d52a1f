"""Pins of the Phase-II track rebuild oracle (reading R11; section 3): hand-built cases on
radial straight tracks (every prediction is exactly on the track, the interpolation's variance is
~12 % of V in the middle of 60 clusters: two three-parameter fits of 30 clusters each), and invariants on a real frame."""
import numpy as np

import oracle
from oracle import merging, rebuild

R = 152
Z0 = 100.0


def frame(recs):
    """recs: (sector, row, y, z) in input order"""
    c = np.zeros(len(recs), dtype=oracle.CLUSTER_DTYPE)
    a = np.array(recs, dtype=np.float64)
    c["sector"], c["row"], c["y"], c["z"] = a[:, 0], a[:, 1], a[:, 2], a[:, 3]
    return c


def one_segment_tracks(cl, lists, rows):
    """Fabricated merged tracks: one segment each, `lists[k]` = original cluster ids (ascending rows),
    rows[k] = (first, last).  Returns what rebuild.rebuild needs."""
    n = len(lists)
    tracks = np.zeros(n, dtype=oracle.TRACK_DTYPE)
    fit = np.zeros(n, dtype=oracle.FIT_DTYPE)
    merged = np.zeros(n, dtype=merging.MERGED_DTYPE)
    ids = []
    for k, (l, (f, la)) in enumerate(zip(lists, rows)):
        tracks[k]["sector"], tracks[k]["row_first"], tracks[k]["row_last"] = cl["sector"][l[0]], f, la
        tracks[k]["seed_id"], tracks[k]["n_clusters"] = l[0], len(l)
        merged[k] = (k, 1, len(l), 0, len(ids), k, f, la, cl["sector"][l[0]], cl["sector"][l[0]])
        ids += list(l)
    return tracks, fit, merged, np.arange(n, dtype=np.uint32), np.asarray(ids, dtype=np.uint32)


def test_additional_attachment_and_candidate_lists():
    """A radial straight track on rows 20..80 whose ORIGINAL list lacks its clusters on rows 40..42
    (they are in the frame): the rebuild attaches them again ("allowing additional attachment during
    the fit").  Row 50 also holds decoys: with W ~ 0.12 V the candidate chi2 is d^2/(1.12 V):
      (0.20, z0+0.20): 7.1;  (0.35, z0): 10.9;  (0.45, z0): 18.1 > 16: no candidate; own cluster: 0.
    Expected candidates of row 50, in order: own, first decoy, second decoy; attached: own."""
    rows = list(range(20, 81))
    recs = [(0, r, 0.0, Z0) for r in rows]
    decoys = [(0, 50, 0.20, Z0 + 0.20), (0, 50, 0.35, Z0), (0, 50, 0.45, Z0)]
    cl = frame(decoys + recs)
    own = {r: 3 + i for i, r in enumerate(rows)}
    lst = [own[r] for r in rows if r not in (40, 41, 42)]
    tracks, fit, merged, seg, ids = one_segment_tracks(cl, [lst], [(20, 80)])
    r = rebuild.rebuild(cl, tracks, fit, merged, seg, ids)
    assert r.fit["flags"][0] == 0 and len(r.attached) == 61
    assert r.attached.tolist() == [own[x] for x in rows]            # rows 40..42 are back
    assert r.shared.sum() == 0 and r.used.all() and r.fit["n_used"][0] == 61
    k50 = 50 - 20
    assert r.cand_id[k50].tolist() == [own[50], 0, 1]
    assert r.cand_chi2[k50][0] < 1e-3 and 6.8 < r.cand_chi2[k50][1] < 7.6 and 10.4 < r.cand_chi2[k50][2] < 11.5
    other = np.delete(np.arange(61), k50)
    assert (r.cand_id[other, 1] == -1).all()                        # one candidate on every other row
    assert abs(r.fit["p"][0][0]) < 1e-3 and abs(r.fit["p"][0][1] - Z0) < 1e-3 and r.fit["chi2"][0] < 1e-2


def test_best_candidate_goes_to_the_better_track_the_other_takes_its_second():
    """"tracks failing to get their best candidate attached are still eligible for the
    second candidate".  Tracks A (y = 0, rows 20..80, 60 clusters) and B (y = 0.3, rows 30..70, 40
    clusters), both without a cluster of their own on row 50, which holds c1 at y = 0.15 (0.15 from
    both: chi2 2.0) and c2 at y = 0.5 (0.2 from B: chi2 3.6; 0.5 from A: no candidate).  A is longer
    (Q = 60 > 40): round 1 gives c1 to A; B moves on and gets c2 in round 2, OWNED (not shared).
    Without c2, B takes c1 as SHARED (budget: 1*1000 <= 100*(20+1))."""
    ra, rb = [r for r in range(20, 81) if r != 50], [r for r in range(30, 71) if r != 50]
    for with_c2 in (True, False):
        extra = [(0, 50, 0.15, Z0)] + ([(0, 50, 0.5, Z0)] if with_c2 else [])
        recs = extra + [(0, r, 0.0, Z0) for r in ra] + [(0, r, 0.3, Z0) for r in rb]
        cl = frame(recs)
        ne = len(extra)
        la, lb = list(range(ne, ne + len(ra))), list(range(ne + len(ra), ne + len(ra) + len(rb)))
        tracks, fit, merged, seg, ids = one_segment_tracks(cl, [la, lb], [(20, 80), (30, 70)])
        r = rebuild.rebuild(cl, tracks, fit, merged, seg, ids)
        ka, kb = 50 - 20, int(r.step_ofs[1]) + 50 - 30
        assert r.cand_id[ka].tolist()[:1] == [0] and r.attached[ka] == 0 and r.shared[ka] == 0
        if with_c2:
            assert r.cand_id[kb].tolist() == [0, 1, -1]
            assert r.attached[kb] == 1 and r.shared[kb] == 0
        else:
            assert r.cand_id[kb].tolist() == [0, -1, -1]
            assert r.attached[kb] == 0 and r.shared[kb] == 1
        assert (r.fit["flags"] == 0).all()


def test_plain_cut_of_the_third_iteration():
    """"a simple chi2 cut for final cluster rejection without interpolation".  A cluster
    0.36 cm off on row 50 (its own being absent; the road is 3.5*sqrt(1.12 V) = 0.37 cm) is a candidate
    (chi2 ~ 11.6 <= 16) and gets attached; in pass 3 its chi2 against the one-sided prediction (variance ~0.35 V) is ~9.6: used with the default cut of 16,
    dropped (attached, not used, no pull on the fit) with final_chi2_max = 8."""
    rows = [r for r in range(20, 81) if r != 50]
    cl = frame([(0, 50, 0.36, Z0)] + [(0, r, 0.0, Z0) for r in rows])
    tracks, fit, merged, seg, ids = one_segment_tracks(cl, [list(range(1, 61))], [(20, 80)])
    r = rebuild.rebuild(cl, tracks, fit, merged, seg, ids)
    k = 50 - 20
    assert r.attached[k] == 0 and r.used[k] == 1 and 10.8 < r.cand_chi2[k][0] < 12.4 and r.fit["n_used"][0] == 61
    # the road is part of the candidate definition: at 0.38 cm (chi2 12.9 <= 16, but beyond the 0.37 cm road)
    # the cluster is no candidate
    cl2 = cl.copy()
    cl2["y"][0] = 0.38
    r = rebuild.rebuild(cl2, tracks, fit, merged, seg, ids)
    assert r.cand_id[k].tolist() == [-1, -1, -1] and r.attached[k] == -1 and r.fit["n_used"][0] == 60
    r = rebuild.rebuild(cl, tracks, fit, merged, seg, ids, rparams=rebuild.default_rebuild_params(final_chi2_max=8.0))
    assert r.attached[k] == 0 and r.used[k] == 0 and r.fit["n_used"][0] == 60 and r.fit["n_attached"][0] == 61
    assert abs(r.fit["p"][0][0]) < 1e-4 and r.fit["chi2"][0] < 1e-3


def test_rebuild_invariants_on_a_frame():
    """C2-like frame through the whole chain: candidate lists are sorted by (chi2, id) and below the
    cut, lie on the step's (sector, row); an OWNED cluster belongs to one track only; the shared budget
    holds on every prefix from the outermost step; used <= attached; nearly all original clusters come
    back to their track."""
    from paper_2601_20569_b200 import datagen as dg
    cl, _, _ = dg.generate(dg.preset("C2", tracks_per_event=2500, seed=14))
    o = oracle.run(cl, n_threads=4, want=("tracks",))
    m = merging.merge(cl, o.tracks, o.cluster_ids, o.cluster_shared)
    r = rebuild.rebuild(cl, o.tracks, m.fit, m.merged, m.seg_index, m.cluster_ids)
    have = r.cand_id >= 0
    assert (have[:, 0] >= have[:, 1]).all() and (have[:, 1] >= have[:, 2]).all()
    assert (r.cand_chi2[have] <= 16.0).all()
    c = r.cand_chi2
    two = have[:, 1]
    assert ((c[two, 0] < c[two, 1]) | ((c[two, 0] == c[two, 1]) & (r.cand_id[two, 0] < r.cand_id[two, 1]))).all()
    owned = r.attached[(r.attached >= 0) & (r.shared == 0)]
    assert len(np.unique(owned)) == len(owned)
    assert (r.used <= (r.attached >= 0)).all()
    n_back = 0
    for k, mt in enumerate(m.merged):
        s0, s1 = int(r.step_ofs[k]), int(r.step_ofs[k + 1])
        att, sh = r.attached[s0:s1], r.shared[s0:s1]
        # steps are (sector,row) of the path: the attached cluster sits on the step's row
        got = att >= 0
        # budget on every prefix from the outermost step
        n_acc = np.cumsum(got[::-1])
        n_sh = np.cumsum(sh[::-1])
        assert (n_sh * 1000 <= 100 * np.maximum(n_acc, 1)).all()
        ids = set(m.cluster_ids[int(mt["cluster_ofs"]):int(mt["cluster_ofs"]) + int(mt["n_clusters"])].tolist())
        n_back += len(ids & set(att[got].tolist()))
        segs = r.segs[r.seg_ofs[k]:r.seg_ofs[k + 1]]
        if len(segs) == 1:
            assert (cl["row"][att[got]] == (np.arange(s1 - s0) + segs[0]["row_first"])[got]).all()
            assert (cl["sector"][att[got]] == segs[0]["sector"]).all()
    assert n_back >= 0.995 * len(m.cluster_ids)
    assert (r.fit["flags"] == 0).mean() > 0.98
