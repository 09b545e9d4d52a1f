"""Pins of the oracle's second seeding iteration (reading R7)."""
import numpy as np

import oracle
from oracle import second_iteration as si
from paper_2601_20569_b200 import datagen as dg


def test_isolated_noise_free_track_leaves_nothing():
    cfg = dg.preset("C1", tracks_per_event=1, noise_frac=0.0, smear_y=0.0, smear_z=0.0, p_hit=1.0, seed=11,
                    pt_lo=1.0, pt_hi=1.1)
    cl, _, _ = dg.generate(cfg)
    r = si.run_two_iterations(cl)
    assert r.first.n_tracks == 1 and r.second.n_tracks == 0
    assert r.n_leftover == len(cl) - r.first.n_cluster_ids


def test_second_iteration_uses_leftover_clusters_only_and_adds_tracks():
    cl, _, _ = dg.generate(dg.preset("C5", tracks_per_event=6000))
    p = oracle.default_params(err_y=0.15, err_z=0.15, nf_max_d2=1.6)
    r = si.run_two_iterations(cl, params=p, n_threads=4)
    n1 = r.first.n_cluster_ids
    used1 = np.zeros(len(cl), dtype=bool)
    used1[r.cluster_ids[:n1]] = True
    ids2 = r.cluster_ids[n1:]
    assert r.second.n_tracks > 0                      # dense inner rows: the first pass leaves tracks behind
    assert not used1[ids2].any()                      # R7.1/R7.2: disjoint from everything attached before
    t2 = r.tracks[r.n_tracks_first:]
    assert (t2["flags"] & si.TRACK_ITER2).all() and not (r.tracks[:r.n_tracks_first]["flags"] & si.TRACK_ITER2).any()
    # cluster lists of the second iteration: ascending rows, ids inside the frame, offsets contiguous
    assert int(t2["cluster_ofs"][0]) == n1
    assert (np.diff(t2["cluster_ofs"].astype(np.int64)) == t2["n_clusters"][:-1]).all()
    for t in t2[:50]:
        ids = r.cluster_ids[t["cluster_ofs"]: t["cluster_ofs"] + t["n_clusters"]]
        rows = cl["row"][ids].astype(int)
        assert (np.diff(rows) > 0).all() and (cl["sector"][ids] == t["sector"]).all()
    assert len(np.unique(r.cluster_ids)) >= len(np.unique(r.cluster_ids[:n1]))   # attached clusters never decrease


def test_equals_by_hand_composition_on_a_frame_with_known_leftover():
    """Two copies of a track pattern on top of each other in different sectors are independent;
    removing by hand the clusters iteration 1 attached in sector 0 and running the one-iteration
    oracle on the rest must give exactly the iteration-2 tracks of that sector."""
    cl, _, _ = dg.generate(dg.preset("C2", tracks_per_event=2500, seed=5))
    cl = cl[cl["sector"] < 2]
    r = si.run_two_iterations(cl)
    first = oracle.run(cl, want=("tracks",))
    keep = np.ones(len(cl), dtype=bool)
    keep[first.cluster_ids] = False
    sel = np.flatnonzero(keep & (cl["sector"] == 0))
    by_hand = oracle.run(np.ascontiguousarray(cl[sel]), want=("tracks",))
    t2 = r.tracks[r.n_tracks_first:]
    t2 = t2[t2["sector"] == 0]
    assert len(t2) == by_hand.n_tracks
    a = np.sort(sel[by_hand.tracks["seed_id"]])
    b = np.sort(t2["seed_id"])
    assert (a == b).all()
