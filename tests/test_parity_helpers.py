"""The comparison helpers of oracle/parity.py themselves (host logic, no GPU)."""
import numpy as np

import oracle
from oracle import parity
from paper_2601_20569_b200 import datagen as dg


def _as_gpu_tracks(o):
    from paper_2601_20569_b200.binding import TRACK_DTYPE
    t = np.zeros(len(o.tracks), dtype=TRACK_DTYPE)
    for f in t.dtype.names:
        if f in o.tracks.dtype.names:
            t[f] = o.tracks[f]
    return t


def test_compare_tracks_fast_pairs_by_key_then_by_cluster_overlap():
    cl, _, _ = dg.generate(dg.preset("C1"))
    o = oracle.run(cl, want=("tracks",))
    t = _as_gpu_tracks(o)
    st = parity.compare_tracks_fast(t, o.cluster_ids, o.cluster_shared, o)
    assert st["n_paired_key"] == st["n_oracle"] == len(t) and st["n_paired_overlap"] == 0
    assert st["n_param_bad"] == 0 and st["n_list_diff"] == 0 and st["max_rel"] == 0.0
    # another clone instance won: same clusters, different seed id -> paired by overlap
    t2 = t.copy()
    t2["seed_id"][:7] = 0xFFFFFF00 - np.arange(7)
    st = parity.compare_tracks_fast(t2, o.cluster_ids, o.cluster_shared, o)
    assert st["n_paired_key"] == len(t) - 7 and st["n_paired_overlap"] == 7 and st["n_paired"] == len(t)
    # a track with other clusters is not paired; a parameter off by 1 % is flagged
    ids = o.cluster_ids.copy()
    k = int(t2["cluster_ofs"][0])
    ids[k:k + int(t2["n_clusters"][0])] = np.setdiff1d(np.arange(len(cl)), o.cluster_ids)[: int(t2["n_clusters"][0])]
    t2["p"][10, 4] *= 1.01
    st = parity.compare_tracks_fast(t2, ids, o.cluster_shared, o)
    assert st["n_paired"] == len(t) - 1 and st["n_param_bad"] == 1


def test_canonical_tracklets_ignores_rows_outside_the_tracklet():
    from paper_2601_20569_b200.binding import TRACKLET_DTYPE
    tl = np.zeros(2, dtype=TRACKLET_DTYPE)
    tl["n_hits"] = [12, 0]
    tl["row_first"] = [3, 0]
    tl["row_last"] = [5, 9]
    tl["seed_id"] = [7, 9]
    rh = np.full((2, 152), 123456789, dtype=np.int32)      # stale workspace content
    rh[0, 3:6] = [2, -1, 0]
    gi = dict(tracklets=tl, row_hit=rh, orig_id=np.array([40, 41, 42], dtype=np.uint32))
    t, r = parity.canonical_tracklets(gi)
    assert (r[0, 3:6] == [42, -1, 40]).all() and (np.delete(r[0], [3, 4, 5]) == -1).all() and (r[1] == -1).all()
