"""CPU ORACLE of the second seeding iteration on leftover clusters (TEST INFRASTRUCTURE, see
oracle/tpc_oracle.h for who may use it).

Passage followed: PAPER.md:67 (section 3, Phase III): "... the seeding ... in multiple iterations
on the leftover clusters after ambiguity solving".  The paper says no more; reading R7
fixes it, and this module follows R7 step by step with the single-iteration oracle (``run``,
R0..R6) as the library routine of each step:

  R7.1  used = every cluster that appears in a cluster list of an iteration-1 track (accepted as
        owned or as shared).
  R7.2  leftover frame = the input records that are not used, in input order (records that were
        ignored or dropped in iteration 1 stay in it and are ignored or dropped again).
  R7.3  R1..R6 on the leftover frame, same geometry and parameters.
  R7.4  iteration-2 results re-expressed in ORIGINAL input indices (the index map of R7.2 is
        strictly increasing, so every tie-break on the original index, rule D2, is the same in
        both index spaces); output = iteration-1 tracks followed by iteration-2 tracks, the latter
        with flag bit TRACK_ITER2.

Pins (tests/test_oracle_second_iteration.py): a noise-free isolated track leaves nothing to a
second iteration; iteration-2 tracks use leftover clusters only; the result equals a by-hand
composition on a frame whose leftover is known by construction; attached clusters never decrease.
"""
from __future__ import annotations

import numpy as np

from . import TRACK_DTYPE, run

TRACK_ITER2 = 2   # tpc_track.flags bit 1


class TwoIterations:
    """Tracks, cluster ids and shared flags of both iterations, in original cluster indices."""

    def __init__(self, first, second, left_ids):
        self.first, self.second, self.left_ids = first, second, left_ids
        t2 = second.tracks.copy()
        t2["seed_id"] = left_ids[t2["seed_id"]] if len(t2) else t2["seed_id"]
        t2["cluster_ofs"] = t2["cluster_ofs"] + np.uint32(first.n_cluster_ids)
        t2["flags"] = t2["flags"] | TRACK_ITER2
        ids2 = left_ids[second.cluster_ids] if second.n_cluster_ids else second.cluster_ids
        self.tracks = np.concatenate([first.tracks, t2]).astype(TRACK_DTYPE)
        self.cluster_ids = np.concatenate([first.cluster_ids, ids2]).astype(np.uint32)
        self.cluster_shared = np.concatenate([first.cluster_shared, second.cluster_shared]).astype(np.uint8)
        self.n_tracks = len(self.tracks)
        self.n_cluster_ids = len(self.cluster_ids)
        self.n_tracks_first = first.n_tracks
        self.n_clusters = first.n_clusters
        self.n_leftover = len(left_ids)


def run_two_iterations(clusters: np.ndarray, geom=None, params=None, n_threads: int = 1) -> TwoIterations:
    first = run(clusters, geom=geom, params=params, n_threads=n_threads, want=("tracks",))          # R1..R6
    used = np.zeros(len(clusters), dtype=bool)
    used[first.cluster_ids] = True                                                                  # R7.1
    left_ids = np.flatnonzero(~used).astype(np.uint32)                                              # R7.2
    second = run(np.ascontiguousarray(clusters[left_ids]), geom=geom, params=params, n_threads=n_threads,
                 want=("tracks",))                                                                  # R7.3
    return TwoIterations(first, second, left_ids)                                                   # R7.4
