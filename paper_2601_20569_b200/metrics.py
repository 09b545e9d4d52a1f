"""Track-finding quality metrics against the generator's MC labels (evaluation only).

Definitions after PAPER.md:63 (Fig. 2 caption: efficiency, clone rate, fake rate; a track is
findable with >= 70 TPC hits) as concretised in DESIGN.md "Metrics".  The same function is
applied to the output of the CUDA path and to the output of the oracle; it contains none of
the tracking method's arithmetic and imports neither side.

label per cluster = particle*8 + leg (every leg of a looper is its own particle for matching,
PAPER.md:57 "one track per leg"); noise = -1.
"""
from __future__ import annotations

import numpy as np


FINDABLE_MIN_HITS = 70   # findable = at least 70 hits in the TPC


def track_quality(n_clusters_per_track, cluster_ofs, cluster_ids, track_sector, labels,
                  min_findable: int = FINDABLE_MIN_HITS, purity: float = 0.9) -> dict:
    """Efficiency / clone rate / fake rate.

    n_clusters_per_track, cluster_ofs, track_sector: per-track arrays; cluster_ids: the
    concatenated original cluster indices; labels: per input cluster.
    """
    labels = np.asarray(labels)
    nt = len(n_clusters_per_track)
    lab_all, cnt_all = np.unique(labels[labels >= 0], return_counts=True)
    findable = lab_all[cnt_all >= min_findable]
    out = {"n_tracks": int(nt), "n_findable": int(len(findable))}
    if nt == 0:
        out.update(efficiency=0.0, clone_rate=0.0, fake_rate=0.0, n_matched=0, n_fake=0, n_found=0)
        return out
    n_per = np.asarray(n_clusters_per_track, dtype=np.int64)
    ofs = np.asarray(cluster_ofs, dtype=np.int64)
    # expand (track, label) pairs
    tr_idx = np.repeat(np.arange(nt, dtype=np.int64), n_per)
    within = np.arange(n_per.sum(), dtype=np.int64) - np.repeat(np.cumsum(n_per) - n_per, n_per)
    lab = labels[np.asarray(cluster_ids)[np.repeat(ofs, n_per) + within]].astype(np.int64)
    order = np.lexsort((lab, tr_idx))
    tr_s, lab_s = tr_idx[order], lab[order]
    new_run = np.ones(len(tr_s), dtype=bool)
    new_run[1:] = (tr_s[1:] != tr_s[:-1]) | (lab_s[1:] != lab_s[:-1])
    run_start = np.flatnonzero(new_run)
    run_len = np.diff(np.append(run_start, len(tr_s)))
    run_tr, run_lab = tr_s[run_start], lab_s[run_start]
    # majority label per track (largest run; ties -> smaller label)
    best_len = np.zeros(nt, dtype=np.int64)
    np.maximum.at(best_len, run_tr, run_len)
    is_best = run_len == best_len[run_tr]
    best_lab = np.full(nt, np.iinfo(np.int64).max)
    np.minimum.at(best_lab, run_tr[is_best], run_lab[is_best])
    matched = (best_lab >= 0) & (best_len >= purity * n_per)
    n_matched = int(matched.sum())
    m_lab = best_lab[matched]
    m_sec = np.asarray(track_sector, dtype=np.int64)[matched]
    distinct = len(np.unique(m_lab * 64 + m_sec)) if n_matched else 0
    found = np.intersect1d(np.unique(m_lab), findable)
    out.update(
        efficiency=float(len(found) / len(findable)) if len(findable) else 0.0,
        clone_rate=float((n_matched - distinct) / n_matched) if n_matched else 0.0,
        fake_rate=float((nt - n_matched) / nt),
        n_matched=n_matched, n_fake=int(nt - n_matched), n_found=int(len(found)))
    return out
