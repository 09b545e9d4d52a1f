"""Element-by-element comparison of a CUDA-path result with an oracle result (TEST
INFRASTRUCTURE, used by tests/, __graft_entry__.smoke() and bench.py's parity sample).

Takes plain numpy arrays from both sides (it imports neither the product nor the oracle
library).  Everything is compared in ORIGINAL cluster indices (rule D3) and in canonical order
(rule D4: tracklets by (sector, seed id), tracks by (sector, seed id, segment)) — the order in
which the library emits tracks is not part of the result.
"""
from __future__ import annotations

import numpy as np


def _bits(a):
    return np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)


def links_to_orig(link_sorted, orig_id, n_clusters):
    """GPU links live in sorted-index space; express them in original indices."""
    out = np.full(n_clusters, -1, dtype=np.int32)
    ok = link_sorted >= 0
    vals = np.full(len(link_sorted), -1, dtype=np.int32)
    vals[ok] = orig_id[link_sorted[ok]].astype(np.int32)
    out[orig_id] = vals
    return out


def compare_grid(gi, o, stable_order=True):
    """Bin index + sorted order.  Returns a dict of mismatch counts (all 0 = parity)."""
    bad = {}
    bad["n_sorted"] = int(gi["n_sorted"] != o.n_sorted)
    bad["n_bins"] = int(gi["n_bins"] != o.n_bins)
    if bad["n_sorted"] or bad["n_bins"]:
        return bad
    for f in ("ny", "nz", "bin_ofs", "clu_ofs", "count"):
        bad["row_desc." + f] = int((gi["row_desc"][f] != o.row_desc[f]).sum())
    nonempty = o.row_desc["count"] > 0
    for f in ("y0", "z0"):
        bad["row_desc." + f] = int((_bits(gi["row_desc"][f][nonempty]) != _bits(o.row_desc[f][nonempty])).sum())
    bad["bin_start"] = int((gi["bin_start"] != o.bin_start).sum())
    if stable_order:
        bad["orig_id"] = int((gi["orig_id"] != o.sorted_ids).sum())
    else:  # same id SET in every bin
        bs = o.bin_start.astype(np.int64)
        binno = np.repeat(np.arange(len(bs) - 1), np.diff(bs))
        a = np.lexsort((gi["orig_id"], binno))
        bad["orig_id"] = int((gi["orig_id"][a] != o.sorted_ids).sum())
    return bad


def compare_links(gi, o, n_clusters, sector_mask=None):
    bad = {}
    for k in ("link_up", "link_dn", "link_up2", "link_dn2"):
        g = links_to_orig(gi[k], gi["orig_id"], n_clusters)
        ref = getattr(o, k)
        if sector_mask is not None:
            g, ref = g[sector_mask], ref[sector_mask]
        bad[k] = int((g != ref).sum())
    return bad


def canonical_tracklets(gi):
    """GPU tracklets -> canonical order, row_hit in original ids restricted to the tracklet's
    row range, rejected tracklets blanked (the oracle blanks them too)."""
    tl = gi["tracklets"]
    rh = gi["row_hit"].copy()
    n_rows = rh.shape[1] if rh.ndim == 2 else 0
    if len(tl):
        rows = np.arange(n_rows)[None, :]
        inside = (rows >= tl["row_first"][:, None]) & (rows <= tl["row_last"][:, None]) & (tl["n_hits"][:, None] > 0)
        valid = inside & (rh >= 0)          # entries outside the row range are undefined (stale workspace)
        rh = np.where(valid, gi["orig_id"][np.where(valid, rh, 0)].astype(np.int64), -1).astype(np.int32)
    order = np.lexsort((tl["seed_id"], tl["sector"]))
    return tl[order], rh[order]


def compare_tracklets(gi, o, sector=None):
    bad = {}
    tl, rh = canonical_tracklets(gi)
    if sector is not None:
        m = tl["sector"] == sector
        tl, rh = tl[m], rh[m]
    bad["n_seeds"] = int(len(tl) != len(o.tracklets))
    if bad["n_seeds"]:
        bad["n_seeds"] = abs(len(tl) - len(o.tracklets))
        return bad
    ot = o.tracklets
    bad["seed_id"] = int((tl["seed_id"] != ot["seed_id"]).sum())
    bad["seed_len"] = int((tl["seed_len"].astype(np.int32) != o.seeds["len"]).sum())
    bad["n_hits"] = int((tl["n_hits"].astype(np.int32) != ot["n_hits"]).sum())
    keep = ot["n_hits"] > 0
    for f in ("row_first", "row_last", "sector"):
        bad[f] = int((tl[f].astype(np.int32)[keep] != ot[f][keep]).sum())
    for f in ("x", "p", "c", "chi2"):
        bad[f + "_bits"] = int((_bits(tl[f][keep]) != _bits(ot[f][keep])).sum())
    bad["row_hit"] = int((rh != o.row_hit).sum())
    return bad


def canonical_tracks(tracks, cluster_ids, cluster_shared):
    order = np.lexsort((tracks["segment"], tracks["seed_id"], tracks["sector"]))
    tr = tracks[order]
    n_per = tr["n_clusters"].astype(np.int64)
    ofs = tr["cluster_ofs"].astype(np.int64)
    within = np.arange(int(n_per.sum()), dtype=np.int64) - np.repeat(np.cumsum(n_per) - n_per, n_per)
    gather = np.repeat(ofs, n_per) + within
    return tr, np.asarray(cluster_ids)[gather], np.asarray(cluster_shared)[gather]


def compare_tracks(g_tracks, g_ids, g_shared, o, sector=None):
    """Deterministic-mode comparison of the final output (bit level)."""
    bad = {}
    if sector is not None:
        g_tracks = g_tracks[g_tracks["sector"] == sector]
    tr, ids, sh = canonical_tracks(g_tracks, g_ids, g_shared)
    otr, oids, osh = canonical_tracks(o.tracks, o.cluster_ids, o.cluster_shared)
    bad["n_tracks"] = abs(len(tr) - len(otr))
    if bad["n_tracks"]:
        return bad
    for f in ("seed_id", "n_clusters", "n_shared", "sector", "row_first", "row_last", "flags",
              "n_hits_tracklet", "segment"):
        bad[f] = int((tr[f].astype(np.int64) != otr[f].astype(np.int64)).sum())
    for f in ("x", "p", "c", "chi2"):
        bad[f + "_bits"] = int((_bits(tr[f]) != _bits(otr[f])).sum())
    bad["n_ids"] = abs(len(ids) - len(oids))
    if not bad["n_ids"]:
        bad["cluster_ids"] = int((ids != oids).sum())
        bad["cluster_shared"] = int((sh != osh).sum())
    return bad


def _overlap_pairs(tr, ids, otr, oids, un_g, un_o, n_clusters_total, frac=0.9):
    """Pair leftover tracks by cluster overlap: a GPU track and an oracle track are the same
    physical track if they share >= frac of the larger cluster list.  (Clone instances of one
    track collect the same clusters from different seeds; which instance wins the ambiguity
    solving is decided by a weight difference at rounding level, so in fast mode the winner's
    seed id may differ from the oracle's while the track is the same.)"""
    if len(un_g) == 0 or len(un_o) == 0:
        return np.zeros(0, dtype=np.int64), np.zeros(0, dtype=np.int64)
    og_ofs = np.cumsum(tr["n_clusters"].astype(np.int64)) - tr["n_clusters"].astype(np.int64)
    oo_ofs = np.cumsum(otr["n_clusters"].astype(np.int64)) - otr["n_clusters"].astype(np.int64)
    owner = np.full(n_clusters_total, -1, dtype=np.int64)      # cluster -> leftover oracle track
    for j in un_o:
        owner[oids[oo_ofs[j]:oo_ofs[j] + int(otr["n_clusters"][j])]] = j
    pg, po, used = [], [], set()
    for i in un_g:
        n = int(tr["n_clusters"][i])
        cand = owner[ids[og_ofs[i]:og_ofs[i] + n]]
        cand = cand[cand >= 0]
        if len(cand) == 0:
            continue
        vals, cnt = np.unique(cand, return_counts=True)
        j = int(vals[np.argmax(cnt)])
        if j in used or tr["sector"][i] != otr["sector"][j]:
            continue
        if cnt.max() >= frac * max(n, int(otr["n_clusters"][j])):
            pg.append(i); po.append(j); used.add(j)
    return np.asarray(pg, dtype=np.int64), np.asarray(po, dtype=np.int64)


def compare_tracks_fast(g_tracks, g_ids, g_shared, o, rel=1e-3):
    """Fast-mode comparison (north star): tracks paired by (sector, seed id, segment), falling
    back to >= 90 % cluster overlap; on the key pairs |dp_i| <= rel*max(|p_i|, scale_i), scales
    (1 cm, 1 cm, 0.1, 0.1, 0.1 c/GeV), z taken relative to the oracle track's z.  Returns a dict
    of statistics (n_paired = key pairs + overlap pairs)."""
    def keyof(t):
        return (t["sector"].astype(np.int64) << 40) | (t["seed_id"].astype(np.int64) << 8) | t["segment"].astype(np.int64)
    tr, ids, sh = canonical_tracks(g_tracks, g_ids, g_shared)
    otr, oids, osh = canonical_tracks(o.tracks, o.cluster_ids, o.cluster_shared)
    kg, ko = keyof(tr), keyof(otr)
    common, ig, io = np.intersect1d(kg, ko, return_indices=True)
    out = {"n_gpu": len(tr), "n_oracle": len(otr), "n_paired_key": len(common)}
    un_g = np.setdiff1d(np.arange(len(tr)), ig)
    un_o = np.setdiff1d(np.arange(len(otr)), io)
    pg, po = _overlap_pairs(tr, ids, otr, oids, un_g, un_o, o.n_clusters)
    out["n_paired_overlap"] = len(pg)
    out["n_paired"] = len(common) + len(pg)
    scale = np.array([1.0, 1.0, 0.1, 0.1, 0.1])

    def relerr_of(a, b):
        pa, pb = a["p"].astype(np.float64), b["p"].astype(np.float64)
        denom = np.maximum(np.abs(pb), scale)
        denom[:, 1] = 1.0  # z: relative to the track's own z (offset-free), scale 1 cm
        return np.abs(pa - pb) / denom
    out.update(n_param_bad=0, n_list_diff=0, max_rel=0.0, n_param_bad_overlap=0, max_rel_overlap=0.0)
    if len(common):
        a, b = tr[ig], otr[io]
        relerr = relerr_of(a, b)
        same_list = (a["n_clusters"] == b["n_clusters"]) & (a["n_shared"] == b["n_shared"])
        out["n_list_diff"] = int((~same_list).sum())
        out["n_param_bad"] = int(((relerr > rel).any(axis=1) & same_list).sum())
        out["max_rel"] = float(relerr[same_list].max()) if same_list.any() else 0.0
    if len(pg):
        a, b = tr[pg], otr[po]
        ok = (a["row_first"] == b["row_first"]) & (a["flags"] == 0) & (b["flags"] == 0)   # parameters at the same x
        if ok.any():
            relerr = relerr_of(a[ok], b[ok])
            out["n_param_bad_overlap"] = int((relerr > rel).any(axis=1).sum())
            out["max_rel_overlap"] = float(relerr.max())
    return out


def all_zero(bad: dict) -> bool:
    return all(v == 0 for v in bad.values())
