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


def _z_floor(z_ref):
    """What fp32 cannot represent at the frame's absolute z: the state's z is carried at time-frame
    coordinates (|z| up to ~7500 cm, ulp 4.9e-4 cm) and every row step rounds it there; 4 ulp(z) is
    the floor under which two fp32 evaluation orders cannot agree."""
    return 4.0 * np.spacing(np.abs(np.asarray(z_ref)).astype(np.float32)).astype(np.float64)


_SCALE = np.array([1.0, 1.0, 0.1, 0.1, 0.1])


def param_relerr(pa, pb):
    """|dp_i| / max(|p_i|, scale_i), scales (1 cm, 1 cm, 0.1, 0.1, 0.1 c/GeV); z: absolute error above
    the fp32 floor at that z, against a scale of 1 cm (offset-free)."""
    pa, pb = np.asarray(pa, dtype=np.float64), np.asarray(pb, dtype=np.float64)
    denom = np.maximum(np.abs(pb), _SCALE)
    denom[:, 1] = 1.0
    err = np.abs(pa - pb)
    err[:, 1] = np.maximum(0.0, err[:, 1] - _z_floor(pb[:, 1]))
    return err / denom


def compare_tracklets_fast(gi, o, rel=1e-3):
    """Fast mode at the tracklet level (needs TPC_KEEP_INTERMEDIATES): tracklets paired by
    (sector, seed id); where EVERY decision of the follower coincides (identical row_hit arrays in
    original ids) the fitted parameters must agree to `rel` -- fast mode may differ from the oracle
    through rounding only.  Returns statistics and the keys of the identical tracklets."""
    tl, rh = canonical_tracklets(gi)
    ot, orh = o.tracklets, o.row_hit
    kg = (tl["sector"].astype(np.int64) << 32) | tl["seed_id"].astype(np.int64)
    ko = (ot["sector"].astype(np.int64) << 32) | ot["seed_id"].astype(np.int64)
    common, ig, io = np.intersect1d(kg, ko, return_indices=True)
    out = {"n_gpu": len(tl), "n_oracle": len(ot), "n_paired": len(common)}
    a, b = tl[ig], ot[io]
    both = (a["n_hits"] > 0) & (b["n_hits"] > 0)
    out["n_accept_diff"] = int(((a["n_hits"] > 0) != (b["n_hits"] > 0)).sum())
    same = both & (rh[ig] == orh[io]).all(axis=1)
    out["n_both_accepted"] = int(both.sum())
    out["n_identical_hits"] = int(same.sum())
    relerr = param_relerr(a["p"][same], b["p"][same]) if same.any() else np.zeros((0, 5))
    out["n_param_bad"] = int((relerr > rel).any(axis=1).sum())
    out["max_rel_per_param"] = [float(v) for v in relerr.max(axis=0)] if len(relerr) else []
    # the same deviations in units of the parameter's own uncertainty (weakly constrained q/pT of
    # short tracklets: rounding scales with sigma, not with the value)
    if len(relerr):
        sig = np.sqrt(np.maximum(b["c"][same][:, [0, 2, 5, 9, 14]].astype(np.float64), 1e-30))
        err = np.abs(a["p"][same].astype(np.float64) - b["p"][same].astype(np.float64))
        err[:, 1] = np.maximum(0.0, err[:, 1] - _z_floor(b["p"][same][:, 1]))
        over = relerr > rel                      # only the entries beyond the relative bound
        out["max_err_in_sigma"] = float((err / sig)[over].max()) if over.any() else 0.0
    else:
        out["max_err_in_sigma"] = 0.0
    # the worst cases in full (for the record): parameter, error, value, its own uncertainty, hits
    diag = np.array([0, 2, 5, 9, 14])
    worst = []
    if len(relerr):
        bb = b[same]
        for k in np.argsort(-relerr.max(axis=1))[:8]:
            i = int(relerr[k].argmax())
            if relerr[k, i] <= rel:
                break
            worst.append({"param": i, "rel": float(relerr[k, i]), "value": float(bb["p"][k][i]),
                          "sigma": float(np.sqrt(max(bb["c"][k][diag[i]], 0.0))), "n_hits": int(bb["n_hits"][k]),
                          "sinphi": float(bb["p"][k][2]), "rows": [int(bb["row_first"][k]), int(bb["row_last"][k])]})
    out["worst"] = worst
    chi = np.abs(a["chi2"][same].astype(np.float64) - b["chi2"][same]) / np.maximum(np.abs(b["chi2"][same]), 1.0)
    out["max_rel_chi2"] = float(chi.max()) if len(chi) else 0.0
    return out, set(common[same].tolist())


def compare_tracks_fast(g_tracks, g_ids, g_shared, o, rel=1e-3, identical_tracklets=None):
    """Fast-mode comparison (north star): tracks paired by (sector, seed id, segment), falling
    back to >= 90 % cluster overlap; on the key pairs |dp_i| <= rel*max(|p_i|, scale_i), scales
    (1 cm, 1 cm, 0.1, 0.1, 0.1 c/GeV), z as in param_relerr.  n_param_bad counts key pairs with
    IDENTICAL cluster lists (and, when identical_tracklets is given, whose tracklet took the same
    decisions on every row) whose parameters differ by more than rel.  Returns a dict of
    statistics (n_paired = key pairs + overlap pairs)."""
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
    def relerr_of(a, b):
        return param_relerr(a["p"], b["p"])
    out.update(n_param_bad=0, n_list_diff=0, max_rel=0.0, n_param_bad_overlap=0, max_rel_overlap=0.0,
               n_param_bad_any_list=0)
    if len(common):
        a, b = tr[ig], otr[io]
        relerr = relerr_of(a, b)
        # identical cluster LISTS (ids and shared flags, not just their counts)
        same_list = (a["n_clusters"] == b["n_clusters"]) & (a["n_shared"] == b["n_shared"])
        g_ofs = np.cumsum(tr["n_clusters"].astype(np.int64)) - tr["n_clusters"].astype(np.int64)
        o_ofs = np.cumsum(otr["n_clusters"].astype(np.int64)) - otr["n_clusters"].astype(np.int64)
        cand = np.flatnonzero(same_list)
        if len(cand):
            n_per = a["n_clusters"][cand].astype(np.int64)
            within = np.arange(int(n_per.sum()), dtype=np.int64) - np.repeat(np.cumsum(n_per) - n_per, n_per)
            gg = np.repeat(g_ofs[ig[cand]], n_per) + within
            oo = np.repeat(o_ofs[io[cand]], n_per) + within
            diff = (ids[gg] != oids[oo]) | (sh[gg] != osh[oo])
            n_diff = np.add.reduceat(diff.astype(np.int64), np.cumsum(n_per) - n_per)
            same_list[cand[n_diff > 0]] = False
        out["n_list_diff"] = int((~same_list).sum())
        if identical_tracklets is not None:      # only tracks whose tracklet made the same decisions everywhere
            tk = (a["sector"].astype(np.int64) << 32) | a["seed_id"].astype(np.int64)
            same_list &= np.fromiter((int(k) in identical_tracklets for k in tk), dtype=bool, count=len(tk))
            out["n_identical_tracklet_and_list"] = int(same_list.sum())
        out["n_param_bad"] = int(((relerr > rel).any(axis=1) & same_list).sum())
        out["n_param_bad_any_list"] = int((relerr > rel).any(axis=1).sum())
        out["max_rel"] = float(relerr[same_list].max()) if same_list.any() else 0.0
        out["max_rel_per_param"] = [float(v) for v in relerr[same_list].max(axis=0)] if same_list.any() else []
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
