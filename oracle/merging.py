"""R9 track merging of the CPU ORACLE (TEST INFRASTRUCTURE): PAPER.md:29 (section 2: in-sector,
adjacent sectors, central electrode) on top of the sector-track refit R8.  The
matching itself is oracle/tpc_merge_oracle.cpp; this module prepares its input from an oracle
result and assembles the chains (pure bookkeeping)."""
from __future__ import annotations

import ctypes as C

import numpy as np

import oracle

MERGE_TRACK_DTYPE = np.dtype(
    [("sector", "<i4"), ("row_first", "<i4"), ("row_last", "<i4"), ("valid", "<i4"), ("seed_id", "<u4"),
     ("segment", "<i4"), ("iter", "<i4"), ("p_in", "<f4", (5,)), ("c_in", "<f4", (15,)), ("p_out", "<f4", (5,)),
     ("c_out", "<f4", (15,))])
MERGED_DTYPE = np.dtype(
    [("head", "<u4"), ("n_segments", "<u4"), ("n_clusters", "<u4"), ("n_shared", "<u4"), ("cluster_ofs", "<u4"),
     ("seg_ofs", "<u4"), ("row_first", "<i4"), ("row_last", "<i4"), ("sector_first", "<i4"), ("sector_last", "<i4")])


class MergeParams(C.Structure):
    _fields_ = [("gap_in_sector", C.c_int32), ("gap_adjacent_back", C.c_int32), ("gap_adjacent", C.c_int32),
                ("gap_ce", C.c_int32), ("chi2_max", C.c_float), ("sys", C.c_float * 5), ("ce_sys_z", C.c_float),
                ("pre_dy", C.c_float), ("pre_dz", C.c_float), ("pre_coarse_dz", C.c_float), ("stages", C.c_int32)]


def _lib():
    L = oracle.lib()
    if not getattr(L, "_merge_ready", False):
        vp = C.c_void_p
        L.orc_merge_default_params.argtypes = [C.POINTER(MergeParams)]
        L.orc_merge_links.restype = C.c_int
        L.orc_merge_links.argtypes = [C.POINTER(oracle.Geom), C.POINTER(oracle.Params), C.POINTER(MergeParams), vp,
                                      C.c_int32, vp, vp, vp]
        L.orc_merge_rotate.restype = C.c_int
        L.orc_merge_rotate.argtypes = [C.POINTER(oracle.Geom), vp, vp, C.c_int, C.c_float]
        L._merge_ready = True
    return L


def default_merge_params(**kw) -> MergeParams:
    m = MergeParams()
    _lib().orc_merge_default_params(C.byref(m))
    for k, v in kw.items():
        if k == "sys":
            for i in range(5):
                m.sys[i] = v[i]
        else:
            setattr(m, k, v)
    return m


def merge_tracks_input(tracks: np.ndarray, fit: np.ndarray) -> np.ndarray:
    """The merging's view of every sector track: descriptor + the two R8 end states."""
    t = np.zeros(len(tracks), dtype=MERGE_TRACK_DTYPE)
    for f in ("sector", "row_first", "row_last", "seed_id", "segment"):
        t[f] = tracks[f]
    t["iter"] = (tracks["flags"].astype(np.int64) >> 1) & 1
    t["valid"] = (fit["flags"] == 0).astype(np.int32)
    t["p_in"], t["c_in"], t["p_out"], t["c_out"] = fit["p"], fit["c"], fit["p_out"], fit["c_out"]
    return t


def links(mt: np.ndarray, geom=None, params=None, mparams=None):
    """(next, prev, link_chi2) of the three merging stages."""
    geom = geom or oracle.default_geom()
    params = params or oracle.default_params()
    mparams = mparams or default_merge_params()
    mt = np.ascontiguousarray(mt)
    n = len(mt)
    nxt = np.full(n, -1, dtype=np.int32)
    prv = np.full(n, -1, dtype=np.int32)
    chi = np.zeros(n, dtype=np.float32)
    rc = _lib().orc_merge_links(C.byref(geom), C.byref(params), C.byref(mparams), mt.ctypes.data, n, nxt.ctypes.data,
                                prv.ctypes.data, chi.ctypes.data)
    if rc < 0:
        raise ValueError("oracle merge: bad argument")
    return nxt, prv, chi


def assemble(tracks, cluster_ids, cluster_shared, nxt, prv):
    """Chains -> merged tracks.  Heads (prev < 0) in the order of `tracks`; the cluster list of a
    merged track is the concatenation of its segments' lists in chain order (ascending rows inside
    a sector).  Returns (merged[MERGED_DTYPE], seg_index, merged_ids, merged_shared)."""
    heads = np.flatnonzero(prv < 0)
    merged = np.zeros(len(heads), dtype=MERGED_DTYPE)
    seg, ids, sh = [], [], []
    n_ids = 0
    for m, h in enumerate(heads):
        k, first = int(h), len(seg)
        nc = ns = 0
        while k >= 0:
            seg.append(k)
            o, n = int(tracks["cluster_ofs"][k]), int(tracks["n_clusters"][k])
            ids.append(cluster_ids[o:o + n])
            sh.append(cluster_shared[o:o + n])
            nc += n
            ns += int(tracks["n_shared"][k])
            last = k
            k = int(nxt[k])
        merged[m] = (h, len(seg) - first, nc, ns, n_ids, first, tracks["row_first"][h], tracks["row_last"][last],
                     tracks["sector"][h], tracks["sector"][last])
        n_ids += nc
    cat = lambda parts, dt: np.concatenate(parts).astype(dt) if parts else np.zeros(0, dtype=dt)
    return merged, np.asarray(seg, dtype=np.uint32), cat(ids, np.uint32), cat(sh, np.uint8)


class MergeResult:
    pass


def merge(clusters, tracks, cluster_ids, cluster_shared, geom=None, params=None, mparams=None) -> MergeResult:
    """R8 + R9 on the tracks of an oracle result."""
    r = MergeResult()
    r.fit = oracle.refit_tracks(clusters, tracks, cluster_ids, geom, params)
    r.input = merge_tracks_input(tracks, r.fit)
    r.next, r.prev, r.link_chi2 = links(r.input, geom, params, mparams)
    r.merged, r.seg_index, r.cluster_ids, r.cluster_shared = assemble(tracks, cluster_ids, cluster_shared, r.next, r.prev)
    return r


def rotate(state20, x, sign, geom=None, max_sinphi=0.95):
    geom = geom or oracle.default_geom()
    st = np.array(state20, dtype=np.float32, copy=True)
    xx = C.c_float(x)
    ok = _lib().orc_merge_rotate(C.byref(geom), st.ctypes.data, C.addressof(xx), sign, max_sinphi)
    return bool(ok), st, float(xx.value)
