"""R11 Phase-II track rebuild, CPU ORACLE side (TEST INFRASTRUCTURE): PAPER.md:59,65 (section 3).  The
arithmetic is oracle/tpc_rebuild_oracle.cpp; this module lays out its input from a merged result."""
from __future__ import annotations

import ctypes as C

import numpy as np

import oracle

NCAND = 3
SEG_DTYPE = np.dtype([("sector", "<i4"), ("row_first", "<i4"), ("row_last", "<i4")])
REBUILD_FIT_DTYPE = np.dtype([("x", "<f4"), ("p", "<f4", (5,)), ("c", "<f4", (15,)), ("chi2", "<f4"), ("n_attached", "<i4"),
                              ("n_used", "<i4"), ("flags", "<u4")])


class RebuildParams(C.Structure):
    _fields_ = [("cand_chi2_max", C.c_float), ("final_chi2_max", C.c_float), ("min_clusters", C.c_int32), ("ce_var", C.c_float)]


def _lib():
    L = oracle.lib()
    if not getattr(L, "_rb_ready", False):
        vp = C.c_void_p
        L.orc_rebuild_default_params.argtypes = [C.POINTER(RebuildParams)]
        L.orc_rebuild_path_len.restype = C.c_int64
        L.orc_rebuild_path_len.argtypes = [vp, C.c_int32]
        L.orc_rebuild.restype = C.c_int
        L.orc_rebuild.argtypes = [C.POINTER(oracle.Geom), C.POINTER(oracle.Params), C.POINTER(RebuildParams), vp, C.c_uint64,
                                  C.c_int32] + [vp] * 18
        L._rb_ready = True
    return L


def default_rebuild_params(**kw) -> RebuildParams:
    r = RebuildParams()
    _lib().orc_rebuild_default_params(C.byref(r))
    for k, v in kw.items():
        setattr(r, k, v)
    return r


def track_key_id(tracks, heads):
    """Unique 64-bit id of a merged track = that of its head segment (sector, iteration, seed id, segment)."""
    h = np.asarray(heads, dtype=np.int64)
    it = (tracks["flags"][h].astype(np.uint64) >> np.uint64(1)) & np.uint64(1)
    return ((tracks["sector"][h].astype(np.uint64) << np.uint64(41)) | (it << np.uint64(40)) |
            (tracks["seed_id"][h].astype(np.uint64) << np.uint64(8)) | tracks["segment"][h].astype(np.uint64))


class RebuildResult:
    pass


def rebuild(clusters, tracks, refit, merged, seg_index, merged_ids, geom=None, params=None, rparams=None) -> RebuildResult:
    """R11 on the merged tracks of a frame."""
    geom = geom or oracle.default_geom()
    params = params or oracle.default_params()
    rparams = rparams or default_rebuild_params()
    L = _lib()
    nm = len(merged)
    seg_ofs = np.zeros(nm + 1, dtype=np.int32)
    seg_ofs[1:] = np.cumsum(merged["n_segments"])
    segs = np.zeros(int(seg_ofs[-1]), dtype=SEG_DTYPE)
    clu_ofs = np.zeros(nm + 1, dtype=np.int64)
    clu_ofs[1:] = np.cumsum(merged["n_clusters"].astype(np.int64))
    ids = np.zeros(int(clu_ofs[-1]), dtype=np.uint32)
    stq = np.zeros((nm, 3), dtype=np.float32)
    valid = np.zeros(nm, dtype=np.uint8)
    step_ofs = np.zeros(nm + 1, dtype=np.int64)
    for m, mt in enumerate(merged):
        sl = seg_index[int(mt["seg_ofs"]):int(mt["seg_ofs"]) + int(mt["n_segments"])].astype(np.int64)
        s = segs[seg_ofs[m]:seg_ofs[m + 1]]
        s["sector"], s["row_first"], s["row_last"] = tracks["sector"][sl], tracks["row_first"][sl], tracks["row_last"][sl]
        o, n = int(mt["cluster_ofs"]), int(mt["n_clusters"])
        ids[clu_ofs[m]:clu_ofs[m + 1]] = merged_ids[o:o + n]
        tail = int(sl[-1])
        valid[m] = 1 if refit["flags"][tail] == 0 else 0
        stq[m] = refit["p_out"][tail][2:5]
        step_ofs[m + 1] = step_ofs[m] + int(L.orc_rebuild_path_len(s.ctypes.data, len(s)))
    key = track_key_id(tracks, merged["head"])
    ns = int(step_ofs[-1])
    r = RebuildResult()
    r.step_ofs = step_ofs
    r.cand_id = np.full((ns, NCAND), -1, dtype=np.int32)
    r.cand_chi2 = np.zeros((ns, NCAND), dtype=np.float32)
    r.attached = np.full(ns, -1, dtype=np.int32)
    r.shared = np.zeros(ns, dtype=np.uint8)
    r.used = np.zeros(ns, dtype=np.uint8)
    fit = np.zeros((nm, 21), dtype=np.float32)
    chi2 = np.zeros(nm, dtype=np.float32)
    n_att = np.zeros(nm, dtype=np.int32)
    n_used = np.zeros(nm, dtype=np.int32)
    flags = np.zeros(nm, dtype=np.uint8)
    cl = np.ascontiguousarray(clusters)
    p = lambda a: a.ctypes.data
    rc = L.orc_rebuild(C.byref(geom), C.byref(params), C.byref(rparams), p(cl), len(cl), nm, p(seg_ofs), p(segs), p(clu_ofs),
                       p(ids), p(stq), p(valid), p(key), p(step_ofs), p(r.cand_id), p(r.cand_chi2), p(r.attached), p(r.shared),
                       p(r.used), p(fit), p(chi2), p(n_att), p(n_used), p(flags))
    if rc != 0:
        raise ValueError(f"oracle rebuild: error {rc}")
    r.fit = np.zeros(nm, dtype=REBUILD_FIT_DTYPE)
    r.fit["x"], r.fit["p"], r.fit["c"] = fit[:, 0], fit[:, 1:6], fit[:, 6:21]
    r.fit["chi2"], r.fit["n_attached"], r.fit["n_used"], r.fit["flags"] = chi2, n_att, n_used, flags
    r.segs, r.seg_ofs, r.key = segs, seg_ofs, key
    return r
