"""R10 three-iteration track fit with the Phase-I interpolation rejection, CPU ORACLE side (TEST
INFRASTRUCTURE): PAPER.md:31,37 (section 2), PAPER.md:57 (section 3).  The arithmetic is
oracle/tpc_fit_oracle.cpp; this module hands it the cluster lists of merged tracks."""
from __future__ import annotations

import ctypes as C

import numpy as np

import oracle

TRACK_FIT3_DTYPE = np.dtype([("x", "<f4"), ("p", "<f4", (5,)), ("c", "<f4", (15,)), ("chi2", "<f4"), ("n_clusters", "<u4"),
                             ("n_used", "<u4"), ("flags", "<u4")])


class FitParams(C.Structure):
    _fields_ = [("fit_chi2_max", C.c_float), ("fit_min_clusters", C.c_int32), ("ce_var", C.c_float)]


def _lib():
    L = oracle.lib()
    if not getattr(L, "_fit_ready", False):
        vp = C.c_void_p
        L.orc_fit_default_params.argtypes = [C.POINTER(FitParams)]
        L.orc_float_to_half.restype = C.c_uint16
        L.orc_float_to_half.argtypes = [C.c_float]
        L.orc_half_to_float.restype = C.c_float
        L.orc_half_to_float.argtypes = [C.c_uint16]
        L.orc_fit_track.restype = C.c_float
        L.orc_fit_track.argtypes = [C.POINTER(oracle.Geom), C.POINTER(oracle.Params), C.POINTER(FitParams), vp, vp, vp, vp,
                                    C.c_int, vp, vp, vp, vp, vp]
        L._fit_ready = True
    return L


def default_fit_params(**kw) -> FitParams:
    f = FitParams()
    _lib().orc_fit_default_params(C.byref(f))
    for k, v in kw.items():
        setattr(f, k, v)
    return f


def float_to_half(x: float) -> int:
    return int(_lib().orc_float_to_half(float(x)))


def half_to_float(h: int) -> float:
    return float(_lib().orc_half_to_float(int(h)))


def fit_track(sector, row, y, z, start_stq, geom=None, params=None, fparams=None):
    """One track (clusters in chain order).  Returns (chi2 or None, x, p, c, n_used, chi2_cluster, rejected)."""
    geom = geom or oracle.default_geom()
    params = params or oracle.default_params()
    fparams = fparams or default_fit_params()
    sector = np.ascontiguousarray(sector, dtype=np.int32)
    row = np.ascontiguousarray(row, dtype=np.int32)
    y = np.ascontiguousarray(y, dtype=np.float32)
    z = np.ascontiguousarray(z, dtype=np.float32)
    stq = np.ascontiguousarray(start_stq, dtype=np.float32)
    n = len(row)
    out = np.zeros(24, dtype=np.float32)
    chi = np.zeros(n, dtype=np.float32)
    rej = np.zeros(n, dtype=np.uint8)
    n_used = C.c_int32(0)
    chi2 = _lib().orc_fit_track(C.byref(geom), C.byref(params), C.byref(fparams), sector.ctypes.data, row.ctypes.data,
                                y.ctypes.data, z.ctypes.data, n, stq.ctypes.data, out.ctypes.data, chi.ctypes.data,
                                rej.ctypes.data, C.addressof(n_used))
    ok = chi2 >= 0
    return (float(chi2) if ok else None), float(out[0]), out[1:6].copy(), out[6:21].copy(), int(n_used.value), chi, rej


def fit_merged(clusters, tracks, refit, merged, seg_index, merged_ids, geom=None, params=None, fparams=None):
    """R10 for every merged track: start parameters = the refit's outer state (R8) of the chain's LAST
    segment.  Returns (fit[n_merged] records, chi2_cluster[n_ids], rejected[n_ids])."""
    out = np.zeros(len(merged), dtype=TRACK_FIT3_DTYPE)
    chi_all = np.zeros(len(merged_ids), dtype=np.float32)
    rej_all = np.zeros(len(merged_ids), dtype=np.uint8)
    for k, m in enumerate(merged):
        o, n = int(m["cluster_ofs"]), int(m["n_clusters"])
        ids = merged_ids[o:o + n]
        tail = int(seg_index[int(m["seg_ofs"]) + int(m["n_segments"]) - 1])
        out[k]["n_clusters"] = n
        if refit["flags"][tail] != 0:
            out[k]["flags"] = 1
            continue
        r = fit_track(clusters["sector"][ids], clusters["row"][ids], clusters["y"][ids], clusters["z"][ids],
                      refit["p_out"][tail][2:5], geom, params, fparams)
        chi_all[o:o + n], rej_all[o:o + n] = r[5], r[6]
        out[k]["n_used"] = r[4]
        if r[0] is None:
            out[k]["flags"] = 1
            continue
        out[k]["chi2"], out[k]["x"], out[k]["p"], out[k]["c"] = r[0], r[1], r[2], r[3]
    return out, chi_all, rej_all
