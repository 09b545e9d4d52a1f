"""ctypes binding of the CPU ORACLE (oracle/tpc_oracle.cpp) — TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  Nothing under paper_2601_20569_b200/ does; the oracle imports nothing
from the product either.  See tpc_oracle.h for what it computes and how it is pinned.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = os.path.join(_HERE, "liboracle.so")
_SRCS = [os.path.join(_HERE, f) for f in ("tpc_oracle.cpp", "tpc_merge_oracle.cpp", "tpc_fit_oracle.cpp",
                                          "tpc_rebuild_oracle.cpp", "tpc_oracle.h", "tpc_oracle_math.hpp")]

CLUSTER_DTYPE = np.dtype(
    [("y", "<f4"), ("z", "<f4"), ("q", "<f4"), ("sector", "u1"), ("row", "u1"), ("flags", "<u2")])
ROW_DESC_DTYPE = np.dtype(
    [("y0", "<f4"), ("z0", "<f4"), ("ny", "<i4"), ("nz", "<i4"), ("bin_ofs", "<u4"),
     ("clu_ofs", "<u4"), ("count", "<u4"), ("pad_", "<u4")])
SEED_DTYPE = np.dtype([("start_id", "<u4"), ("len", "<i4"), ("sector", "<i4"), ("row", "<i4")])
TRACKLET_DTYPE = np.dtype(
    [("x", "<f4"), ("p", "<f4", (5,)), ("c", "<f4", (15,)), ("chi2", "<f4"), ("seed_id", "<u4"),
     ("n_hits", "<i4"), ("row_first", "<i4"), ("row_last", "<i4"), ("sector", "<i4"), ("seed_len", "<i4")])
TRACK_DTYPE = np.dtype(
    [("x", "<f4"), ("p", "<f4", (5,)), ("c", "<f4", (15,)), ("chi2", "<f4"), ("cluster_ofs", "<u4"),
     ("seed_id", "<u4"), ("n_clusters", "<i4"), ("n_shared", "<i4"), ("sector", "<i4"),
     ("row_first", "<i4"), ("row_last", "<i4"), ("flags", "<i4"), ("n_hits_tracklet", "<i4"),
     ("segment", "<i4")])
TRACE_DTYPE = np.dtype(
    [("seed", "<i4"), ("row", "<i4"), ("dir", "<i4"), ("searched", "<i4"), ("y", "<f4"), ("z", "<f4"),
     ("c00", "<f4"), ("c10", "<f4"), ("c11", "<f4"), ("chi2", "<f4"), ("picked_id", "<i4"), ("accepted", "<i4")])


class Geom(C.Structure):
    _fields_ = [("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("n_inner_rows", C.c_int32),
                ("r_min", C.c_float), ("r_max", C.c_float), ("pad_pitch_inner", C.c_float),
                ("pad_pitch_outer", C.c_float), ("z_max", C.c_float), ("bz_tesla", C.c_float),
                ("sector_half_angle_deg", C.c_float)]


class Params(C.Structure):
    _fields_ = [("err_y", C.c_float), ("err_z", C.c_float),
                ("nf_slope_y", C.c_float), ("nf_slope_z", C.c_float), ("nf_max_d2", C.c_float),
                ("seed_min_len", C.c_int32),
                ("init_var_sinphi", C.c_float), ("init_var_tanl", C.c_float), ("init_var_qpt", C.c_float),
                ("max_sinphi", C.c_float), ("max_qpt", C.c_float),
                ("road_nsigma", C.c_float), ("road_min", C.c_float), ("road_max", C.c_float),
                ("chi2_max_hit", C.c_float),
                ("max_gap_follow", C.c_int32), ("min_hits_tracklet", C.c_int32),
                ("sel_chi2_weight", C.c_float),
                ("shared_permille", C.c_int32), ("max_gap_select", C.c_int32), ("min_hits_track", C.c_int32),
                ("grid_dy", C.c_float), ("grid_dz", C.c_float), ("shared_fixed_cap", C.c_int32)]


def default_geom(**kw) -> Geom:
    g = Geom(36, 152, 63, 85.0, 245.0, 0.4, 0.6, 250.0, 0.5, 10.0)
    for k, v in kw.items():
        setattr(g, k, v)
    return g


def build(force: bool = False) -> str:
    """Compile the oracle (host C++ only; -ffp-contract=off is rule D1)."""
    if (not force and os.path.exists(_LIB)
            and all(os.path.getmtime(_LIB) >= os.path.getmtime(s) for s in _SRCS)):
        return _LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC", "-pthread",
           _SRCS[0], _SRCS[1], _SRCS[2], _SRCS[3], "-o", _LIB]
    subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        vp = C.c_void_p
        L.orc_default_params.argtypes = [C.POINTER(Params)]
        L.orc_run.restype = vp
        L.orc_run.argtypes = [vp, C.c_uint64, C.POINTER(Geom), C.POINTER(Params), C.c_int, C.c_int, C.c_int]
        L.orc_free.argtypes = [vp]
        L.orc_sizes.argtypes = [vp, vp]
        L.orc_stage_seconds.argtypes = [vp, vp]
        L.orc_set_trace.argtypes = [C.c_int]
        L.orc_trace_size.restype = C.c_uint64
        L.orc_trace_size.argtypes = [vp]
        L.orc_fetch_trace.argtypes = [vp, vp]
        L.orc_fetch_grid.argtypes = [vp] * 4
        L.orc_fetch_links.argtypes = [vp] * 5
        L.orc_fetch_seeds.argtypes = [vp] * 2
        L.orc_fetch_tracklets.argtypes = [vp] * 3
        L.orc_fetch_tracks.argtypes = [vp] * 4
        L.orc_geom_tables.argtypes = [C.POINTER(Geom), vp, vp, vp]
        L.orc_propagate_f.restype = C.c_int
        L.orc_propagate_f.argtypes = [vp, C.c_float, C.c_float, C.c_float, vp]
        L.orc_propagate_d.restype = C.c_int
        L.orc_propagate_d.argtypes = [vp, C.c_double, C.c_double, C.c_double, vp]
        L.orc_update_f.restype = C.c_float
        L.orc_update_f.argtypes = [vp] + [C.c_float] * 6 + [vp]
        L.orc_update_d.restype = C.c_double
        L.orc_update_d.argtypes = [vp] + [C.c_double] * 6 + [vp]
        L.orc_fit_hits.restype = C.c_float
        L.orc_fit_hits.argtypes = [C.POINTER(Geom), C.POINTER(Params), vp, vp, vp, C.c_int, vp]
        L.orc_refit_hits.restype = C.c_float
        L.orc_refit_hits.argtypes = [C.POINTER(Geom), C.POINTER(Params), vp, vp, vp, C.c_int, vp]
        L.orc_select_only.restype = vp
        L.orc_select_only.argtypes = [C.POINTER(Geom), C.POINTER(Params), C.c_uint64, C.c_int, vp, vp, vp, vp]
        _lib = L
    return _lib


def default_params(**kw) -> Params:
    p = Params()
    lib().orc_default_params(C.byref(p))
    for k, v in kw.items():
        setattr(p, k, v)
    return p


def _ptr(a):
    return None if a is None else a.ctypes.data


class Result:
    """Everything one oracle run produced, as numpy arrays (original cluster indices)."""

    def __init__(self, handle, n_rows, n_clusters, want=("grid", "links", "seeds", "tracklets", "tracks")):
        L = lib()
        sz = np.zeros(10, dtype=np.uint64)
        L.orc_sizes(handle, sz.ctypes.data)
        (self.n_rows_total, self.n_bins, self.n_sorted, self.n_seeds, self.n_tracks, self.n_cluster_ids,
         self.n_ignored, self.n_dropped, self.n_bad, self.n_tracklets) = [int(v) for v in sz]
        st = np.zeros(5, dtype=np.float64)
        L.orc_stage_seconds(handle, st.ctypes.data)
        self.stage_seconds = st
        self.n_rows = n_rows
        self.n_clusters = n_clusters
        self._fill(handle, want)

    def _fill(self, h, want):
        L = lib()
        n = self.n_clusters
        if "grid" in want:
            self.row_desc = np.zeros(self.n_rows_total, dtype=ROW_DESC_DTYPE)
            self.bin_start = np.zeros(self.n_bins + 1, dtype=np.uint32)
            self.sorted_ids = np.zeros(self.n_sorted, dtype=np.uint32)
            L.orc_fetch_grid(h, _ptr(self.row_desc), _ptr(self.bin_start), _ptr(self.sorted_ids))
        if "links" in want:
            self.link_up, self.link_dn, self.link_up2, self.link_dn2 = (
                np.empty(n, dtype=np.int32) for _ in range(4))
            L.orc_fetch_links(h, _ptr(self.link_up), _ptr(self.link_dn), _ptr(self.link_up2), _ptr(self.link_dn2))
        if "seeds" in want:
            self.seeds = np.zeros(self.n_seeds, dtype=SEED_DTYPE)
            L.orc_fetch_seeds(h, _ptr(self.seeds))
        if "tracklets" in want:
            self.tracklets = np.zeros(self.n_seeds, dtype=TRACKLET_DTYPE)
            self.row_hit = np.zeros((self.n_seeds, self.n_rows), dtype=np.int32)
            L.orc_fetch_tracklets(h, _ptr(self.tracklets), _ptr(self.row_hit))
        if "trace" in want:
            self.trace = np.zeros(int(L.orc_trace_size(h)), dtype=TRACE_DTYPE)
            L.orc_fetch_trace(h, _ptr(self.trace))
        if "tracks" in want:
            self.tracks = np.zeros(self.n_tracks, dtype=TRACK_DTYPE)
            self.cluster_ids = np.zeros(self.n_cluster_ids, dtype=np.uint32)
            self.cluster_shared = np.zeros(self.n_cluster_ids, dtype=np.uint8)
            L.orc_fetch_tracks(h, _ptr(self.tracks), _ptr(self.cluster_ids), _ptr(self.cluster_shared))


def run(clusters: np.ndarray, geom: Geom | None = None, params: Params | None = None,
        sector_lo: int = 0, sector_hi: int = 1 << 30, n_threads: int = 1,
        want=("grid", "links", "seeds", "tracklets", "tracks")) -> Result:
    """Run the whole path (R0..R6) on sectors [sector_lo, sector_hi) of ``clusters``."""
    assert clusters.dtype.itemsize == 16
    clusters = np.ascontiguousarray(clusters)
    geom = geom or default_geom()
    params = params or default_params()
    L = lib()
    L.orc_set_trace(1 if "trace" in want else 0)
    try:
        h = L.orc_run(clusters.ctypes.data, len(clusters), C.byref(geom), C.byref(params),
                      sector_lo, min(sector_hi, geom.n_sectors), 1 if "trace" in want else n_threads)
    finally:
        L.orc_set_trace(0)
    if not h:
        raise ValueError("oracle: bad argument")
    try:
        return Result(h, geom.n_rows, len(clusters), want)
    finally:
        L.orc_free(h)


def select_only(row_hit: np.ndarray, n_hits, chi2, seed_id, n_clusters: int,
                geom: Geom | None = None, params: Params | None = None) -> Result:
    """R6 alone on hand-made tracklets (row_hit[n_tracklets][n_rows] of cluster ids / -1)."""
    geom = geom or default_geom()
    params = params or default_params()
    row_hit = np.ascontiguousarray(row_hit, dtype=np.int32)
    n_hits = np.ascontiguousarray(n_hits, dtype=np.int32)
    chi2 = np.ascontiguousarray(chi2, dtype=np.float32)
    seed_id = np.ascontiguousarray(seed_id, dtype=np.uint32)
    assert row_hit.shape == (len(n_hits), geom.n_rows)
    L = lib()
    h = L.orc_select_only(C.byref(geom), C.byref(params), n_clusters, len(n_hits), _ptr(row_hit),
                          _ptr(n_hits), _ptr(chi2), _ptr(seed_id))
    try:
        return Result(h, geom.n_rows, n_clusters, want=("tracks",))
    finally:
        L.orc_free(h)


def geom_tables(geom: Geom | None = None):
    geom = geom or default_geom()
    x = np.zeros(geom.n_rows, dtype=np.float32)
    ymax = np.zeros(geom.n_rows, dtype=np.float32)
    consts = np.zeros(2, dtype=np.float32)
    lib().orc_geom_tables(C.byref(geom), _ptr(x), _ptr(ymax), _ptr(consts))
    return x, ymax, float(consts[0]), float(consts[1])


def propagate(state: np.ndarray, dx, cfield, max_sinphi=0.95):
    """One propagation step on a 20-vector (y,z,s,t,q,c[15]); dtype float32 or float64 selects
    the instantiation.  Returns (ok, new_state, jac6=(f02,f04,f12,f13,f14,f24))."""
    st = np.array(state, copy=True)
    jac = np.zeros(6, dtype=st.dtype)
    if st.dtype == np.float32:
        ok = lib().orc_propagate_f(_ptr(st), dx, cfield, max_sinphi, _ptr(jac))
    else:
        assert st.dtype == np.float64
        ok = lib().orc_propagate_d(_ptr(st), dx, cfield, max_sinphi, _ptr(jac))
    return bool(ok), st, jac


def update(state: np.ndarray, ym, zm, vy, vz, max_sinphi=0.95, max_qpt=20.0):
    """Kalman update; returns (chi2, stop, new_state)."""
    st = np.array(state, copy=True)
    stop = C.c_int(0)
    if st.dtype == np.float32:
        chi2 = lib().orc_update_f(_ptr(st), ym, zm, vy, vz, max_sinphi, max_qpt, C.addressof(stop))
    else:
        chi2 = lib().orc_update_d(_ptr(st), ym, zm, vy, vz, max_sinphi, max_qpt, C.addressof(stop))
    return chi2, bool(stop.value), st


def fit_hits(rows, y, z, geom: Geom | None = None, params: Params | None = None):
    """Kalman fit of a given hit list as the follower does it (up pass, turn, refit down).
    Returns (chi2, x, p[5], c[15], n_hits, row_first) or None if the leg stopped."""
    geom = geom or default_geom()
    params = params or default_params()
    rows = np.ascontiguousarray(rows, dtype=np.int32)
    y = np.ascontiguousarray(y, dtype=np.float32)
    z = np.ascontiguousarray(z, dtype=np.float32)
    out = np.zeros(24, dtype=np.float32)
    chi2 = lib().orc_fit_hits(C.byref(geom), C.byref(params), _ptr(rows), _ptr(y), _ptr(z), len(rows), _ptr(out))
    if chi2 < 0:
        return None
    return float(chi2), float(out[0]), out[1:6].copy(), out[6:21].copy(), int(out[21]), int(out[22])


FIT_DTYPE = np.dtype([("x", "<f4"), ("p", "<f4", (5,)), ("c", "<f4", (15,)), ("chi2", "<f4"), ("n_clusters", "<u4"),
                      ("flags", "<u4"), ("x_out", "<f4"), ("p_out", "<f4", (5,)), ("c_out", "<f4", (15,)),
                      ("pad_", "<u4", (3,))])


def refit_hits(rows, y, z, geom: Geom | None = None, params: Params | None = None, both_ends: bool = False):
    """R8 sector-track refit of a given cluster list (rows strictly ascending, holes allowed).
    Returns (chi2, x, p[5], c[15], n) or None if the fit left the |sin phi| range; with both_ends
    also (x_out, p_out[5], c_out[15]), the state after the outward pass at the last cluster."""
    geom = geom or default_geom()
    params = params or default_params()
    rows = np.ascontiguousarray(rows, dtype=np.int32)
    y = np.ascontiguousarray(y, dtype=np.float32)
    z = np.ascontiguousarray(z, dtype=np.float32)
    out = np.zeros(48, dtype=np.float32)
    chi2 = lib().orc_refit_hits(C.byref(geom), C.byref(params), _ptr(rows), _ptr(y), _ptr(z), len(rows), _ptr(out))
    if chi2 < 0:
        return None
    r = (float(chi2), float(out[0]), out[1:6].copy(), out[6:21].copy(), int(out[21]))
    if both_ends:
        r = r + (float(out[22]), out[23:28].copy(), out[28:43].copy())
    return r


def refit_tracks(clusters: np.ndarray, tracks: np.ndarray, cluster_ids: np.ndarray, geom=None, params=None):
    """R8 for every track of a result: (fit[n_tracks] records, FIT_DTYPE) from the tracks' cluster
    lists (original indices into ``clusters``)."""
    out = np.zeros(len(tracks), dtype=FIT_DTYPE)
    for k, t in enumerate(tracks):
        ids = cluster_ids[int(t["cluster_ofs"]): int(t["cluster_ofs"]) + int(t["n_clusters"])]
        r = refit_hits(clusters["row"][ids], clusters["y"][ids], clusters["z"][ids], geom, params, both_ends=True)
        if r is None:
            out[k]["flags"] = 1
            out[k]["n_clusters"] = len(ids)
            continue
        (out[k]["chi2"], out[k]["x"], out[k]["p"], out[k]["c"], out[k]["n_clusters"],
         out[k]["x_out"], out[k]["p_out"], out[k]["c_out"]) = r
    return out
