"""Thin ctypes binding of the C-ABI library libtpctrack.so (include/tpc_track.h).

Argument marshalling only: every step of the path (grid, neighbour finder, link cleanup,
seeds, Kalman follower, ambiguity solving) runs in the CUDA kernels of csrc/.  PyTorch is used
for device memory and streams, nothing else.  There is NO CPU fallback: importing this module
without the built library, or calling it without a CUDA device, raises.

Low level: the functions ``tpc_*`` have the names and arguments of the header.
High level: ``SectorTracker`` owns a context and a workspace and returns results as arrays.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .build import LIB_PATH

TPC_OK, TPC_E_ARG, TPC_E_WORKSPACE, TPC_E_OVERFLOW, TPC_E_CUDA, TPC_E_STATE = 0, -1, -2, -3, -4, -5
TPC_DETERMINISTIC, TPC_KEEP_INTERMEDIATES, TPC_STAGE_TIMERS, TPC_GRID_ONLY = 1, 2, 4, 8
TPC_N_STAGES = 6
STAGE_NAMES = ("grid", "neighbours", "cleanup_seeds", "follower", "selector", "total")

CLUSTER_DTYPE = np.dtype(
    [("y", "<f4"), ("z", "<f4"), ("q", "<f4"), ("sector", "u1"), ("row", "u1"), ("flags", "<u2")])
TRACK_DTYPE = np.dtype(
    [("x", "<f4"), ("p", "<f4", (5,)), ("c", "<f4", (15,)), ("chi2", "<f4"), ("cluster_ofs", "<u4"),
     ("seed_id", "<u4"), ("n_clusters", "<u2"), ("n_shared", "<u2"), ("sector", "u1"),
     ("row_first", "u1"), ("row_last", "u1"), ("flags", "u1"), ("n_hits_tracklet", "<u2"),
     ("segment", "u1"), ("pad_", "u1")])
TRACKLET_DTYPE = np.dtype(
    [("x", "<f4"), ("p", "<f4", (5,)), ("c", "<f4", (15,)), ("chi2", "<f4"), ("seed_sorted", "<u4"),
     ("seed_id", "<u4"), ("n_hits", "<i2"), ("row_first", "u1"), ("row_last", "u1"), ("sector", "u1"),
     ("seed_len", "u1"), ("pad_", "<u2"), ("pad2_", "<u4", (2,))])
ROW_DESC_DTYPE = np.dtype(
    [("y0", "<f4"), ("z0", "<f4"), ("ny", "<i4"), ("nz", "<i4"), ("bin_ofs", "<u4"),
     ("clu_ofs", "<u4"), ("count", "<u4"), ("pad_", "<u4")])
assert TRACK_DTYPE.itemsize == 108 and TRACKLET_DTYPE.itemsize == 112 and ROW_DESC_DTYPE.itemsize == 32


class GeomDesc(C.Structure):
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
                ("grid_dy", C.c_float), ("grid_dz", C.c_float),
                ("max_bins", C.c_uint64), ("max_seeds", C.c_uint32), ("shared_fixed_cap", C.c_uint32),
                ("max_ids", C.c_uint32), ("reserved", C.c_uint32)]


class TrackView(C.Structure):
    _fields_ = [("n_tracks", C.c_uint64), ("n_cluster_ids", C.c_uint64),
                ("d_tracks", C.c_void_p), ("d_cluster_ids", C.c_void_p), ("d_cluster_shared", C.c_void_p),
                ("n_ignored", C.c_uint64), ("n_dropped", C.c_uint64), ("n_seeds", C.c_uint64),
                ("n_tracklets", C.c_uint64), ("n_bins", C.c_uint64),
                ("n_follow_steps", C.c_uint64), ("n_follow_updates", C.c_uint64),
                ("n_follow_candidates", C.c_uint64), ("follow_work", (C.c_uint64 * 3) * 3),
                ("grid_by_rows", C.c_uint64), ("n_rows_generic", C.c_uint64)]


class MergeParams(C.Structure):
    _fields_ = [("gap_in_sector", C.c_int32), ("gap_adjacent_back", C.c_int32), ("gap_adjacent", C.c_int32),
                ("gap_ce", C.c_int32), ("chi2_max", C.c_float), ("sys", C.c_float * 5), ("ce_sys_z", C.c_float),
                ("pre_dy", C.c_float), ("pre_dz", C.c_float), ("pre_coarse_dz", C.c_float), ("stages", C.c_int32)]


class MergedView(C.Structure):
    _fields_ = [("n_tracks", C.c_uint64), ("n_merged", C.c_uint64), ("n_links", C.c_uint64),
                ("n_cluster_ids", C.c_uint64), ("d_merged", C.c_void_p), ("d_seg_index", C.c_void_p),
                ("d_cluster_ids", C.c_void_p), ("d_cluster_shared", C.c_void_p), ("d_next", C.c_void_p),
                ("d_prev", C.c_void_p), ("d_link_chi2", C.c_void_p)]


MERGED_DTYPE = np.dtype(
    [("head", "<u4"), ("n_segments", "<u4"), ("n_clusters", "<u4"), ("n_shared", "<u4"), ("cluster_ofs", "<u4"),
     ("seg_ofs", "<u4"), ("row_first", "<i4"), ("row_last", "<i4"), ("sector_first", "<i4"), ("sector_last", "<i4")])
assert MERGED_DTYPE.itemsize == 40 and C.sizeof(MergeParams) == 60


class FitParams(C.Structure):
    _fields_ = [("fit_chi2_max", C.c_float), ("fit_min_clusters", C.c_int32), ("ce_var", C.c_float)]


class FitView(C.Structure):
    _fields_ = [("n_merged", C.c_uint64), ("n_cluster_ids", C.c_uint64), ("d_fit", C.c_void_p),
                ("d_chi2_cluster", C.c_void_p), ("d_rejected", C.c_void_p)]


TRACK_FIT3_DTYPE = np.dtype([("x", "<f4"), ("p", "<f4", (5,)), ("c", "<f4", (15,)), ("chi2", "<f4"),
                             ("n_clusters", "<u4"), ("n_used", "<u4"), ("flags", "<u4")])
assert TRACK_FIT3_DTYPE.itemsize == 100 and C.sizeof(FitParams) == 12


class RebuildParams(C.Structure):
    _fields_ = [("cand_chi2_max", C.c_float), ("final_chi2_max", C.c_float), ("min_clusters", C.c_int32), ("ce_var", C.c_float)]


class RebuildView(C.Structure):
    _fields_ = [("n_merged", C.c_uint64), ("n_steps", C.c_uint64), ("d_step_ofs", C.c_void_p), ("d_cand_id", C.c_void_p),
                ("d_cand_chi2", C.c_void_p), ("d_attached", C.c_void_p), ("d_shared", C.c_void_p), ("d_used", C.c_void_p),
                ("d_fit", C.c_void_p)]


class DebugView(C.Structure):
    _fields_ = [("n_clusters", C.c_uint64), ("n_sorted", C.c_uint64), ("n_rows_total", C.c_uint64),
                ("n_bins", C.c_uint64), ("n_seeds", C.c_uint64), ("tracklet_stride", C.c_uint64),
                ("d_row_desc", C.c_void_p), ("d_bin_start", C.c_void_p), ("d_yz_sorted", C.c_void_p),
                ("d_orig_id", C.c_void_p), ("d_link_up", C.c_void_p), ("d_link_dn", C.c_void_p),
                ("d_link_up2", C.c_void_p), ("d_link_dn2", C.c_void_p), ("d_seeds", C.c_void_p),
                ("d_tracklets", C.c_void_p), ("d_row_hit", C.c_void_p)]


EXPORTS = ("tpc_default_params", "tpc_geom_init", "tpc_workspace_bytes", "tpc_sector_track",
           "tpc_get_tracks", "tpc_get_intermediates", "tpc_get_stage_ms", "tpc_get_kernel_ms",
           "tpc_sector_track_host", "tpc_sector_track_host_chunks", "tpc_workspace_bytes_two_iterations",
           "tpc_sector_track_two_iterations", "tpc_refit_tracks", "tpc_get_refit", "tpc_merge_default_params",
           "tpc_merge_workspace_bytes", "tpc_merge_tracks", "tpc_get_merged", "tpc_fit_default_params",
           "tpc_fit_workspace_bytes", "tpc_fit_tracks", "tpc_get_fit", "tpc_fit_tracks_noalloc", "tpc_rebuild_default_params", "tpc_set_tracks",
           "tpc_rebuild_prepare", "tpc_rebuild_workspace_bytes", "tpc_rebuild_tracks", "tpc_get_rebuild",
           "tpc_last_launch_count",
           "tpc_destroy", "tpc_strerror", "tpc_last_cuda_error")

_lib = None


def load_library():
    """dlopen libtpctrack.so and declare the prototypes of include/tpc_track.h.  Raises if
    the library has not been built (python -m paper_2601_20569_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2601_20569_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    L.tpc_default_params.restype = None
    L.tpc_default_params.argtypes = [C.POINTER(Params)]
    L.tpc_geom_init.restype = C.c_int
    L.tpc_geom_init.argtypes = [C.POINTER(GeomDesc), C.POINTER(Params), C.POINTER(vp)]
    L.tpc_workspace_bytes.restype = C.c_size_t
    L.tpc_workspace_bytes.argtypes = [vp, C.c_uint64]
    L.tpc_sector_track.restype = C.c_int
    L.tpc_sector_track.argtypes = [vp, vp, C.c_uint64, vp, C.c_size_t, vp, C.c_uint32]
    L.tpc_get_tracks.restype = C.c_int
    L.tpc_get_tracks.argtypes = [vp, C.POINTER(TrackView)]
    L.tpc_get_intermediates.restype = C.c_int
    L.tpc_get_intermediates.argtypes = [vp, C.POINTER(DebugView)]
    L.tpc_get_stage_ms.restype = C.c_int
    L.tpc_get_stage_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.tpc_get_kernel_ms.restype = C.c_int
    L.tpc_get_kernel_ms.argtypes = [vp, C.c_int, C.POINTER(C.c_char_p), C.POINTER(C.c_float)]
    L.tpc_workspace_bytes_two_iterations.restype = C.c_size_t
    L.tpc_workspace_bytes_two_iterations.argtypes = [vp, C.c_uint64]
    L.tpc_sector_track_two_iterations.restype = C.c_int
    L.tpc_sector_track_two_iterations.argtypes = [vp, vp, C.c_uint64, vp, C.c_size_t, vp, C.c_uint32]
    L.tpc_refit_tracks.restype = C.c_int
    L.tpc_refit_tracks.argtypes = [vp, vp]
    L.tpc_get_refit.restype = C.c_int
    L.tpc_get_refit.argtypes = [vp, C.POINTER(C.c_void_p)]
    L.tpc_sector_track_host_chunks.restype = C.c_int
    L.tpc_sector_track_host_chunks.argtypes = [vp, vp, C.c_uint64, C.POINTER(C.c_uint64), C.c_int, vp, vp, C.c_size_t, vp,
                                               C.c_uint32, vp, C.c_uint64, vp, vp, C.c_uint64, vp]
    L.tpc_sector_track_host.restype = C.c_int
    L.tpc_sector_track_host.argtypes = [vp, vp, C.c_uint64, vp, vp, C.c_size_t, vp, C.c_uint32, vp, C.c_uint64,
                                        vp, vp, C.c_uint64, C.POINTER(TrackView)]
    L.tpc_merge_default_params.restype = None
    L.tpc_merge_default_params.argtypes = [C.POINTER(MergeParams)]
    L.tpc_merge_workspace_bytes.restype = C.c_size_t
    L.tpc_merge_workspace_bytes.argtypes = [vp, C.c_uint64, C.c_uint64]
    L.tpc_merge_tracks.restype = C.c_int
    L.tpc_merge_tracks.argtypes = [vp, C.POINTER(MergeParams), vp, C.c_size_t, vp]
    L.tpc_get_merged.restype = C.c_int
    L.tpc_get_merged.argtypes = [vp, C.POINTER(MergedView)]
    L.tpc_fit_default_params.restype = None
    L.tpc_fit_default_params.argtypes = [C.POINTER(FitParams)]
    L.tpc_fit_workspace_bytes.restype = C.c_size_t
    L.tpc_fit_workspace_bytes.argtypes = [vp, C.c_uint64, C.c_uint64]
    L.tpc_fit_tracks.restype = C.c_int
    L.tpc_fit_tracks.argtypes = [vp, C.POINTER(FitParams), vp, C.c_size_t, vp]
    L.tpc_get_fit.restype = C.c_int
    L.tpc_get_fit.argtypes = [vp, C.POINTER(FitView)]
    L.tpc_fit_tracks_noalloc.restype = C.c_int
    L.tpc_fit_tracks_noalloc.argtypes = [vp, C.POINTER(FitParams), vp, C.c_uint64, vp, C.c_uint64, vp, C.c_uint64, vp, vp,
                                         C.c_uint64, vp, vp, vp, C.c_uint32, vp]
    L.tpc_set_tracks.restype = C.c_int
    L.tpc_set_tracks.argtypes = [vp, vp, C.c_uint64, vp, vp, C.c_uint64, vp]
    L.tpc_rebuild_default_params.restype = None
    L.tpc_rebuild_default_params.argtypes = [C.POINTER(RebuildParams)]
    L.tpc_rebuild_prepare.restype = C.c_int
    L.tpc_rebuild_prepare.argtypes = [vp, vp, C.POINTER(C.c_uint64)]
    L.tpc_rebuild_workspace_bytes.restype = C.c_size_t
    L.tpc_rebuild_workspace_bytes.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_uint64]
    L.tpc_rebuild_tracks.restype = C.c_int
    L.tpc_rebuild_tracks.argtypes = [vp, C.POINTER(RebuildParams), vp, C.c_size_t, vp]
    L.tpc_get_rebuild.restype = C.c_int
    L.tpc_get_rebuild.argtypes = [vp, C.POINTER(RebuildView)]
    L.tpc_last_launch_count.restype = C.c_int
    L.tpc_last_launch_count.argtypes = [vp]
    L.tpc_destroy.restype = None
    L.tpc_destroy.argtypes = [vp]
    L.tpc_strerror.restype = C.c_char_p
    L.tpc_strerror.argtypes = [C.c_int]
    L.tpc_last_cuda_error.restype = C.c_char_p
    L.tpc_last_cuda_error.argtypes = [vp]
    _lib = L
    return L


# ---------------------------------------------------------------- header-named thin wrappers
def tpc_default_params(**overrides) -> Params:
    p = Params()
    load_library().tpc_default_params(C.byref(p))
    for k, v in overrides.items():
        setattr(p, k, v)
    return p


def default_geom(**overrides) -> GeomDesc:
    """The TPC of BASELINE.json config 1: 36 sectors x 152 rows, 85-245 cm, 0.5 T."""
    g = GeomDesc(36, 152, 63, 85.0, 245.0, 0.4, 0.6, 250.0, 0.5, 10.0)
    for k, v in overrides.items():
        setattr(g, k, v)
    return g


class TpcError(RuntimeError):
    def __init__(self, code, where, detail=""):
        self.code = code
        msg = load_library().tpc_strerror(code).decode()
        super().__init__(f"{where}: {msg} ({code}) {detail}".strip())


def tpc_geom_init(geom: GeomDesc, params: Params | None) -> int:
    ctx = C.c_void_p()
    rc = load_library().tpc_geom_init(C.byref(geom), C.byref(params) if params is not None else None, C.byref(ctx))
    if rc != TPC_OK:
        raise TpcError(rc, "tpc_geom_init")
    return ctx.value


def tpc_workspace_bytes(ctx: int, n_clusters: int) -> int:
    return int(load_library().tpc_workspace_bytes(ctx, n_clusters))


def tpc_sector_track(ctx: int, d_clusters: int, n_clusters: int, d_workspace: int, workspace_bytes: int,
                     cuda_stream: int, flags: int) -> int:
    return load_library().tpc_sector_track(ctx, d_clusters, n_clusters, d_workspace, workspace_bytes,
                                           cuda_stream, flags)


def tpc_get_tracks(ctx: int):
    v = TrackView()
    rc = load_library().tpc_get_tracks(ctx, C.byref(v))
    return rc, v


def tpc_get_intermediates(ctx: int):
    v = DebugView()
    rc = load_library().tpc_get_intermediates(ctx, C.byref(v))
    return rc, v


def tpc_get_stage_ms(ctx: int):
    out = (C.c_float * TPC_N_STAGES)()
    rc = load_library().tpc_get_stage_ms(ctx, out)
    return rc, [float(x) for x in out]


def tpc_get_kernel_ms(ctx: int, max_kernels: int = 32):
    names = (C.c_char_p * max_kernels)()
    ms = (C.c_float * max_kernels)()
    rc = load_library().tpc_get_kernel_ms(ctx, max_kernels, names, ms)
    if rc < 0:
        return rc, []
    return rc, [(names[i].decode(), float(ms[i])) for i in range(rc)]


def tpc_sector_track_host(ctx: int, h_clusters: int, n_clusters: int, d_staging: int, d_workspace: int,
                          workspace_bytes: int, cuda_stream: int, flags: int, h_tracks: int, cap_tracks: int,
                          h_cluster_ids: int, h_cluster_shared: int, cap_ids: int):
    v = TrackView()
    rc = load_library().tpc_sector_track_host(ctx, h_clusters, n_clusters, d_staging, d_workspace, workspace_bytes,
                                              cuda_stream, flags, h_tracks, cap_tracks, h_cluster_ids,
                                              h_cluster_shared, cap_ids, C.byref(v))
    return rc, v


def tpc_sector_track_host_chunks(ctx: int, h_clusters: int, n_clusters: int, chunk_ofs, d_staging: int,
                                 d_workspace: int, workspace_bytes: int, cuda_stream: int, flags: int,
                                 h_tracks: int, cap_tracks: int, h_cluster_ids: int, h_cluster_shared: int,
                                 cap_ids: int):
    v = TrackView()
    ofs = (C.c_uint64 * len(chunk_ofs))(*[int(x) for x in chunk_ofs])
    rc = load_library().tpc_sector_track_host_chunks(ctx, h_clusters, n_clusters, ofs, len(chunk_ofs) - 1, d_staging,
                                                     d_workspace, workspace_bytes, cuda_stream, flags, h_tracks,
                                                     cap_tracks, h_cluster_ids, h_cluster_shared, cap_ids, C.byref(v))
    return rc, v


def tpc_workspace_bytes_two_iterations(ctx: int, n_clusters: int) -> int:
    return load_library().tpc_workspace_bytes_two_iterations(ctx, n_clusters)


def tpc_sector_track_two_iterations(ctx: int, d_clusters: int, n_clusters: int, d_workspace: int, workspace_bytes: int,
                                    cuda_stream: int, flags: int) -> int:
    return load_library().tpc_sector_track_two_iterations(ctx, d_clusters, n_clusters, d_workspace, workspace_bytes,
                                                          cuda_stream, flags)


TRACK_FIT_DTYPE = np.dtype([("x", "<f4"), ("p", "<f4", (5,)), ("c", "<f4", (15,)), ("chi2", "<f4"),
                            ("n_clusters", "<u4"), ("flags", "<u4"), ("x_out", "<f4"), ("p_out", "<f4", (5,)),
                            ("c_out", "<f4", (15,)), ("pad_", "<u4", (3,))])
assert TRACK_FIT_DTYPE.itemsize == 192


def tpc_refit_tracks(ctx: int, cuda_stream: int) -> int:
    return load_library().tpc_refit_tracks(ctx, cuda_stream)


def tpc_get_refit(ctx: int):
    p = C.c_void_p()
    rc = load_library().tpc_get_refit(ctx, C.byref(p))
    return rc, p.value


def tpc_merge_default_params(**overrides) -> MergeParams:
    m = MergeParams()
    load_library().tpc_merge_default_params(C.byref(m))
    for k, v in overrides.items():
        if k == "sys":
            for i in range(5):
                m.sys[i] = v[i]
        else:
            setattr(m, k, v)
    return m


def tpc_merge_workspace_bytes(ctx: int, n_tracks: int, n_cluster_ids: int) -> int:
    return int(load_library().tpc_merge_workspace_bytes(ctx, n_tracks, n_cluster_ids))


def tpc_merge_tracks(ctx: int, params, d_workspace: int, workspace_bytes: int, cuda_stream: int) -> int:
    return load_library().tpc_merge_tracks(ctx, C.byref(params) if params is not None else None, d_workspace,
                                           workspace_bytes, cuda_stream)


def tpc_get_merged(ctx: int):
    v = MergedView()
    rc = load_library().tpc_get_merged(ctx, C.byref(v))
    return rc, v


def tpc_fit_default_params(**overrides) -> FitParams:
    f = FitParams()
    load_library().tpc_fit_default_params(C.byref(f))
    for k, v in overrides.items():
        setattr(f, k, v)
    return f


def tpc_fit_workspace_bytes(ctx: int, n_merged: int, n_cluster_ids: int) -> int:
    return int(load_library().tpc_fit_workspace_bytes(ctx, n_merged, n_cluster_ids))


def tpc_fit_tracks(ctx: int, params, d_workspace: int, workspace_bytes: int, cuda_stream: int) -> int:
    return load_library().tpc_fit_tracks(ctx, C.byref(params) if params is not None else None, d_workspace,
                                         workspace_bytes, cuda_stream)


TPC_E_LIMIT = -6
TPC_FIT_NOALLOC_MAX_IDS = 1 << 20


def tpc_fit_tracks_noalloc(ctx: int, params, d_clusters: int, n_clusters: int, d_refit: int, n_tracks: int, d_merged: int,
                           n_merged: int, d_seg_index: int, d_cluster_ids: int, n_cluster_ids: int, d_fit_out: int,
                           d_chi2_out: int, d_rejected_out: int, flags: int, cuda_stream: int) -> int:
    """The three-iteration fit with every input / output passed as a device pointer and the scratch inside
    the library (no workspace, no allocation; at most TPC_FIT_NOALLOC_MAX_IDS cluster ids)."""
    return load_library().tpc_fit_tracks_noalloc(ctx, C.byref(params) if params is not None else None, d_clusters, n_clusters,
                                                 d_refit, n_tracks, d_merged, n_merged, d_seg_index, d_cluster_ids,
                                                 n_cluster_ids, d_fit_out, d_chi2_out, d_rejected_out, flags, cuda_stream)


def tpc_get_fit(ctx: int):
    v = FitView()
    rc = load_library().tpc_get_fit(ctx, C.byref(v))
    return rc, v


def tpc_set_tracks(ctx: int, h_tracks: int, n_tracks: int, h_cluster_ids: int, h_cluster_shared: int, n_cluster_ids: int,
                   cuda_stream: int) -> int:
    return load_library().tpc_set_tracks(ctx, h_tracks, n_tracks, h_cluster_ids, h_cluster_shared, n_cluster_ids, cuda_stream)


def tpc_rebuild_default_params(**overrides) -> RebuildParams:
    r = RebuildParams()
    load_library().tpc_rebuild_default_params(C.byref(r))
    for k, v in overrides.items():
        setattr(r, k, v)
    return r


def tpc_rebuild_prepare(ctx: int, cuda_stream: int):
    n = C.c_uint64(0)
    rc = load_library().tpc_rebuild_prepare(ctx, cuda_stream, C.byref(n))
    return rc, int(n.value)


def tpc_rebuild_workspace_bytes(ctx: int, n_steps: int, n_merged: int, n_clusters: int) -> int:
    return int(load_library().tpc_rebuild_workspace_bytes(ctx, n_steps, n_merged, n_clusters))


def tpc_rebuild_tracks(ctx: int, params, d_workspace: int, workspace_bytes: int, cuda_stream: int) -> int:
    return load_library().tpc_rebuild_tracks(ctx, C.byref(params) if params is not None else None, d_workspace,
                                             workspace_bytes, cuda_stream)


def tpc_get_rebuild(ctx: int):
    v = RebuildView()
    rc = load_library().tpc_get_rebuild(ctx, C.byref(v))
    return rc, v


def tpc_last_launch_count(ctx: int) -> int:
    return load_library().tpc_last_launch_count(ctx)


def tpc_destroy(ctx: int) -> None:
    load_library().tpc_destroy(ctx)


def tpc_last_cuda_error(ctx: int) -> str:
    return load_library().tpc_last_cuda_error(ctx).decode()


# ---------------------------------------------------------------- convenience class
class SectorTracker:
    """One context + one workspace.  ``track(d_clusters)`` enqueues the path on a stream;
    ``tracks()`` / ``intermediates()`` synchronise and return arrays."""

    def __init__(self, geom: GeomDesc | None = None, params: Params | None = None, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("SectorTracker needs a CUDA device (there is no CPU fallback)")
        self.torch = torch
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self.geom = geom or default_geom()
        self.params = params
        self.ctx = tpc_geom_init(self.geom, params)
        self.workspace = None
        self._clusters = None
        self.n = 0

    def close(self):
        if self.ctx:
            tpc_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def upload(self, clusters: np.ndarray):
        """Host structured array (16-byte records) -> device uint8 tensor."""
        assert clusters.dtype.itemsize == 16
        t = self.torch.from_numpy(np.ascontiguousarray(clusters).view(np.uint8).reshape(-1))
        return t.to(self.device)

    def ensure_workspace(self, n: int):
        need = tpc_workspace_bytes(self.ctx, n)
        if need == 0 and n:
            raise TpcError(TPC_E_ARG, "tpc_workspace_bytes")
        if self.workspace is None or self.workspace.numel() < need:
            self.workspace = None
            self.workspace = self.torch.empty(need + 256, dtype=self.torch.uint8, device=self.device)
        return need

    def track(self, d_clusters, flags: int = 0, stream=None) -> None:
        """d_clusters: device uint8 tensor holding n 16-byte cluster records."""
        n = d_clusters.numel() // 16
        need = self.ensure_workspace(n)
        ws_ptr = (self.workspace.data_ptr() + 255) // 256 * 256
        st = stream if stream is not None else self.torch.cuda.current_stream(self.device)
        rc = tpc_sector_track(self.ctx, d_clusters.data_ptr(), n, ws_ptr, need, st.cuda_stream, flags)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_sector_track", tpc_last_cuda_error(self.ctx))
        self._clusters = d_clusters  # keep alive until the results are read
        self.n = n

    def _view(self, ptr: int, nbytes: int):
        off = ptr - self.workspace.data_ptr()
        assert 0 <= off and off + nbytes <= self.workspace.numel()
        return self.workspace[off:off + nbytes]

    def _to_numpy(self, ptr: int, count: int, dtype) -> np.ndarray:
        dtype = np.dtype(dtype)
        if count == 0:
            return np.zeros(0, dtype=dtype)
        return self._view(ptr, count * dtype.itemsize).cpu().numpy().view(dtype).copy()

    def counts(self, check: bool = True):
        rc, v = tpc_get_tracks(self.ctx)
        if check and rc != TPC_OK:
            raise TpcError(rc, "tpc_get_tracks", tpc_last_cuda_error(self.ctx))
        return rc, v

    def tracks(self):
        """Synchronise and copy out (tracks, cluster_ids, cluster_shared, view)."""
        rc, v = self.counts()
        tr = self._to_numpy(v.d_tracks, v.n_tracks, TRACK_DTYPE)
        ids = self._to_numpy(v.d_cluster_ids, v.n_cluster_ids, np.uint32)
        sh = self._to_numpy(v.d_cluster_shared, v.n_cluster_ids, np.uint8)
        return tr, ids, sh, v

    def stage_ms(self) -> dict:
        rc, ms = tpc_get_stage_ms(self.ctx)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_get_stage_ms")
        return dict(zip(STAGE_NAMES, ms))

    def kernel_ms(self) -> list:
        rc, out = tpc_get_kernel_ms(self.ctx)
        if rc < 0:
            raise TpcError(rc, "tpc_get_kernel_ms")
        return out

    def track_two_iterations(self, d_clusters, flags: int = 0, stream=None) -> None:
        """The path plus a second seeding iteration on the leftover clusters; read the
        combined result with tracks()."""
        n = d_clusters.numel() // 16
        need = tpc_workspace_bytes_two_iterations(self.ctx, n)
        if self.workspace is None or self.workspace.numel() < need + 256:
            self.workspace = None
            self.workspace = self.torch.empty(need + 256, dtype=self.torch.uint8, device=self.device)
        ws_ptr = (self.workspace.data_ptr() + 255) // 256 * 256
        st = stream if stream is not None else self.torch.cuda.current_stream(self.device)
        rc = tpc_sector_track_two_iterations(self.ctx, d_clusters.data_ptr(), n, ws_ptr, need, st.cuda_stream, flags)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_sector_track_two_iterations", tpc_last_cuda_error(self.ctx))
        self.n = n
        self._clusters = d_clusters

    def refit(self, stream=None):
        """Sector-track refit of the current result; returns the tpc_track_fit records."""
        st = stream if stream is not None else self.torch.cuda.current_stream(self.device)
        rc = tpc_refit_tracks(self.ctx, st.cuda_stream)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_refit_tracks", tpc_last_cuda_error(self.ctx))
        rc, ptr = tpc_get_refit(self.ctx)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_get_refit", tpc_last_cuda_error(self.ctx))
        rc, v = self.counts()
        return self._to_numpy(ptr, v.n_tracks, TRACK_FIT_DTYPE)

    def merge(self, mparams: MergeParams | None = None, stream=None, fetch: bool = True):
        """Track merging (reading R9) of the current result; tpc_refit_tracks must have
        run on it (refit()).  Returns a dict of arrays (merged, seg_index, cluster_ids, cluster_shared,
        next, prev, link_chi2) or, with fetch=False, the view."""
        rc, v = self.counts()
        need = tpc_merge_workspace_bytes(self.ctx, v.n_tracks, v.n_cluster_ids)
        if getattr(self, "merge_ws", None) is None or self.merge_ws.numel() < need + 256:
            self.merge_ws = None
            self.merge_ws = self.torch.empty(need + 256, dtype=self.torch.uint8, device=self.device)
        ws_ptr = (self.merge_ws.data_ptr() + 255) // 256 * 256
        st = stream if stream is not None else self.torch.cuda.current_stream(self.device)
        rc = tpc_merge_tracks(self.ctx, mparams, ws_ptr, need, st.cuda_stream)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_merge_tracks", tpc_last_cuda_error(self.ctx))
        if not fetch:
            return None
        rc, mv = tpc_get_merged(self.ctx)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_get_merged", tpc_last_cuda_error(self.ctx))

        def arr(ptr, count, dtype):
            dtype = np.dtype(dtype)
            if count == 0:
                return np.zeros(0, dtype=dtype)
            off = ptr - self.merge_ws.data_ptr()
            return self.merge_ws[off:off + count * dtype.itemsize].cpu().numpy().view(dtype).copy()
        nt = int(mv.n_tracks)
        return dict(view=mv, merged=arr(mv.d_merged, int(mv.n_merged), MERGED_DTYPE),
                    seg_index=arr(mv.d_seg_index, nt, np.uint32),
                    cluster_ids=arr(mv.d_cluster_ids, int(mv.n_cluster_ids), np.uint32),
                    cluster_shared=arr(mv.d_cluster_shared, int(mv.n_cluster_ids), np.uint8),
                    next=arr(mv.d_next, nt, np.int32), prev=arr(mv.d_prev, nt, np.int32),
                    link_chi2=arr(mv.d_link_chi2, nt, np.float32))

    def fit(self, fparams: FitParams | None = None, stream=None, fetch: bool = True):
        """Three-iteration track fit with interpolation rejection (reading R10) of
        the merged tracks; merge() must have run.  Returns (fit records, chi2_cluster, rejected)."""
        rc, mv = tpc_get_merged(self.ctx)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_get_merged", tpc_last_cuda_error(self.ctx))
        need = tpc_fit_workspace_bytes(self.ctx, int(mv.n_merged), int(mv.n_cluster_ids))
        if getattr(self, "fit_ws", None) is None or self.fit_ws.numel() < need + 256:
            self.fit_ws = None
            self.fit_ws = self.torch.empty(need + 256, dtype=self.torch.uint8, device=self.device)
        ws_ptr = (self.fit_ws.data_ptr() + 255) // 256 * 256
        st = stream if stream is not None else self.torch.cuda.current_stream(self.device)
        rc = tpc_fit_tracks(self.ctx, fparams, ws_ptr, need, st.cuda_stream)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_fit_tracks", tpc_last_cuda_error(self.ctx))
        if not fetch:
            return None
        rc, fv = tpc_get_fit(self.ctx)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_get_fit", tpc_last_cuda_error(self.ctx))

        def arr(ptr, count, dtype):
            dtype = np.dtype(dtype)
            if count == 0:
                return np.zeros(0, dtype=dtype)
            off = ptr - self.fit_ws.data_ptr()
            return self.fit_ws[off:off + count * dtype.itemsize].cpu().numpy().view(dtype).copy()
        return (arr(fv.d_fit, int(fv.n_merged), TRACK_FIT3_DTYPE), arr(fv.d_chi2_cluster, int(fv.n_cluster_ids), np.float32),
                arr(fv.d_rejected, int(fv.n_cluster_ids), np.uint8))

    def set_tracks(self, tracks, cluster_ids, cluster_shared, stream=None):
        """Loads sector tracks of the current frame that were made elsewhere (tpc_set_tracks): numpy
        arrays TRACK_DTYPE / uint32 / uint8 with frame cluster indices."""
        st = stream if stream is not None else self.torch.cuda.current_stream(self.device)
        t = np.ascontiguousarray(tracks, dtype=TRACK_DTYPE)
        i = np.ascontiguousarray(cluster_ids, dtype=np.uint32)
        s = np.ascontiguousarray(cluster_shared, dtype=np.uint8)
        if len(i) != len(s):
            raise ValueError("cluster_ids and cluster_shared differ in length")
        rc = tpc_set_tracks(self.ctx, t.ctypes.data, len(t), i.ctypes.data, s.ctypes.data, len(i), st.cuda_stream)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_set_tracks", tpc_last_cuda_error(self.ctx))

    def rebuild(self, rparams: RebuildParams | None = None, stream=None, fetch: bool = True):
        """Phase-II track rebuild (reading R11) of the merged tracks; merge() must have
        run and the tracking workspace must be intact.  Returns a dict of arrays."""
        st = stream if stream is not None else self.torch.cuda.current_stream(self.device)
        rc, n_steps = tpc_rebuild_prepare(self.ctx, st.cuda_stream)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_rebuild_prepare", tpc_last_cuda_error(self.ctx))
        rc, mv = tpc_get_merged(self.ctx)
        need = tpc_rebuild_workspace_bytes(self.ctx, n_steps, int(mv.n_merged), self.n)
        if getattr(self, "rebuild_ws", None) is None or self.rebuild_ws.numel() < need + 256:
            self.rebuild_ws = None
            self.rebuild_ws = self.torch.empty(need + 256, dtype=self.torch.uint8, device=self.device)
        ws_ptr = (self.rebuild_ws.data_ptr() + 255) // 256 * 256
        rc = tpc_rebuild_tracks(self.ctx, rparams, ws_ptr, need, st.cuda_stream)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_rebuild_tracks", tpc_last_cuda_error(self.ctx))
        if not fetch:
            return None
        rc, rv = tpc_get_rebuild(self.ctx)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_get_rebuild", tpc_last_cuda_error(self.ctx))

        def arr(buf, ptr, count, dtype):
            dtype = np.dtype(dtype)
            if count == 0:
                return np.zeros(0, dtype=dtype)
            off = ptr - buf.data_ptr()
            return buf[off:off + count * dtype.itemsize].cpu().numpy().view(dtype).copy()
        ns, nm = int(rv.n_steps), int(rv.n_merged)
        w = self.rebuild_ws
        return dict(view=rv, step_ofs=arr(self.merge_ws, rv.d_step_ofs, nm + 1, np.uint32) if nm else np.zeros(1, np.uint32),
                    cand_id=arr(w, rv.d_cand_id, 3 * ns, np.int32).reshape(-1, 3),
                    cand_chi2=arr(w, rv.d_cand_chi2, 3 * ns, np.float32).reshape(-1, 3),
                    attached=arr(w, rv.d_attached, ns, np.int32), shared=arr(w, rv.d_shared, ns, np.uint8),
                    used=arr(w, rv.d_used, ns, np.uint8), fit=arr(w, rv.d_fit, nm, TRACK_FIT3_DTYPE))

    def track_host(self, h_clusters, d_staging, h_tracks, h_ids, h_shared, flags: int = 0, stream=None):
        """End-to-end call with HOST buffers (torch CPU tensors, pinned for speed): copies the
        clusters in, tracks, copies tracks / cluster ids / shared flags out.  Returns the view."""
        n = h_clusters.numel() // 16
        need = self.ensure_workspace(n)
        ws_ptr = (self.workspace.data_ptr() + 255) // 256 * 256
        st = stream if stream is not None else self.torch.cuda.current_stream(self.device)
        rc, v = tpc_sector_track_host(self.ctx, h_clusters.data_ptr(), n, d_staging.data_ptr(), ws_ptr, need,
                                      st.cuda_stream, flags, h_tracks.data_ptr(),
                                      h_tracks.numel() // TRACK_DTYPE.itemsize, h_ids.data_ptr(),
                                      h_shared.data_ptr(), min(h_ids.numel() // 4, h_shared.numel()))
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_sector_track_host", tpc_last_cuda_error(self.ctx))
        self.n = n
        return v

    def track_host_chunks(self, h_clusters, chunk_ofs, d_staging, h_tracks, h_ids, h_shared, flags: int = 0,
                          stream=None):
        """track_host for a frame given as consecutive chunks of whole sectors (chunk_ofs: record
        offsets, first 0, last n): copy-in, tracking and copy-out of successive chunks overlap."""
        n = h_clusters.numel() // 16
        n_max = max(int(chunk_ofs[i + 1]) - int(chunk_ofs[i]) for i in range(len(chunk_ofs) - 1))
        one = (tpc_workspace_bytes(self.ctx, n_max) + 255) // 256 * 256
        need = 2 * one
        if self.workspace is None or self.workspace.numel() < need + 256:
            self.workspace = None
            self.workspace = self.torch.empty(need + 256, dtype=self.torch.uint8, device=self.device)
        ws_ptr = (self.workspace.data_ptr() + 255) // 256 * 256
        st = stream if stream is not None else self.torch.cuda.current_stream(self.device)
        rc, v = tpc_sector_track_host_chunks(self.ctx, h_clusters.data_ptr(), n, chunk_ofs, d_staging.data_ptr(), ws_ptr,
                                             need, st.cuda_stream, flags, h_tracks.data_ptr(),
                                             h_tracks.numel() // TRACK_DTYPE.itemsize, h_ids.data_ptr(),
                                             h_shared.data_ptr(), min(h_ids.numel() // 4, h_shared.numel()))
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_sector_track_host_chunks", tpc_last_cuda_error(self.ctx))
        self.n = n
        return v

    def launch_count(self) -> int:
        return tpc_last_launch_count(self.ctx)

    def intermediates(self) -> dict:
        """Everything tpc_get_intermediates exposes, as numpy arrays (needs the run to have
        been made with TPC_KEEP_INTERMEDIATES)."""
        rc, v = tpc_get_intermediates(self.ctx)
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_get_intermediates", tpc_last_cuda_error(self.ctx))
        ns, nb, nseeds, stride = v.n_sorted, v.n_bins, v.n_seeds, v.tracklet_stride
        out = dict(n_sorted=ns, n_bins=nb, n_seeds=nseeds)
        out["row_desc"] = self._to_numpy(v.d_row_desc, v.n_rows_total, ROW_DESC_DTYPE)
        out["bin_start"] = self._to_numpy(v.d_bin_start, nb + 1, np.uint32)
        out["yz_sorted"] = self._to_numpy(v.d_yz_sorted, 2 * ns, np.float32).reshape(-1, 2)
        out["orig_id"] = self._to_numpy(v.d_orig_id, ns, np.uint32)
        for k in ("link_up", "link_dn", "link_up2", "link_dn2"):
            out[k] = self._to_numpy(getattr(v, "d_" + k), ns, np.int32)
        out["seeds"] = self._to_numpy(v.d_seeds, nseeds, np.uint32)
        out["tracklets"] = self._to_numpy(v.d_tracklets, nseeds, TRACKLET_DTYPE)
        n_rows = self.geom.n_rows
        if nseeds:
            rh = self._view(v.d_row_hit, 4 * nseeds * stride).view(self.torch.int32).reshape(nseeds, stride)
            out["row_hit"] = rh[:, :n_rows].contiguous().cpu().numpy()
        else:
            out["row_hit"] = np.zeros((0, n_rows), dtype=np.int32)
        return out
