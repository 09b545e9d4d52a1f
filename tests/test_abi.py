"""The C-ABI library loads and exports every symbol include/tpc_track.h declares (no compute
calls: this runs without a GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_header_symbols():
    from paper_2601_20569_b200 import build, binding
    path = build.build_tpctrack()
    lib = ctypes.CDLL(path)
    header = open(os.path.join(ROOT, "include", "tpc_track.h")).read()
    declared = set(re.findall(r"\b(tpc_[a-z_]+)\s*\(", header))
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_struct_layouts_match_header():
    from paper_2601_20569_b200 import binding as B
    assert B.CLUSTER_DTYPE.itemsize == 16
    assert B.TRACK_DTYPE.itemsize == 108 and B.TRACKLET_DTYPE.itemsize == 112
    assert ctypes.sizeof(B.GeomDesc) == 40
    assert ctypes.sizeof(B.Params) == 120
    assert B.Params.max_bins.offset == 96 and B.Params.max_seeds.offset == 104
    assert ctypes.sizeof(B.TrackView) == 192 and ctypes.sizeof(B.DebugView) == 136
    assert B.TRACK_FIT_DTYPE.itemsize == 192 and B.MERGED_DTYPE.itemsize == 40
    assert ctypes.sizeof(B.MergeParams) == 60 and ctypes.sizeof(B.MergedView) == 88
    assert B.TRACK_FIT3_DTYPE.itemsize == 100 and ctypes.sizeof(B.FitParams) == 12 and ctypes.sizeof(B.FitView) == 40
    f = B.tpc_fit_default_params()
    assert abs(f.fit_chi2_max - 16.0) < 1e-6 and f.fit_min_clusters == 10
    assert ctypes.sizeof(B.RebuildParams) == 16 and ctypes.sizeof(B.RebuildView) == 72
    assert abs(B.tpc_rebuild_default_params().cand_chi2_max - 16.0) < 1e-6
    m = B.tpc_merge_default_params()
    assert m.gap_in_sector == 30 and abs(m.chi2_max - 20.0) < 1e-6 and m.stages == 7


def test_host_only_calls_without_gpu():
    """tpc_default_params / tpc_strerror / argument checks need no device."""
    from paper_2601_20569_b200 import binding as B
    p = B.tpc_default_params()
    assert abs(p.err_y - 0.1) < 1e-7 and p.shared_permille == 100 and p.min_hits_track == 20
    L = B.load_library()
    assert b"workspace" in L.tpc_strerror(B.TPC_E_WORKSPACE)
    ctx = ctypes.c_void_p()
    bad = B.default_geom(n_rows=2)
    assert L.tpc_geom_init(ctypes.byref(bad), None, ctypes.byref(ctx)) == B.TPC_E_ARG
    assert L.tpc_workspace_bytes(None, 10) == 0


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2601_20569_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h", ".cuh")):
                src = open(os.path.join(dirpath, f), errors="ignore").read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "tpc_oracle" not in src and "liboracle" not in src, f
