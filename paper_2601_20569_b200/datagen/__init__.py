"""Seeded synthetic TPC time frames (input generation only).

This package feeds BOTH the CUDA path and the CPU oracle; it holds none of the tracking
method's arithmetic and imports neither of them.  The generator itself is C++
(``tpcgen.cpp``, built into ``libtpcgen.so`` next to this file); this module only holds the
five workload presets of ``BASELINE.json`` (``configs[0..4]`` = C1..C5, concretised in
DESIGN.md "Input recipe") and marshals arguments.

    clusters, labels, truth = generate(preset("C1"))

``clusters`` is a numpy structured array with the 16-byte layout of ``tpc_cluster``
(include/tpc_track.h), grouped by (sector, row); ``labels`` = particle*8+leg per cluster
(-1 = noise; never shown to the tracker); ``truth`` one record per generated particle.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, asdict, replace

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libtpcgen.so")
_SRC_PATH = os.path.join(_HERE, "tpcgen.cpp")

CLUSTER_DTYPE = np.dtype(
    [("y", "<f4"), ("z", "<f4"), ("q", "<f4"), ("sector", "u1"), ("row", "u1"), ("flags", "<u2")]
)
TRUTH_DTYPE = np.dtype(
    [("event", "<i4"), ("charge", "<i4"), ("pt", "<f4"), ("phi0", "<f4"), ("tanl", "<f4"),
     ("t_coll_us", "<f4"), ("n_clusters", "<i4"), ("pad", "<i4")]
)
assert CLUSTER_DTYPE.itemsize == 16 and TRUTH_DTYPE.itemsize == 32


class _CConfig(ctypes.Structure):
    _fields_ = [
        ("seed", ctypes.c_uint64),
        ("n_events", ctypes.c_int32),
        ("tracks_per_event", ctypes.c_int32),
        ("n_rows", ctypes.c_int32),
        ("row_lo", ctypes.c_int32),
        ("row_hi", ctypes.c_int32),
        ("single_sector", ctypes.c_int32),
        ("r_min", ctypes.c_float),
        ("r_max", ctypes.c_float),
        ("half_angle_deg", ctypes.c_float),
        ("z_max", ctypes.c_float),
        ("bz_tesla", ctypes.c_float),
        ("pt_mean", ctypes.c_float),
        ("pt_lo", ctypes.c_float),
        ("pt_hi", ctypes.c_float),
        ("pt_uniform", ctypes.c_int32),
        ("eta_max", ctypes.c_float),
        ("looper_frac", ctypes.c_float),
        ("looper_lo", ctypes.c_float),
        ("looper_hi", ctypes.c_float),
        ("smear_y", ctypes.c_float),
        ("smear_z", ctypes.c_float),
        ("p_hit", ctypes.c_float),
        ("noise_frac", ctypes.c_float),
        ("noise_inner_peaked", ctypes.c_int32),
        ("t_window_us", ctypes.c_float),
        ("v_drift", ctypes.c_float),
        ("distortion", ctypes.c_int32),
        ("dist_r", ctypes.c_float),
        ("dist_y", ctypes.c_float),
        ("n_threads", ctypes.c_int32),
        ("max_turns", ctypes.c_int32),
    ]


@dataclass(frozen=True)
class GenConfig:
    """Knobs of the generator; see tpcgen.cpp for their meaning."""
    seed: int = 1
    n_events: int = 1
    tracks_per_event: int = 200
    n_rows: int = 152
    row_lo: int = 0
    row_hi: int = 152
    single_sector: int = -1
    r_min: float = 85.0
    r_max: float = 245.0
    half_angle_deg: float = 10.0
    z_max: float = 250.0
    bz_tesla: float = 0.5
    pt_mean: float = 0.6
    pt_lo: float = 0.1
    pt_hi: float = 10.0
    pt_uniform: int = 0
    eta_max: float = 0.9
    looper_frac: float = 0.0
    looper_lo: float = 0.05
    looper_hi: float = 0.15
    smear_y: float = 0.1
    smear_z: float = 0.1
    p_hit: float = 0.8
    noise_frac: float = 0.05
    noise_inner_peaked: int = 0
    t_window_us: float = 0.0
    v_drift: float = 2.58
    distortion: int = 0
    dist_r: float = 8.0
    dist_y: float = 1.0
    n_threads: int = 0
    max_turns: int = 3


_PRESETS = {
    # BASELINE.json configs[0]: 1 sector, 200 tracks from the origin, 5 % noise, seed 1
    "C1": GenConfig(seed=1, n_events=1, tracks_per_event=200, single_sector=0, noise_frac=0.05),
    # configs[1]: one central Pb-Pb-like event, 12000 tracks, 2 % loopers, 10 % noise
    "C2": GenConfig(seed=2, n_events=1, tracks_per_event=12000, looper_frac=0.02, noise_frac=0.10),
    # configs[2]: 100 us drift window, 5 overlapping events (the Poisson(5) mean), noise peaked inside
    "C3": GenConfig(seed=3, n_events=5, tracks_per_event=12000, looper_frac=0.02, noise_frac=0.10,
                    noise_inner_peaked=1, t_window_us=100.0),
    # configs[3]: 2.8 ms time frame, ~140 events, space-charge-like distortion, 10 % noise
    "C4": GenConfig(seed=4, n_events=140, tracks_per_event=12000, looper_frac=0.02, noise_frac=0.10,
                    t_window_us=2800.0, distortion=1),
    # configs[4]: inner-TPC stress, 1 sector, rows 0..62, 50000 low-pT tracks, 20 % noise
    "C5": GenConfig(seed=5, n_events=1, tracks_per_event=50000, single_sector=0, row_hi=63,
                    pt_uniform=1, pt_lo=0.05, pt_hi=0.5, smear_y=0.15, smear_z=0.15, noise_frac=0.20),
}


def preset(name: str, **overrides) -> GenConfig:
    """Return the GenConfig of workload C1..C5, optionally with fields overridden."""
    return replace(_PRESETS[name], **overrides)


def build(force: bool = False) -> str:
    """Compile tpcgen.cpp into libtpcgen.so (host code only)."""
    if (not force and os.path.exists(_LIB_PATH)
            and os.path.getmtime(_LIB_PATH) >= os.path.getmtime(_SRC_PATH)):
        return _LIB_PATH
    cmd = ["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-pthread", _SRC_PATH, "-o", _LIB_PATH]
    subprocess.run(cmd, check=True)
    return _LIB_PATH


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB_PATH)
        lib.tpcgen_run.restype = ctypes.c_void_p
        lib.tpcgen_run.argtypes = [ctypes.POINTER(_CConfig)]
        lib.tpcgen_n_clusters.restype = ctypes.c_int64
        lib.tpcgen_n_clusters.argtypes = [ctypes.c_void_p]
        lib.tpcgen_n_particles.restype = ctypes.c_int64
        lib.tpcgen_n_particles.argtypes = [ctypes.c_void_p]
        lib.tpcgen_fetch.restype = None
        lib.tpcgen_fetch.argtypes = [ctypes.c_void_p] * 4
        lib.tpcgen_free.restype = None
        lib.tpcgen_free.argtypes = [ctypes.c_void_p]
        _lib = lib
    return _lib


def generate(cfg: GenConfig, out_clusters: np.ndarray | None = None):
    """Run the generator.  Returns (clusters, labels, truth) numpy arrays.

    ``out_clusters``: optional preallocated CLUSTER_DTYPE array (e.g. a view of pinned
    memory) of sufficient size; the clusters are written into its head and a view returned.
    """
    lib = _load()
    c = _CConfig(**asdict(cfg))
    h = lib.tpcgen_run(ctypes.byref(c))
    try:
        n = lib.tpcgen_n_clusters(h)
        npart = lib.tpcgen_n_particles(h)
        if out_clusters is not None:
            assert out_clusters.dtype == CLUSTER_DTYPE and out_clusters.size >= n
            clusters = out_clusters[:n]
        else:
            clusters = np.empty(n, dtype=CLUSTER_DTYPE)
        labels = np.empty(n, dtype=np.int32)
        truth = np.empty(npart, dtype=TRUTH_DTYPE)
        lib.tpcgen_fetch(h, clusters.ctypes.data, labels.ctypes.data, truth.ctypes.data)
    finally:
        lib.tpcgen_free(h)
    return clusters, labels, truth
