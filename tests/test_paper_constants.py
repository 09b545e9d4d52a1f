"""The few numbers the paper prints for the hot path (tests/golden/paper_constants.txt, each
with its citation) against the input recipe and the defaults of BOTH sides: a wrong preset or
default (events per frame, drift window, shared fraction, findable cut) fails here."""
import os

import numpy as np

import oracle
from paper_2601_20569_b200 import datagen as dg
from paper_2601_20569_b200 import metrics


def _golden():
    out = {}
    path = os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")
    for ln in open(path):
        ln = ln.split("#")[0].strip()
        if ln:
            k, v = (x.strip() for x in ln.split("="))
            out[k] = float(v)
    return out


def test_recipe_follows_the_papers_numbers():
    g = _golden()
    c3, c4 = dg.preset("C3"), dg.preset("C4")
    # collisions in one drift time / in one time frame at the paper's interaction rate
    assert c3.t_window_us == g["drift_time_us"] and c3.n_events == g["collisions_per_drift_time"]
    assert c4.t_window_us == g["time_frame_ms"] * 1e3
    assert c4.n_events == round(g["interaction_rate_khz"] * g["time_frame_ms"])          # 140
    # 32 LHC orbits (88.92 us each) are the ~2.8 ms of the paper
    assert abs(g["time_frame_orbits"] * 88.92e-3 - g["time_frame_ms"]) < 0.05
    # same collision density in C3 and C4: events per microsecond
    assert abs(c3.n_events / c3.t_window_us - c4.n_events / c4.t_window_us) < 1e-9


def test_defaults_follow_the_papers_numbers():
    g = _golden()
    p = oracle.default_params()
    assert p.shared_permille == 10 * g["shared_fraction_default_pct"]
    from paper_2601_20569_b200 import binding as B      # host-only call, no GPU needed
    q = B.tpc_default_params()
    assert q.shared_permille == 10 * g["shared_fraction_default_pct"]
    assert B.tpc_default_params(shared_permille=int(10 * g["shared_fraction_loose_pct"])).shared_permille == 200
    geom = oracle.default_geom() if hasattr(oracle, "default_geom") else None
    if geom is not None:
        assert geom.n_sectors == g["sectors"]
    assert metrics.FINDABLE_MIN_HITS == g["findable_min_hits"]
