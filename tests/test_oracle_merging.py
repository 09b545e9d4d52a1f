"""Pins of the merging oracle (reading R9; section 2: in-sector, adjacent sectors,
central electrode; section 3: on top of the sector-track refit).  References are closed
forms (exact straight-line / helix geometry in float64), hand-built cases and a second, plain-Python
implementation of the selection rule."""
import numpy as np
import pytest

import oracle
from oracle import merging
from paper_2601_20569_b200 import datagen as dg

R = 152


def frame(recs):
    """recs: (sector, row, y, z)"""
    c = np.zeros(len(recs), dtype=oracle.CLUSTER_DTYPE)
    a = np.array(recs, dtype=np.float64)
    c["sector"], c["row"], c["y"], c["z"] = a[:, 0], a[:, 1], a[:, 2], a[:, 3]
    return c


def track_and_merge(cl, mkw=None, **pkw):
    p = oracle.default_params(**pkw)
    o = oracle.run(cl, params=p, want=("tracks",))
    m = merging.merge(cl, o.tracks, o.cluster_ids, o.cluster_shared, params=p,
                      mparams=merging.default_merge_params(**(mkw or {})))
    return o, m


# ------------------------------------------------------------------ rotation (stage 2 transport)
def test_rotation_matches_exact_geometry_and_finite_differences():
    """A straight track (q/pT = 0) given on the plane x = 150 cm of sector s: the same line seen
    from sector s+1 (frame turned by +20 deg) in closed form: x' = x cos a + y sin a,
    y' = -x sin a + y cos a, phi' = phi - a; z, tan(lambda) unchanged.  Covariance: J C J^T with J
    from central finite differences (float64) of the exact map 'parameters on the plane x -> parameters
    on the plane x' = const through the rotated point'."""
    a = np.deg2rad(20.0)
    x, y, z, phi, t = 150.0, 21.0, -33.0, np.deg2rad(25.0), 0.7

    def exact(par, sign):
        yy, zz, s, tt, q = par
        ph = np.arcsin(s)
        al = sign * a
        # point and direction in the new frame
        xn, yn = x * np.cos(al) + yy * np.sin(al), -x * np.sin(al) + yy * np.cos(al)
        phn = ph - al
        # slide along the line to the plane x' = x0' (x0' from the unperturbed point)
        x0n = x * np.cos(al) + y * np.sin(al)
        d = x0n - xn
        return np.array([yn + d * np.tan(phn), zz + d * tt / np.cos(phn), np.sin(phn), tt, q]), x0n

    p0 = np.array([y, z, np.sin(phi), t, 0.0])
    rng = np.random.default_rng(1)
    A = rng.normal(size=(5, 5)) * np.array([0.1, 0.1, 0.01, 0.01, 0.05])[:, None]
    Cfull = A @ A.T
    tri = [(0, 0), (1, 0), (1, 1), (2, 0), (2, 1), (2, 2), (3, 0), (3, 1), (3, 2), (3, 3), (4, 0), (4, 1), (4, 2), (4, 3), (4, 4)]
    c15 = np.array([Cfull[i, j] for i, j in tri])
    for sign in (+1, -1):
        ref, x0n = exact(p0, sign)
        J = np.zeros((5, 5))
        for k in range(5):
            h = 1e-6
            dp = np.zeros(5); dp[k] = h
            J[:, k] = (exact(p0 + dp, sign)[0] - exact(p0 - dp, sign)[0]) / (2 * h)
        Cref = J @ Cfull @ J.T
        ok, st, xn = merging.rotate(np.concatenate([p0, c15]), x, sign)
        assert ok and abs(xn - x0n) < 1e-4
        assert np.allclose(st[:5], ref, atol=2e-5)
        got = np.array([st[5 + k] for k in range(15)])
        want = np.array([Cref[i, j] for i, j in tri])
        assert np.allclose(got, want, rtol=2e-4, atol=1e-9), (sign, got - want)
    # beyond the |sin phi| range the rotation refuses
    ok, _, _ = merging.rotate(np.concatenate([[0, 0, -0.9, 0, 0], c15]), x, +1)
    assert not ok


# ------------------------------------------------------------------ stage 1: inside a sector
def noise_free(seed_lo=11, want_rows=140):
    for seed in range(seed_lo, seed_lo + 60):
        cfg = dg.preset("C1", tracks_per_event=1, noise_frac=0.0, seed=seed, smear_y=0.0, smear_z=0.0,
                        p_hit=1.0, pt_lo=1.0, pt_hi=1.0001, pt_uniform=1)
        cl, _, _ = dg.generate(cfg)
        if len(cl) >= want_rows and len(np.unique(cl["row"])) == len(cl) and cl["row"].min() == 0:
            return cl
    raise AssertionError("no suitable track")


def test_split_track_merges_across_a_hole_but_not_across_a_wide_one():
    """A noise-free track with a 6-row hole (> max_gap_follow = 4) gives two sector tracks; stage 1
    joins them (gap 7 <= 30): ONE merged track holding all clusters in row order.  With a 35-row
    hole (gap 36 > 30) they stay apart."""
    cl = noise_free()
    r = cl["row"]
    sub = cl[~((r >= 60) & (r < 66))]
    o, m = track_and_merge(sub)
    assert o.n_tracks == 2
    assert len(m.merged) == 1 and m.merged[0]["n_segments"] == 2 and m.merged[0]["n_clusters"] == len(sub)
    assert np.array_equal(np.sort(sub["row"]), sub["row"][m.cluster_ids])           # ascending in row
    assert m.merged[0]["row_first"] == 0 and m.merged[0]["row_last"] == r.max()
    assert m.link_chi2.max() < 1.0                                                   # noise-free: a near-perfect match
    sub = cl[~((r >= 50) & (r < 85))]
    o, m = track_and_merge(sub)
    assert o.n_tracks == 2 and len(m.merged) == 2 and (m.next < 0).all()


def test_two_different_tracks_do_not_merge():
    """The lower half of one track and the upper half of ANOTHER track that runs 2 cm away in y:
    chi2 >= (2 / sqrt(C+C+0.3^2))^2 ~ 40 > 20 -> no link; at 0.2 cm distance they do link."""
    cl = noise_free()
    r = cl["row"]
    lo = cl[r < 60].copy()
    for dy, linked in ((2.0, False), (0.2, True)):
        hi = cl[r >= 66].copy()
        hi["y"] += np.float32(dy)
        o, m = track_and_merge(np.concatenate([lo, hi]))
        assert o.n_tracks == 2
        assert (len(m.merged) == 1) == linked, dy


def test_mutual_best_choice_and_tie_break():
    """One inner segment, two outer candidates: the exact continuation b1 and a copy b2 shifted by
    0.5 cm in z (chi2 ~ 2.5, inside the cut).  a's best is b1, b1's best is a -> link a-b1; b2 stays
    alone although it also matched.  With two IDENTICAL outer candidates the lower (seed id) wins."""
    cl = noise_free()
    r = cl["row"]
    a = cl[r < 60]
    b1 = cl[r >= 66].copy()
    b2 = b1.copy(); b2["z"] += np.float32(0.5)
    full = np.concatenate([a, b1, b2])
    o, m = track_and_merge(full, nf_max_d2=0.7)
    assert o.n_tracks == 3
    heads = m.merged[m.merged["n_segments"] == 2]
    assert len(heads) == 1 and len(m.merged) == 2
    ids = m.cluster_ids[heads[0]["cluster_ofs"]:heads[0]["cluster_ofs"] + heads[0]["n_clusters"]]
    assert ids.max() < len(a) + len(b1)                       # clusters of a and b1 only
    # exact tie: descriptors of two identical candidates handed to the matcher directly
    fit = oracle.refit_tracks(full, o.tracks, o.cluster_ids)
    mt = merging.merge_tracks_input(o.tracks, fit)
    ia = int(np.flatnonzero(mt["row_first"] == 0)[0])
    ib = int(np.flatnonzero(mt["row_first"] == 66)[0])
    tie = np.stack([mt[ia], mt[ib], mt[ib]]).copy()
    tie["seed_id"] = [5, 900, 100]
    nxt, prv, chi = merging.links(tie)
    assert nxt.tolist() == [2, -1, -1] and prv.tolist() == [-1, -1, 0]
    tie["seed_id"] = [5, 100, 900]
    nxt, prv, chi = merging.links(tie)
    assert nxt.tolist() == [1, -1, -1]


# ------------------------------------------------------------------ stage 2: adjacent sectors
def test_track_crossing_a_sector_edge_merges_after_rotation():
    """A noise-free 1 GeV/c helix that leaves sector 0 through its edge and continues in sector 1 (or
    17): the generator's exact helix is cut into two sector tracks; after the rotation by 20 deg and one
    propagation step to b's first row the states agree -> ONE merged track with all clusters; with
    stage 2 switched off they stay apart."""
    found = None
    for seed in range(100, 400):
        cfg = dg.preset("C2", tracks_per_event=1, noise_frac=0.0, seed=seed, smear_y=0.0, smear_z=0.0, p_hit=1.0,
                        pt_lo=1.0, pt_hi=1.0001, pt_uniform=1, looper_frac=0.0)
        cl, _, _ = dg.generate(cfg)
        secs = np.unique(cl["sector"])
        if len(secs) == 2 and all((cl["sector"] == s).sum() >= 40 for s in secs):
            found = cl
            break
    assert found is not None
    cl = found
    o, m = track_and_merge(cl)
    assert o.n_tracks == 2 and len(np.unique(o.tracks["sector"])) == 2
    assert len(m.merged) == 1 and m.merged[0]["n_segments"] == 2 and m.merged[0]["n_clusters"] == o.n_cluster_ids
    assert m.merged[0]["sector_first"] != m.merged[0]["sector_last"]
    assert m.link_chi2.max() < 2.0
    o, m = track_and_merge(cl, mkw=dict(stages=1))
    assert len(m.merged) == 2


# ------------------------------------------------------------------ stage 3: central electrode
def test_track_crossing_the_central_electrode():
    """Hand-built straight track at y = 2 cm: z_true = 0.5*(x_61.5 - x) falls through 0 between rows
    61 and 62; rows 20..61 are seen by sector 3 (A side) as z_true - 30 cm, rows 62..100 by sector 21
    (C side) as z_true + 30 cm (collision time 30 cm / v_drift, R0).  Where the track crosses the
    electrode z_A + z_C = 0 -> stage 3 links them; without stage 3 (stages = 3) nothing happens."""
    x, _, dx, _ = oracle.geom_tables()
    xm = 0.5 * (float(x[61]) + float(x[62]))
    recs = []
    for r in range(20, 101):
        zt = 0.5 * (xm - float(x[r]))
        recs.append((3, r, 2.0, zt - 30.0) if r <= 61 else (21, r, 2.0, zt + 30.0))
    cl = frame(recs)
    o, m = track_and_merge(cl)
    assert o.n_tracks == 2 and sorted(o.tracks["sector"].tolist()) == [3, 21]
    assert len(m.merged) == 1 and m.merged[0]["sector_first"] == 3 and m.merged[0]["sector_last"] == 21
    assert m.merged[0]["n_clusters"] == 81
    o, m = track_and_merge(cl, mkw=dict(stages=3))
    assert len(m.merged) == 2
    # a C-side piece whose z does not mirror (shifted by 20 cm: chi2 >= (20/3)^2 = 44 > 20) is not linked
    cl2 = cl.copy()
    cl2["z"][cl2["sector"] == 21] += np.float32(20.0)
    o, m = track_and_merge(cl2)
    assert len(m.merged) == 2


# ------------------------------------------------------------------ selection rule, second implementation
def test_stage1_links_equal_a_plain_python_implementation():
    """Stage 1 on a real frame (C2-like, distortion-free) redone in Python: transport by
    oracle.propagate (the pinned single step, fp32), chi2 with the diagonal variances + sys^2, cut,
    mutual best with the (seed id, segment) tie-break."""
    cl, _, _ = dg.generate(dg.preset("C2", tracks_per_event=2500, seed=12))
    o = oracle.run(cl, n_threads=4, want=("tracks",))
    fit = oracle.refit_tracks(cl, o.tracks, o.cluster_ids)
    mt = merging.merge_tracks_input(o.tracks, fit)
    mp = merging.default_merge_params(stages=1)
    nxt, prv, chi = merging.links(mt, mparams=mp)
    assert (nxt >= 0).sum() >= 20
    _, _, dx, cf = oracle.geom_tables()
    f32 = np.float32
    sys2 = np.array([f32(s) * f32(s) for s in mp.sys], dtype=f32)
    diag = [0, 2, 5, 9, 14]
    best_out, best_in = {}, {}
    key = lambda k: (int(mt["iter"][k]), int(mt["seed_id"][k]), int(mt["segment"][k]))
    for s_ in range(36):
        idx = np.flatnonzero((mt["sector"] == s_) & (mt["valid"] == 1))
        for a in idx:
            for b in idx:
                gap = int(mt["row_first"][b]) - int(mt["row_last"][a])
                if a == b or gap < 1 or gap > mp.gap_in_sector:
                    continue
                if not abs(f32(mt["p_in"][b][1]) - f32(mt["p_out"][a][1])) <= mp.pre_coarse_dz:
                    continue
                st = np.concatenate([mt["p_out"][a], mt["c_out"][a]]).astype(f32)
                ok = True
                for _ in range(gap):
                    ok, st, _j = oracle.propagate(st, dx, cf)
                    if not ok:
                        break
                if not ok:
                    continue
                if not (abs(f32(mt["p_in"][b][1] - st[1])) <= mp.pre_dz and abs(f32(mt["p_in"][b][0] - st[0])) <= mp.pre_dy):
                    continue
                c2 = f32(0)
                for i in range(5):
                    d = f32(mt["p_in"][b][i] - st[i])
                    var = f32(f32(st[5 + diag[i]] + mt["c_in"][b][diag[i]]) + sys2[i])
                    c2 = f32(c2 + f32(f32(d * d) / var))
                if not c2 <= mp.chi2_max:
                    continue
                if a not in best_out or (c2, key(b)) < best_out[a][:2]:
                    best_out[a] = (c2, key(b), b)
                if b not in best_in or (c2, key(a)) < best_in[b][:2]:
                    best_in[b] = (c2, key(a), a)
    want = np.full(len(mt), -1, dtype=np.int32)
    for a, (c2, _, b) in best_out.items():
        if best_in[b][2] == a:
            want[a] = b
    assert np.array_equal(want, nxt)
    linked = np.flatnonzero(nxt >= 0)
    assert np.array_equal(prv[nxt[linked]], linked)
    assert np.allclose(chi[linked], [best_out[a][0] for a in linked], rtol=0, atol=0)


def test_chains_are_simple_and_cover_every_track_once():
    cl, _, _ = dg.generate(dg.preset("C2", tracks_per_event=3000, seed=13))
    o = oracle.run(cl, n_threads=4, want=("tracks",))
    m = merging.merge(cl, o.tracks, o.cluster_ids, o.cluster_shared)
    assert sorted(m.seg_index.tolist()) == list(range(o.n_tracks))
    assert m.merged["n_clusters"].sum() == o.n_cluster_ids and m.merged["n_segments"].sum() == o.n_tracks
    stages_used = np.flatnonzero(m.next >= 0)
    assert len(stages_used) > 100
    # links raise the first row, join what the stage rules allow
    a, b = stages_used, m.next[stages_used]
    same = o.tracks["sector"][a] == o.tracks["sector"][b]
    assert (o.tracks["row_first"][b][same] > o.tracks["row_last"][a][same]).all()
    d18 = (o.tracks["sector"][a] % 18 - o.tracks["sector"][b] % 18) % 18
    assert np.isin(d18[~same], [1, 17]).all() and (o.tracks["sector"][a] // 18 == o.tracks["sector"][b] // 18).all()


def test_gap_bounds_of_stage_1():
    """1 <= row_first_b - row_last_a <= gap_in_sector, both ends inclusive: a 6-row hole is a gap of
    7 rows: linked with gap_in_sector = 7, not with 6; a 'gap' of 0 rows (b starts on a's last row)
    is never linked, even when the two end states are identical."""
    cl = noise_free()
    r = cl["row"]
    sub = cl[~((r >= 60) & (r < 66))]
    for g, linked in ((7, True), (6, False)):
        o, m = track_and_merge(sub, mkw=dict(gap_in_sector=g))
        assert (len(m.merged) == 1) == linked, g
    o = oracle.run(sub, want=("tracks",))
    mt = merging.merge_tracks_input(o.tracks, oracle.refit_tracks(sub, o.tracks, o.cluster_ids))
    ia, ib = int(np.flatnonzero(mt["row_first"] == 0)[0]), int(np.flatnonzero(mt["row_first"] == 66)[0])
    mt["row_first"][ib] = mt["row_last"][ia]
    mt["p_in"][ib], mt["c_in"][ib] = mt["p_out"][ia], mt["c_out"][ia]
    nxt, prv, _ = merging.links(mt)
    assert (nxt < 0).all()


def test_links_need_mutual_choice():
    """Two inner segments compete for ONE outer segment: a1 is the track's own lower half, a2 a copy
    of it shifted by 0.4 cm in z (chi2 ~ 1.6, inside the cut).  b's best partner is a1; a2's only
    candidate is b, but b did not choose it: a2 stays unlinked."""
    cl = noise_free()
    r = cl["row"]
    a1 = cl[r < 60]
    a2 = a1.copy(); a2["z"] += np.float32(0.4)
    b = cl[r >= 66]
    full = np.concatenate([a1, a2, b])
    o, m = track_and_merge(full)
    assert o.n_tracks == 3 and len(m.merged) == 2
    two = m.merged[m.merged["n_segments"] == 2][0]
    ids = m.cluster_ids[two["cluster_ofs"]:two["cluster_ofs"] + two["n_clusters"]]
    assert not np.any((ids >= len(a1)) & (ids < 2 * len(a1)))           # no cluster of a2
    assert (m.next >= 0).sum() == 1


def test_stages_run_in_the_papers_order_on_free_ends():
    """first inside the sectors, then adjacent sectors, then across the central electrode.
    The A-side piece a (sector 3, rows 20..61) of the electrode-crossing track has TWO possible
    continuations: b in its own sector (rows 68..100, stage 1) and c on the C side (sector 21, rows
    62..100, stage 3).  Stage 1 runs first and uses up a's outer end: a+b merge, c stays alone."""
    x, _, dx, _ = oracle.geom_tables()
    xm = 0.5 * (float(x[61]) + float(x[62]))
    recs = []
    for r in range(20, 101):
        zt = 0.5 * (xm - float(x[r]))
        if r <= 61:
            recs.append((3, r, 2.0, zt - 30.0))
        else:
            recs.append((21, r, 2.0, zt + 30.0))
            if r >= 68:
                recs.append((3, r, 2.0, zt - 30.0))
    cl = frame(recs)
    o, m = track_and_merge(cl)
    assert o.n_tracks == 3
    two = m.merged[m.merged["n_segments"] == 2]
    assert len(m.merged) == 2 and len(two) == 1
    assert two[0]["sector_first"] == 3 and two[0]["sector_last"] == 3 and two[0]["row_last"] == 100
