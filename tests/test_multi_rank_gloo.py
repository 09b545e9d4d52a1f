"""N > 1 host logic on CPU (gloo, world_size 2): the path shards by independent time frames
(DESIGN.md section 8), so what runs across ranks is only the choice of each rank's frame and
the whole-job reductions of bench.py (sum of units, max of times).  The reference arm runs on
rank 0 alone."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    cfg, clusters, labels, _ = bench.make_frame("C1", rank, None, 60)
    n = len(clusters)
    ms_local = 10.0 * (rank + 1)                      # rank 1 is the slow one
    value, ms_total = bench.whole_job_value(n, ms_local, steps=2, world=world)
    all_n = [None] * world
    dist.all_gather_object(all_n, (n, int(cfg.seed), int(clusters["sector"].max())))
    if rank == 0:
        torch.save({"value": value, "ms_total": ms_total, "all": all_n}, out)
    dist.destroy_process_group()


def test_two_ranks_track_independent_frames_and_reduce(tmp_path):
    out = str(tmp_path / "r.pt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    r = torch.load(out)
    (n0, s0, _), (n1, s1, _) = r["all"]
    assert s1 == s0 + 1000 and n0 != n1               # different seeded frames per rank
    assert r["ms_total"] == 20.0                      # max over ranks
    assert np.isclose(r["value"], (n0 + n1) * 2 / 20e-3)   # all ranks' units / slowest rank's time


def test_reference_arm_runs_on_rank_zero_only(capsys):
    import bench

    class A:
        workload = "C1"; events = None; tracks = 40; oracle_budget = 10**6; warmup = 0; steps = 1; gpus = 2
    bench.run_reference(A, rank=1, world=2)
    assert capsys.readouterr().out == ""              # other ranks exit without work
    bench.run_reference(A, rank=0, world=2)
    line = capsys.readouterr().out.strip()
    import json
    d = json.loads(line)
    assert d["impl"] == "reference" and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"


def _split_worker(rank, world, port, out):
    """One frame over `world` ranks by sector: each rank tracks its sectors (the oracle stands in for
    the CUDA path on this CPU box: the subject here is the split / rebase / gather plumbing)."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_2601_20569_b200 import datagen as dg, multigpu as mg
    cl, _, _ = dg.generate(dg.preset("C2", tracks_per_event=1200, seed=21))
    sub, delta = mg.split_by_sector(cl, rank, world)
    o = oracle.run(sub, want=("tracks",))
    tracks, ids = mg.rebase(o.tracks, o.cluster_ids, delta)
    res = mg.gather_to_root(tracks, ids, o.cluster_shared, rank, world)
    if rank == 0:
        torch.save({"tracks": res[0], "ids": res[1], "shared": res[2], "n_sub": len(sub)}, out)
    else:
        assert res is None
    dist.destroy_process_group()


def test_one_frame_split_by_sector_over_two_ranks_equals_single_process(tmp_path):
    """SURVEY.md 8(e) first axis: sectors s mod 2 == r on rank r, variable-length gather to rank 0;
    the gathered result equals the single-process result byte for byte after canonical ordering."""
    import oracle
    from oracle import parity
    from paper_2601_20569_b200 import datagen as dg, multigpu as mg
    out = str(tmp_path / "split.pt")
    mp.spawn(_split_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    r = torch.load(out, weights_only=False)
    cl, _, _ = dg.generate(dg.preset("C2", tracks_per_event=1200, seed=21))
    ref = oracle.run(cl, n_threads=4, want=("tracks",))
    assert 0 < r["n_sub"] < len(cl)
    bad = parity.compare_tracks(r["tracks"], r["ids"], r["shared"], ref)
    assert parity.all_zero(bad), bad
    assert len(r["tracks"]) == ref.n_tracks and len(np.unique(r["tracks"]["sector"])) == 36
    # the split itself: every record lands on exactly one rank, offsets map back to the frame
    seen = np.zeros(len(cl), dtype=np.int32)
    for rank in range(3):
        sub, delta = mg.split_by_sector(cl, rank, 3)
        idx = np.arange(len(sub)) + delta[sub["sector"]]
        assert (cl[idx] == sub).all()
        seen[idx] += 1
    assert (seen == 1).all()
    # a frame that is not grouped by sector is refused
    import pytest
    with pytest.raises(ValueError):
        mg.split_by_sector(cl[::-1], 0, 2)
