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
