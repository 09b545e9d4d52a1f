#!/usr/bin/env python
"""bench.py — throughput of the TPC sector-tracking hot path on B200 (BASELINE.json metric).

    python bench.py --gpus 1 --steps K --warmup W            # the CUDA path (this repo)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle, as it stands

One "step" = one pass of the whole hot path (grid -> neighbour finder -> link cleanup ->
seeds -> Kalman follower -> ambiguity solving) over one
synthetic time frame.  Default workload: BASELINE.json configs[3] (C4), the 2.8 ms Pb-Pb
time frame the metric is quoted on (~2.4e8 clusters, 3.8 GB, fits one B200).

N > 1 (torchrun, one rank per GPU): time frames are independent units (the
farm processes independent time frames), so every rank tracks its own frame (seed + rank),
no data-path collective; scaling = weak; value = all ranks' clusters / max-over-ranks time.

Prints ONE JSON line on rank 0 (contract in the task statement).
states the algorithmic bytes / flops behind the "roofline" object.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "TPC clusters/sec tracked per B200 (2.8 ms Pb-Pb time frame)"
UNIT = "clusters/s"

# ---- tracker parameters per workload (grid_* are performance knobs)
WORKLOAD_PARAMS = {
    "C1": dict(),
    "C2": dict(),
    "C3": dict(),
    "C4": dict(grid_dy=3.0, grid_dz=3.0),
    "C5": dict(err_y=0.15, err_z=0.15, nf_max_d2=1.6),
}

# ---- algorithmic work per kernel launch.
# HBM kernels: bytes as a function of (N input clusters, Ns clusters in the grid, NB bins,
# NSD seeds).  k_follow: fp32 flops from the work counters the kernel keeps.
FLOPS_PROPAGATE, FLOPS_UPDATE, FLOPS_GAIN_ROAD, FLOPS_CAND = 163, 112, 16, 13
FOLLOW_KERNELS = ("k_follow_up", "k_follow_refit", "k_follow_down")


def algorithmic_work(name: str, st: dict):
    N, Ns, NB, NSD, R = st["n"], st["n_sorted"], st["n_bins"], st["n_seeds"], st["n_rows"]
    H = st["follow_work"][0][1] + st["follow_work"][2][1] + NSD   # hits recorded in row_hit
    W, NT, NI = (R + 31) // 32, st["n_tracks"], st["n_ids"]
    hbm = {
        "k_row_stats": 16 * N,
        "k_row_sort": 16 * N + 12 * Ns + 4 * NB,         # records in (once; the re-reads are L2 by design), yz+id+bin_start out
        "k_zero_bins": 4 * NB,
        "k_bin_hist": 16 * N + 4 * N + 8 * Ns,          # cluster in, slot out, counter RMW
        "k_bin_scan": 8 * NB,
        "k_scatter": 16 * N + 4 * N + 4 * Ns + 12 * Ns,  # cluster+slot in, bin_start in, yz+id out
        "k_bin_sort": 4 * NB + 24 * Ns,
        "k_neighbours": 8 * Ns + 8 * Ns + 4 * NB,        # yz in (ideal reuse), links out, bin index
        "k_link_cleanup": 8 * Ns + 8 * Ns + 8 * Ns,      # links in, 2 gathers, links out
        "k_seed_flags": 8 * Ns + 1 * Ns,
        "k_seed_write": 1 * Ns + 4 * NSD,
        "k_zero_owner": 8 * Ns,
        "k_sel_owner": 32 * NSD + 12 * H,                # tracklet head, row_hit in, 8-byte atomic
        "k_sel_masks": 40 * NSD + 12 * H + 8 * W * NSD,  # key+head, row_hit + owner gather in, masks out
        "k_sel_count": 8 * W * NSD + 8 * NSD,            # masks in, counts out
        "k_sel_emit": 8 * NSD + (8 * W + 112 + 108 + 8 * W + 4) * NT,
        "k_sel_ids": (8 * W + 16) * NT + 13 * NI,        # masks, row_hit + orig_id gather in, ids + flags out
    }
    if name in hbm:
        return "hbm", float(hbm[name])
    if name in FOLLOW_KERNELS:
        steps, upd, cands = st["follow_work"][FOLLOW_KERNELS.index(name)]
        fl = (FLOPS_PROPAGATE * steps + FLOPS_UPDATE * upd + FLOPS_GAIN_ROAD * steps + FLOPS_CAND * cands)
        return "alu", float(fl)
    return "hbm", 0.0


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md)", 1965.0


# ------------------------------------------------------------------ clocks sampler
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, reasons, smax, pw = [], set(), None, []
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        try:
            for ln in open(self.path):
                f = [x.strip() for x in ln.split(",")]
                if len(f) < 7:
                    continue
                try:
                    sm.append(float(f[0]))
                    smax = float(f[1])
                    pw.append(float(f[2]))
                except ValueError:
                    continue
                for nm, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=smax, reasons=sorted(reasons), samples=len(sm),
                       power_w_max=max(pw) if pw else None)
        return out


# ------------------------------------------------------------------ workload
def make_frame(workload: str, rank: int, events: int | None, tracks: int | None):
    from paper_2601_20569_b200 import datagen as dg
    base = dg.preset(workload)
    kw = dict(seed=rank_seed(base.seed, rank))
    if events is not None:
        kw["n_events"] = events
        # a shorter frame at the SAME interaction rate (same cluster density per cm of drift)
        kw["t_window_us"] = base.t_window_us * events / base.n_events
    if tracks is not None:
        kw["tracks_per_event"] = tracks
    cfg = dg.preset(workload, **kw)
    t0 = time.time()
    clusters, labels, truth = dg.generate(cfg)
    return cfg, clusters, labels, time.time() - t0


def oracle_params(workload: str):
    import oracle
    return oracle.default_params(**WORKLOAD_PARAMS[workload])


def oracle_sample(clusters: np.ndarray, budget_clusters: int):
    """A bounded sample of the same workload for the CPU oracle: whole sectors (sectors are
    independent units), starting at sector 0, until ~budget_clusters clusters."""
    per_sector = np.bincount(clusters["sector"], minlength=36)
    present = [s for s in range(len(per_sector)) if per_sector[s]]
    lo = present[0]
    hi, tot = lo, 0
    for s in present:
        if tot and tot + per_sector[s] > budget_clusters:
            break
        tot += int(per_sector[s])
        hi = s + 1
    return lo, hi, tot


def time_oracle(clusters, workload, lo, hi, n_threads=1, want=("tracks",)):
    import oracle
    t0 = time.perf_counter()
    o = oracle.run(clusters, params=oracle_params(workload), sector_lo=lo, sector_hi=hi, n_threads=n_threads,
                   want=want)
    return time.perf_counter() - t0, o


# ------------------------------------------------------------------ the reference arm
def run_reference(args, rank, world):
    """--impl reference: the CPU oracle as it stands, on the box's host cores (rank 0 only)."""
    if rank != 0:
        return
    cfg, clusters, labels, gen_s = make_frame(args.workload, 0, args.events, args.tracks)
    lo, hi, n_sample = oracle_sample(clusters, args.oracle_budget)
    for _ in range(min(args.warmup, 1)):
        time_oracle(clusters, args.workload, lo, hi)
    times = []
    for _ in range(args.steps):
        dt, o = time_oracle(clusters, args.workload, lo, hi)
        times.append(dt)
    total = sum(times)
    value = n_sample * args.steps / total
    sample = f"sectors [{lo},{hi}) of the {args.workload} frame: {n_sample} of {len(clusters)} clusters per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{args.workload} (BASELINE.json configs[{int(args.workload[1]) - 1}])",
                   "n_clusters": int(len(clusters)), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------ N > 1: units and reductions
def rank_seed(base_seed: int, rank: int) -> int:
    """Every rank tracks its own independent time frame (no data-path collective)."""
    return base_seed + 1000 * rank


def reduce_over_ranks(x: float, op: str, world: int, device=None) -> float:
    """Whole-job figures: op = "max" for the time of the slowest rank, "sum" for the units."""
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_value(n_local: float, ms_local: float, steps: int, world: int, device=None):
    """value = units all ranks processed / max-over-ranks time; returns (value, ms_total)."""
    ms_total = reduce_over_ranks(ms_local, "max", world, device)
    n_all = reduce_over_ranks(float(n_local), "sum", world, device)
    return n_all * steps / (ms_total * 1e-3), ms_total


# ------------------------------------------------------------------ ONE frame over N GPUs by sector
def run_split_sectors(args, rank, world, local_rank, dev, barrier):
    """SURVEY.md 8(e), first axis (`--split sectors` under torchrun): every rank tracks the sectors
    s mod N == rank of the SAME frame (no collective inside the path), then one variable-length
    gather brings tracks + cluster lists to rank 0 (paper_2601_20569_b200/multigpu.py).  Strong
    scaling: value = the frame's clusters / (max over ranks of tracking + gather time)."""
    import torch
    import torch.distributed as dist
    from paper_2601_20569_b200 import binding as B, multigpu as mg
    cfg, clusters, labels, gen_s = make_frame(args.workload, 0, args.events, args.tracks)   # the same frame on every rank
    sub, delta = mg.split_by_sector(clusters, rank, world)
    pkw = dict(WORKLOAD_PARAMS[args.workload])
    trk = B.SectorTracker(params=B.tpc_default_params(**pkw), device=local_rank)
    stream = torch.cuda.Stream(device=dev)
    d_sub = trk.upload(sub)
    flags = B.TPC_DETERMINISTIC if args.mode == "det" else 0

    def step():
        trk.track(d_sub, flags=flags, stream=stream)
        tracks, ids, shared, v = trk.tracks()
        tracks, ids = mg.rebase(tracks, ids, delta)
        return mg.gather_to_root(tracks, ids, shared, rank, world, dev), v
    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            step()
    barrier()
    t0 = time.perf_counter()
    with torch.cuda.stream(stream):
        for _ in range(args.steps):
            res, v = step()
    barrier()
    ms_total = reduce_over_ranks((time.perf_counter() - t0) * 1e3, "max", world, dev)
    launches = trk.launch_count() * args.steps
    root_leg = None
    if rank == 0:
        # what the gather is for: the root builds the search grid of the whole frame only, loads the
        # gathered sector tracks (tpc_set_tracks) and runs refit + merging on them (timed apart)
        root = B.SectorTracker(params=B.tpc_default_params(**pkw), device=local_rank)
        d_all = root.upload(clusters)
        with torch.cuda.stream(stream):
            for it in range(2):
                torch.cuda.synchronize()
                t1 = time.perf_counter()
                root.track(d_all, flags=flags | B.TPC_GRID_ONLY, stream=stream)
                root.set_tracks(res[0], res[1], res[2], stream=stream)
                assert B.tpc_refit_tracks(root.ctx, stream.cuda_stream) == B.TPC_OK
                root.merge(stream=stream, fetch=False)
                rc_m, mv = B.tpc_get_merged(root.ctx)
                root_ms = (time.perf_counter() - t1) * 1e3
        root_leg = {"ms": root_ms, "what": "grid of the whole frame + tpc_set_tracks (host arrays) + refit + merging on rank 0",
                    "merged_tracks": int(mv.n_merged), "links": int(mv.n_links)}
        root.close()
    if rank == 0:
        n = len(clusters)
        print(json.dumps({
            "metric": METRIC, "value": n * args.steps / (ms_total * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{args.workload}, one frame split by sector over {world} ranks + gather to rank 0",
                       "n_clusters": n, "mode": args.mode, "n_tracks_gathered": int(len(res[0])),
                       "timing": "host clock around tracking + result read-back + gather, max over ranks"},
            "root_merging": root_leg, "gpu_launches": launches}), flush=True)
    trk.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


# ------------------------------------------------------------------ the CUDA arm
def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2601_20569_b200 import binding as B

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this path has no CPU fallback; use --impl reference "
                         "for the CPU oracle)")
    B.load_library()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x: float) -> float:
        return reduce_over_ranks(x, "max", world, dev)

    def sum_over_ranks(x: float) -> float:
        return reduce_over_ranks(x, "sum", world, dev)

    if args.split == "sectors":
        run_split_sectors(args, rank, world, local_rank, dev, barrier)
        return
    cfg, clusters, labels, gen_s = make_frame(args.workload, rank, args.events, args.tracks)
    n = len(clusters)
    flags = B.TPC_STAGE_TIMERS | (B.TPC_DETERMINISTIC if args.mode == "det" else 0)
    pkw = dict(WORKLOAD_PARAMS[args.workload])
    if args.grid_dy:
        pkw["grid_dy"] = args.grid_dy
    if args.grid_dz:
        pkw["grid_dz"] = args.grid_dz
    if args.max_bins:
        pkw["max_bins"] = args.max_bins
    trk = B.SectorTracker(params=B.tpc_default_params(**pkw), device=local_rank)
    stream = torch.cuda.Stream(device=dev)

    # pinned host copy of the frame (e2e leg) and the device-resident copy (kernel leg)
    h_clusters = torch.empty(n * 16, dtype=torch.uint8).pin_memory()
    h_clusters.numpy()[:] = clusters.view(np.uint8).reshape(-1)
    d_clusters = torch.empty(n * 16, dtype=torch.uint8, device=dev)
    d_clusters.copy_(h_clusters)
    ws_bytes = (B.tpc_workspace_bytes_two_iterations(trk.ctx, n) if args.second_iteration
                else trk.ensure_workspace(n))
    torch.cuda.synchronize()

    def step():
        if args.second_iteration:     # the path, then the path on the leftover clusters
            trk.track_two_iterations(d_clusters, flags=flags, stream=stream)
        else:
            trk.track(d_clusters, flags=flags, stream=stream)
        rc, v = trk.counts()          # tpc_get_tracks: syncs the stream, reads the counters
        return v

    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            v = step()
    kernel_ms: dict = {}
    order: list = []
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ev0 = torch.cuda.Event(enable_timing=True)
    ev1 = torch.cuda.Event(enable_timing=True)
    barrier()
    with torch.cuda.stream(stream):
        ev0.record(stream)
        for _ in range(args.steps):
            v = step()
            for name, ms in trk.kernel_ms():
                if name not in kernel_ms:
                    kernel_ms[name] = [0.0, 0]
                    order.append(name)
                kernel_ms[name][0] += ms
                kernel_ms[name][1] += 1
        ev1.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_total = max_over_ranks(ev0.elapsed_time(ev1))
    n_all = sum_over_ranks(float(n))
    launches = trk.launch_count() * args.steps
    stage_ms = trk.stage_ms()
    value = n_all * args.steps / (ms_total * 1e-3)

    refit = None

    if args.second_iteration:
        # reduced line: kernel times / roofline would describe the second pass only
        if rank == 0:
            print(json.dumps({
                "metric": METRIC + ", with a second seeding iteration on the leftover clusters", "value": value,
                "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": {"workload": f"{args.workload} + second iteration (SURVEY.md 8(f) row 1)", "n_clusters_per_gpu": n,
                           "mode": args.mode, "tracker_params": pkw, "n_tracks": int(v.n_tracks),
                           "n_seeds_both_iterations": int(v.n_seeds), "workspace_gb": ws_bytes / 1e9},
                "gpu_launches": launches}), flush=True)
        trk.close()
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- end-to-end: HOST buffers through the C ABI, copies inside the timed region
    cap_tracks = int(v.n_tracks * 1.05) + 1024
    cap_ids = int(v.n_cluster_ids * 1.05) + 1024
    h_tracks = torch.empty(cap_tracks * B.TRACK_DTYPE.itemsize, dtype=torch.uint8).pin_memory()
    h_ids = torch.empty(cap_ids * 4, dtype=torch.uint8).pin_memory()
    h_shared = torch.empty(cap_ids, dtype=torch.uint8).pin_memory()
    e2e_flags = flags & ~B.TPC_STAGE_TIMERS
    # the frame is handed over in chunks of whole sectors (sectors are independent units): copy-in,
    # tracking and copy-out of successive chunks overlap inside tpc_sector_track_host_chunks.  The
    # chunk offsets are part of the input's description (the generator emits sectors in order).
    sec = clusters["sector"]
    n_chunks = max(1, min(args.e2e_chunks or 1, int(sec.max()) + 1 if n else 1))
    cuts = [int(round((int(sec.max()) + 1) * c / n_chunks)) for c in range(n_chunks + 1)] if n else [0, 0]
    if args.e2e_cuts and n:       # explicit sector boundaries, e.g. "0,2,6,12,20,28,34,36"
        cuts = [int(x) for x in args.e2e_cuts.split(",")]
        n_chunks = len(cuts) - 1
    elif args.e2e_chunks == 0 and n >= 20_000_000:   # (small frames go in one shot: a chunk costs a host synchronisation)
        # default: small chunks first and last (short pipeline fill and drain), large ones between
        # (measured on the C4 frame: 112.0 ms against 119.7 ms for six equal chunks)
        ns = int(sec.max()) + 1
        cuts = sorted({int(round(ns * f)) for f in (0, 1 / 18, 1 / 6, 1 / 3, 5 / 9, 7 / 9, 17 / 18, 1)})
        n_chunks = len(cuts) - 1
    chunk_ofs = [int(x) for x in np.searchsorted(sec, cuts[:-1])] + [n]

    def e2e_step():
        if n_chunks > 1:
            return trk.track_host_chunks(h_clusters, chunk_ofs, d_clusters, h_tracks, h_ids, h_shared, flags=e2e_flags,
                                         stream=stream)
        return trk.track_host(h_clusters, d_clusters, h_tracks, h_ids, h_shared, flags=e2e_flags, stream=stream)

    with torch.cuda.stream(stream):
        for _ in range(min(args.warmup, 2)):
            ve = e2e_step()
    barrier()
    with torch.cuda.stream(stream):
        ev0.record(stream)
        for _ in range(args.steps):
            ve = e2e_step()
        ev1.record(stream)
    barrier()
    e2e_ms = max_over_ranks(ev0.elapsed_time(ev1))
    h2d = n * 16
    d2h = int(ve.n_tracks) * B.TRACK_DTYPE.itemsize + int(ve.n_cluster_ids) * 5 + 48
    e2e = {"value": n_all * args.steps / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms / args.steps,
           "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
           "call": f"tpc_sector_track_host_chunks, {n_chunks} chunks of whole sectors" if n_chunks > 1
                   else "tpc_sector_track_host"}

    if rank != 0:
        trk.close()
        if world > 1:
            dist.barrier()            # rank 0 prints after its CPU-side bookkeeping; leave together
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (live CUDA-event times over the timed region)
    hbm_peak, peak_src, sm_max_mhz = load_peaks()
    rc, iv = B.tpc_get_tracks(trk.ctx)
    st = dict(n=n, n_sorted=n - int(v.n_ignored) - int(v.n_dropped), n_bins=int(v.n_bins), n_seeds=int(v.n_seeds),
              n_rows=trk.geom.n_rows, follow_steps=int(v.n_follow_steps), follow_updates=int(v.n_follow_updates),
              follow_cands=int(v.n_follow_candidates), n_tracks=int(v.n_tracks), n_ids=int(v.n_cluster_ids),
              follow_work=[[int(v.follow_work[a][b]) for b in range(3)] for a in range(3)])
    per_kernel = []
    for name in order:
        tot, cnt = kernel_ms[name]
        per_step = tot / args.steps            # all launches of that name in one step
        bound, work = algorithmic_work(name, st)
        launches_per_step = cnt // args.steps
        per_kernel.append(dict(name=name, ms_per_step=per_step, launches_per_step=launches_per_step, bound=bound,
                               work_per_step=work * (1 if launches_per_step <= 1 else 1)))
    ksum = sum(k["ms_per_step"] for k in per_kernel)
    dom = max(per_kernel, key=lambda k: k["ms_per_step"])
    alu_peak_tflops = 148 * 128 * sm_max_mhz * 1e6 * (1 if args.mode == "det" else 2) / 1e12
    if dom["bound"] == "hbm":
        achieved = dom["work_per_step"] / (dom["ms_per_step"] * 1e-3) / 1e9
        roof = {"kernel": dom["name"], "bound": "hbm", "achieved": achieved, "peak": hbm_peak, "unit": "GB/s",
                "frac": achieved / hbm_peak, "traffic": None, "peak_source": peak_src}
    else:
        achieved = dom["work_per_step"] / (dom["ms_per_step"] * 1e-3) / 1e12
        roof = {"kernel": dom["name"], "bound": "alu", "achieved": achieved, "peak": alu_peak_tflops,
                "unit": "TFLOP/s", "frac": achieved / alu_peak_tflops, "traffic": None,
                "peak_source": "148 SM x 128 fp32 lanes x sm_max_mhz x (2 if FMA) — DESIGN.md"}
    roof["share_of_step"] = dom["ms_per_step"] / ksum if ksum else None
    traffic_file = os.path.join(ROOT, "profiles", "traffic.csv")   # from an ncu --set full capture (profiles/traffic.md)
    if os.path.exists(traffic_file):
        try:
            for ln in open(traffic_file).read().splitlines()[1:]:
                k, b = ln.split(",")
                if k == dom["name"]:
                    roof["traffic"] = float(b)
        except Exception:
            pass
    # north star: HBM fraction of the grid and neighbour stages
    stages = {}
    grid_names = ("k_row_stats", "k_row_desc", "k_row_sort", "k_zero_bins", "k_bin_hist", "k_bin_scan", "k_scatter", "k_bin_sort")
    # both grid paths are enqueued, the one k_row_desc did not choose returns at once: count only
    # the path that ran (the other's launches cost a few microseconds and move no data)
    kms = {k["name"]: k["ms_per_step"] for k in per_kernel}
    by_rows = kms.get("k_row_sort", 0.0) > kms.get("k_scatter", 0.0)
    idle = ("k_zero_bins", "k_bin_hist", "k_bin_scan", "k_scatter", "k_bin_sort") if by_rows else ("k_row_sort",)
    gb = sum(k["work_per_step"] for k in per_kernel if k["name"] in grid_names and k["name"] not in idle)
    gms = sum(k["ms_per_step"] for k in per_kernel if k["name"] in grid_names)
    nb = next((k for k in per_kernel if k["name"] == "k_neighbours"), None)
    if gms:
        stages["grid_path"] = "per-row build (k_row_sort)" if by_rows else "generic (histogram, scan, scatter)"
        stages["grid"] = {"ms": gms, "GB/s": gb / gms / 1e6, "frac_hbm": gb / gms / 1e6 / hbm_peak}
    if nb and nb["ms_per_step"]:
        stages["neighbours"] = {"ms": nb["ms_per_step"], "GB/s": nb["work_per_step"] / nb["ms_per_step"] / 1e6,
                                "frac_hbm": nb["work_per_step"] / nb["ms_per_step"] / 1e6 / hbm_peak}

    # ---- CPU baseline: the oracle as it stands on a bounded sample (rank 0, N=1 only)
    cpu = None
    cpu_all = None
    cpu_o, cpu_lo, cpu_hi = None, 0, 0
    if world == 1 and not args.no_cpu_baseline:
        lo, hi, n_sample = oracle_sample(clusters, args.oracle_budget)
        dt, o = time_oracle(clusters, args.workload, lo, hi, want=("seeds", "tracklets", "tracks"))
        cpu_o, cpu_lo, cpu_hi = o, lo, hi
        names = ("grid", "neighbours", "cleanup_seeds", "follower", "selector")
        cpu = {"value": n_sample / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
               "sample": f"sectors [{lo},{hi}) of the same {args.workload} frame: {n_sample} of {n} clusters, "
                         "single thread",
               "stage_seconds": {k: round(float(x), 3) for k, x in zip(names, o.stage_seconds)}}
        # the same oracle with the sectors spread over all host cores (one sector per thread)
        ncores = os.cpu_count() or 1
        per_sector = np.bincount(clusters["sector"], minlength=36)
        present = [s_ for s_ in range(len(per_sector)) if per_sector[s_]]
        if len(present) > 1 and ncores > 1:
            hi_all = present[min(ncores, len(present)) - 1] + 1
            n_all_s = int(per_sector[present[0]:hi_all].sum())
            n_thr = min(ncores, hi_all - present[0])
            dta, _oa = time_oracle(clusters, args.workload, present[0], hi_all, n_threads=n_thr)
            del _oa
            cpu_all = {"value": n_all_s / dta, "unit": UNIT, "cores": n_thr, "host_cores": ncores, "kind": "oracle",
                       "seconds": dta,
                       "sample": f"sectors [{present[0]},{hi_all}) of the same frame on {n_thr} threads (one sector each): "
                                 f"{n_all_s} of {n} clusters"}

    # ---- further legs on the same resident frame (rank 0, N = 1; a few steps each; none is part of `value`)
    extras = {}
    parity_obj = None
    if world == 1 and not args.no_extras:
        ex_steps = max(1, min(args.steps, 3))

        def timed(fn, sync):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(stream):
                fn(); sync()
                e0.record(stream)
                for _ in range(ex_steps):
                    fn()
                e1.record(stream)
                sync()
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) / ex_steps
        # (1) the fast result of the sampled sectors against the oracle's (the parity sample of the headline build)
        with torch.cuda.stream(stream):
            trk.track(d_clusters, flags=flags & ~B.TPC_STAGE_TIMERS, stream=stream)
            g_tracks, g_ids, g_shared, gv = trk.tracks()
        if cpu is not None and args.mode == "fast":
            # tracklet level on the sampled sectors tracked alone with intermediates kept (where every
            # decision of the follower coincides, parameters must agree), track level on the frame's run
            from oracle import parity as op_
            sel = (clusters["sector"] >= cpu_lo) & (clusters["sector"] < cpu_hi)
            base = int(np.flatnonzero(sel)[0])
            t2 = B.SectorTracker(params=B.tpc_default_params(**pkw), device=local_rank)
            t2.track(t2.upload(clusters[sel]), flags=B.TPC_KEEP_INTERMEDIATES)
            gi = t2.intermediates()
            t2.close()
            gi["orig_id"] = gi["orig_id"] + np.uint32(base)
            gi["tracklets"]["seed_id"] += np.uint32(base)
            tls, identical = op_.compare_tracklets_fast(gi, cpu_o)
            del gi
            m = (g_tracks["sector"] >= cpu_lo) & (g_tracks["sector"] < cpu_hi)
            stp = op_.compare_tracks_fast(g_tracks[m], g_ids, g_shared, cpu_o, identical_tracklets=identical)
            parity_obj = {"what": f"fast build vs oracle, sectors [{cpu_lo},{cpu_hi}) of this frame (DESIGN.md section 7)",
                          "tracklets": {k: tls[k] for k in ("n_paired", "n_both_accepted", "n_identical_hits", "n_param_bad",
                                                            "max_err_in_sigma", "max_rel_per_param")},
                          "tracks": {k: stp[k] for k in ("n_gpu", "n_oracle", "n_paired_key", "n_paired_overlap",
                                                         "n_list_diff", "n_param_bad")}}
        # (2) sector-track refit + merging
        ms_refit = timed(lambda: B.tpc_refit_tracks(trk.ctx, stream.cuda_stream), lambda: B.tpc_get_refit(trk.ctx))
        extras["refit"] = {"ms": ms_refit, "tracks": int(gv.n_tracks), "clusters_refitted_per_s": int(gv.n_cluster_ids) / (ms_refit * 1e-3)}
        refit = extras["refit"]
        ms_merge = timed(lambda: trk.merge(stream=stream, fetch=False), lambda: B.tpc_get_merged(trk.ctx))
        rc_m, mv = B.tpc_get_merged(trk.ctx)
        extras["merge"] = {"ms": ms_merge, "links": int(mv.n_links), "merged_tracks": int(mv.n_merged),
                           "note": "includes one stream synchronisation per call (track count to the host)"}
        # (2b) the three-iteration track fit with interpolation rejection on the merged tracks (8(f) row 3)
        ms_fit = timed(lambda: trk.fit(stream=stream, fetch=False), lambda: B.tpc_get_fit(trk.ctx))
        fit3, _chi, rej3 = trk.fit(stream=stream)
        extras["fit3"] = {"ms": ms_fit, "merged_tracks": int(len(fit3)), "failed": int((fit3["flags"] != 0).sum()),
                          "clusters": int(len(rej3)), "clusters_rejected": int(rej3.sum())}
        del fit3, _chi, rej3
        trk.fit_ws = None
        # (2c) the Phase-II rebuild of the merged tracks (8(f) row 4, reading R11); the summary counts are
        # taken on the device (the per-step arrays of a C4 frame are several GB)
        try:
            ms_rb = timed(lambda: trk.rebuild(stream=stream, fetch=False), lambda: B.tpc_get_rebuild(trk.ctx))
            rc_r, rv = B.tpc_get_rebuild(trk.ctx)
            ns_, w_ = int(rv.n_steps), trk.rebuild_ws

            def dev(ptr, count, dt, size):
                off = ptr - w_.data_ptr()
                return w_[off:off + count * size].view(dt)
            att_ = dev(rv.d_attached, ns_, torch.int32, 4)
            fl_ = dev(rv.d_fit, int(rv.n_merged) * 25, torch.int32, 4).view(-1, 25)[:, 24]
            extras["rebuild"] = {"ms": ms_rb, "merged_tracks": int(rv.n_merged), "path_steps": ns_,
                                 "attached": int((att_ >= 0).sum()), "shared": int(dev(rv.d_shared, ns_, torch.uint8, 1).sum()),
                                 "used": int(dev(rv.d_used, ns_, torch.uint8, 1).sum()), "failed": int((fl_ != 0).sum()),
                                 "workspace_gb": w_.numel() / 1e9,
                                 "note": "includes one stream synchronisation per call (path length to the host)"}
            del att_, fl_, w_
        except Exception as e:
            extras["rebuild"] = {"error": str(e)[:200]}
        trk.rebuild_ws = None
        trk.merge_ws = None
        # (3) deterministic mode on the same frame
        if args.mode == "fast":
            det_flags = (flags | B.TPC_DETERMINISTIC) & ~B.TPC_STAGE_TIMERS
            ms_det = timed(lambda: trk.track(d_clusters, flags=det_flags, stream=stream), lambda: trk.counts())
            extras["det"] = {"ms_per_step": ms_det, "clusters_per_s": n / (ms_det * 1e-3)}
        # (4) the path + a second seeding iteration on the leftover clusters
        try:
            f2 = flags & ~B.TPC_STAGE_TIMERS
            ms_two = timed(lambda: trk.track_two_iterations(d_clusters, flags=f2, stream=stream), lambda: trk.counts())
            rc2, v2 = trk.counts()
            extras["second_iteration"] = {"ms_per_step": ms_two, "n_tracks": int(v2.n_tracks),
                                          "workspace_gb": B.tpc_workspace_bytes_two_iterations(trk.ctx, n) / 1e9}
        except Exception as e:      # (the two-iteration workspace is more than twice the plain one)
            extras["second_iteration"] = {"error": str(e)[:200]}

    idx = int(args.workload[1]) - 1
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{args.workload} (BASELINE.json configs[{idx}])", "n_clusters_per_gpu": n,
                   "n_events": cfg.n_events, "tracks_per_event": cfg.tracks_per_event, "mode": args.mode,
                   "tracker_params": pkw, "parallelism": f"independent time frames x{world}",
                   "l2": "inputs larger than L2 (frame %.2f GB + workspace %.1f GB)" % (n * 16 / 1e9, ws_bytes / 1e9),
                   "n_seeds": int(v.n_seeds), "n_tracklets": int(v.n_tracklets), "n_tracks": int(v.n_tracks),
                   "n_bins": int(v.n_bins), "follow_steps": st["follow_steps"],
                   "follow_updates": st["follow_updates"], "follow_cands": st["follow_cands"], "follow_work": st["follow_work"],
                   "generator_s": gen_s},
        "time_frames_per_s": world * args.steps / (ms_total * 1e-3),
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
        "roofline": roof, "stages_hbm": stages,
        "stage_ms": {k: round(x, 4) for k, x in stage_ms.items()},
        "kernels_ms_per_step": {k["name"]: round(k["ms_per_step"], 4) for k in per_kernel},
        "cpu_baseline": cpu, "cpu_baseline_all_cores": cpu_all, "refit": refit, "merge": extras.get("merge"), "fit3": extras.get("fit3"),
        "rebuild": extras.get("rebuild"),
        "det": extras.get("det"), "second_iteration": extras.get("second_iteration"), "parity": parity_obj,
    }
    print(json.dumps(line), flush=True)
    trk.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--workload", default="C4", choices=tuple(WORKLOAD_PARAMS))
    ap.add_argument("--mode", default="fast", choices=("fast", "det"))
    ap.add_argument("--events", type=int, default=None, help="override the preset's n_events (smaller frame)")
    ap.add_argument("--tracks", type=int, default=None, help="override tracks_per_event")
    ap.add_argument("--grid-dy", type=float, default=0.0)
    ap.add_argument("--grid-dz", type=float, default=0.0)
    ap.add_argument("--max-bins", type=int, default=0, help="bin-index capacity (0 = library default)")
    ap.add_argument("--oracle-budget", type=int, default=7_000_000,
                    help="clusters in the CPU oracle's bounded sample (~20 s single thread)")
    ap.add_argument("--e2e-chunks", type=int, default=0, help="equal chunks of whole sectors in the end-to-end leg (1 = one shot, 0 = ramped schedule)")
    ap.add_argument("--e2e-cuts", default="", help="sector boundaries of the chunks of the end-to-end leg (overrides --e2e-chunks)")
    ap.add_argument("--refit", action="store_true", help="(kept for compatibility: the refit, merging, deterministic-mode and second-iteration legs run by default)")
    ap.add_argument("--no-extras", action="store_true", help="skip the refit / merging / det / second-iteration legs and the parity sample")
    ap.add_argument("--second-iteration", action="store_true",
                    help="time tpc_sector_track_two_iterations (the path + a second seeding iteration) instead")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--split", default="frames", choices=("frames", "sectors"),
                    help="N > 1: independent frames per rank (default, weak scaling) or ONE frame split by sector + gather")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
