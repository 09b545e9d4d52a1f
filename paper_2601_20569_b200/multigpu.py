"""One time frame over several GPUs by SECTOR (first axis).

Sectors are the independent units of the sector tracking (a sector never reads
another sector's clusters; cross-sector work starts at merging), so a frame shards
with no collective inside the path: rank r tracks the sectors s with s mod N == r, and one
variable-length gather brings tracks + cluster lists to the merging rank.  Plumbing only (index
bookkeeping and torch.distributed calls; it runs on gloo / CPU tensors as well as on NCCL / CUDA
tensors): the tracking itself is the CUDA path behind the C ABI.
"""
from __future__ import annotations

import numpy as np


def sector_ranges(clusters: np.ndarray, n_sectors: int = 36):
    """(start, end) record range of every sector of a frame grouped by sector (clusteriser
    order); raises if a sector's records are not contiguous."""
    sec = clusters["sector"].astype(np.int64)
    if len(sec) and np.any(np.diff(sec) < 0):
        raise ValueError("split by sector needs the frame grouped by sector")
    starts = np.searchsorted(sec, np.arange(n_sectors), side="left")
    ends = np.searchsorted(sec, np.arange(n_sectors), side="right")
    return starts, ends


def split_by_sector(clusters: np.ndarray, rank: int, world: int, n_sectors: int = 36):
    """The sub-frame of rank `rank` (its sectors' records, concatenated in sector order) and, per
    sector, the offset that turns an index into the sub-frame into an index into the frame."""
    starts, ends = sector_ranges(clusters, n_sectors)
    mine = [s for s in range(n_sectors) if s % world == rank]
    parts, delta = [], np.zeros(n_sectors, dtype=np.int64)
    pos = 0
    for s in mine:
        parts.append(clusters[starts[s]:ends[s]])
        delta[s] = int(starts[s]) - pos
        pos += int(ends[s] - starts[s])
    sub = np.concatenate(parts) if parts else clusters[:0]
    return sub, delta


def rebase(tracks: np.ndarray, cluster_ids: np.ndarray, delta: np.ndarray):
    """Express a rank's result in indices of the whole frame: cluster ids and seed ids shift by
    their sector's offset (a sector track holds clusters of one sector only)."""
    tracks = tracks.copy()
    d = delta[tracks["sector"].astype(np.int64)]
    n_per = tracks["n_clusters"].astype(np.int64)
    ids = cluster_ids.astype(np.int64)
    ofs = tracks["cluster_ofs"].astype(np.int64)
    within = np.arange(int(n_per.sum()), dtype=np.int64) - np.repeat(np.cumsum(n_per) - n_per, n_per)
    g = np.repeat(ofs, n_per) + within
    ids[g] += np.repeat(d, n_per)
    tracks["seed_id"] = (tracks["seed_id"].astype(np.int64) + d).astype(tracks["seed_id"].dtype)
    return tracks, ids.astype(np.uint32)


def gather_to_root(tracks: np.ndarray, cluster_ids: np.ndarray, cluster_shared: np.ndarray, rank: int, world: int,
                   device=None):
    """Variable-length gather of every rank's (tracks, cluster ids, shared flags) to rank 0: an
    all-gather of the counts, then one send/recv per array and rank.  Rank 0 returns the concatenated
    result (tracks' cluster_ofs shifted to the concatenated id list), other ranks return None."""
    import torch
    import torch.distributed as dist
    if world == 1:
        return tracks, cluster_ids, cluster_shared
    dev = device if device is not None else torch.device("cpu")
    counts = torch.tensor([len(tracks), len(cluster_ids)], dtype=torch.int64, device=dev)
    all_counts = [torch.zeros(2, dtype=torch.int64, device=dev) for _ in range(world)]
    dist.all_gather(all_counts, counts)
    all_counts = [tuple(int(x) for x in c.cpu()) for c in all_counts]
    isz = tracks.dtype.itemsize

    def as_tensor(a):
        return torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1).copy()).to(dev)
    if rank != 0:
        for a in (tracks, cluster_ids, cluster_shared):
            if a.size:
                dist.send(as_tensor(a), dst=0)
        return None
    t_parts, i_parts, s_parts = [tracks.copy()], [cluster_ids], [cluster_shared]
    id_base = len(cluster_ids)
    for r in range(1, world):
        nt, ni = all_counts[r]
        bufs = []
        for nbytes in (nt * isz, ni * 4, ni):
            b = torch.empty(nbytes, dtype=torch.uint8, device=dev)
            if nbytes:
                dist.recv(b, src=r)
            bufs.append(b.cpu().numpy())
        tr = bufs[0].view(tracks.dtype).copy()
        tr["cluster_ofs"] = (tr["cluster_ofs"].astype(np.int64) + id_base).astype(tr["cluster_ofs"].dtype)
        t_parts.append(tr)
        i_parts.append(bufs[1].view(np.uint32))
        s_parts.append(bufs[2].view(np.uint8))
        id_base += ni
    return np.concatenate(t_parts), np.concatenate(i_parts), np.concatenate(s_parts)
