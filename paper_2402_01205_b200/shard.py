"""One time frame over several GPUs: the sector-sharded latency mode.

The paper's deployment gives whole time frames to the GPUs round-robin, "avoiding any GPU intercommunication"
 — that is `bench.py --gpus N` (replicas, throughput mode).  This module is the other mode: one frame is
cut into G contiguous ranges of (sector,row) planes balanced by digit count; planes are independent (R2), so
every rank runs the unchanged single-GPU path on its digit slice, and the concatenation of the per-rank outputs in rank
order IS the global (sector,row,pad,time) order.  The only exchange is the one the path really has: an all-gather of
8-byte counts and a variable-size gather of the 32-byte records into the root's buffer (point-to-point sends over
NCCL/NVLink, or gloo on CPU tensors in the tests).  No halo, no reduction.

Host logic and torch.distributed plumbing only: the clusters come from ClusterFinder (CUDA).
"""
import numpy as np


def plane_counts(digits, n_sectors, n_rows):
    """digits: sorted structured array (sector,row,...) on the host -> digit index where every plane starts
    (n_planes + 1 entries), by binary search on the (sector,row) key."""
    key = digits["sector"].astype(np.int64) * n_rows + digits["row"].astype(np.int64)
    return np.searchsorted(key, np.arange(n_sectors * n_rows + 1, dtype=np.int64), side="left")


def plane_partition(plane_start, world):
    """plane_start: n_planes + 1 digit indices (plane_counts).  Returns `world` tuples (plane_begin, plane_end,
    digit_begin, digit_end): contiguous, covering every plane once, cut where the running digit count crosses
    r / world of the total (so no rank holds more than total / world + one plane's digits)."""
    plane_start = np.asarray(plane_start, dtype=np.int64)
    n_planes = plane_start.shape[0] - 1
    total = int(plane_start[-1])
    cuts = [0]
    for r in range(1, world):
        target = (total * r) // world
        c = int(np.searchsorted(plane_start, target, side="left"))       # first plane starting at or after the target
        c = min(max(c, cuts[-1]), n_planes)
        cuts.append(c)
    cuts.append(n_planes)
    return [(cuts[r], cuts[r + 1], int(plane_start[cuts[r]]), int(plane_start[cuts[r + 1]])) for r in range(world)]


def gather_records(local, n_local, record_bytes=32, dst=0, group=None):
    """local: torch uint8 tensor holding n_local records of this rank (device or CPU, matching the backend).
    Returns (records, counts) on rank dst — records = the ranks' records concatenated in rank order — and
    (None, counts) elsewhere.  counts: python list of per-rank record counts (all ranks).
    A rank whose compute failed passes n_local < 0: the all-gather of the counts tells every rank, and ALL of them
    raise before any record moves (nobody is left waiting in a send or receive)."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    mine = torch.tensor([int(n_local)], dtype=torch.int64, device=local.device)
    allc = [torch.zeros(1, dtype=torch.int64, device=local.device) for _ in range(world)]
    dist.all_gather(allc, mine, group=group)
    counts = [int(c.item()) for c in allc]
    failed = [r for r, c in enumerate(counts) if c < 0]
    if failed:
        raise RuntimeError("sharded run failed on rank(s) %r (this is rank %d)" % (failed, rank))
    if rank != dst:
        if n_local:
            dist.send(local[:n_local * record_bytes].contiguous(), dst=dst, group=group)
        return None, counts
    out = torch.empty(sum(counts) * record_bytes, dtype=torch.uint8, device=local.device)
    off = 0
    reqs = []
    for r, c in enumerate(counts):
        seg = out[off * record_bytes:(off + c) * record_bytes]
        if r == dst:
            seg.copy_(local[:c * record_bytes])
        elif c:
            reqs.append(dist.irecv(seg, src=r, group=group))
        off += c
    for q in reqs:
        q.wait()
    return out, counts


class ShardedClusterFinder:
    """Latency mode: every rank holds the whole frame's digits on the host (or only its slice), runs the single-GPU
    cluster finder on the planes plane_partition gives it, and rank 0 receives the frame's clusters in global order."""

    def __init__(self, n_sectors, n_rows, max_pads, n_time, npads=None, max_digits=1 << 20, max_clusters=None,
                 device="cuda:0", group=None):
        from .binding import ClusterFinder
        self.geom = (n_sectors, n_rows, max_pads, n_time)
        self.group = group
        self.finder = ClusterFinder(n_sectors, n_rows, max_pads, n_time, npads=npads, max_digits=max_digits,
                                    max_clusters=max_clusters, device=device)

    def run(self, digits_host, flags=None):
        """digits_host: the frame's sorted digits (numpy, DIGIT).  Returns (clusters tensor on rank 0 or None, counts,
        this rank's partition entry)."""
        import torch
        import torch.distributed as dist
        from .binding import DIGITS_SORTED, STATUS, to_device
        world, rank = dist.get_world_size(self.group), dist.get_rank(self.group)
        part = plane_partition(plane_counts(digits_host, self.geom[0], self.geom[1]), world)[rank]
        mine = digits_host[part[2]:part[3]]
        n = int(mine.shape[0])
        n_cl, err = 0, None
        try:
            if n:
                d = to_device(mine, device=self.finder.device)
                # the launch shape comes from the WHOLE frame's line length, not from this rank's slice
                self.finder.set_frame_digits(int(digits_host.shape[0]))
                self.finder.run(d, n, flags=DIGITS_SORTED if flags is None else flags)
                raw = self.finder.status.cpu().numpy().view(STATUS)[0]      # synchronises this rank's stream
                st = {k: int(raw[k]) for k in STATUS.names}
                if st["path"] == 0 or st["overflow"]:
                    raise RuntimeError("shard %d: cluster finder status %r" % (rank, st))
                n_cl = st["n_clusters"]
        except Exception as e:                                   # tell the peers (count -1) before raising
            n_cl, err = -1, e
        try:
            out, counts = gather_records(self.finder.clusters, n_cl, 32, 0, self.group)
        except RuntimeError:
            if err is not None:
                raise err
            raise
        return out, counts, part

    def close(self):
        self.finder.close()
