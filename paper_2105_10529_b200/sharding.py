"""Event-range sharding of one VEGAS iteration over ranks.

Events are independent and the RNG is keyed by the global event index, so rank r of R evaluates
indices [r N / R, (r+1) N / R) with no data-path collective; the only exchange is one all-reduce of
the 2 + d*n_bins raw sums and the two counters per iteration (2.8 KB for gg -> tt~g), after which
every rank runs the same deterministic refinement and so holds the same grid.
"""
import numpy as np


def shard_range(n_total, rank, world):
    first = n_total * rank // world
    return first, n_total * (rank + 1) // world - first


def allreduce_sums(acc, counts, dist=None, device=None):
    """sum (acc, counts) over the ranks of torch.distributed; identity without a process group"""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return acc, counts
    import torch
    buf = torch.from_numpy(np.concatenate([acc, counts.astype(np.float64)]))   # counts < 2^53: exact
    if device is not None:
        buf = buf.to(device)
    dist.all_reduce(buf, op=dist.ReduceOp.SUM)
    out = buf.cpu().numpy()
    return out[:len(acc)].copy(), np.rint(out[len(acc):]).astype(np.uint64)


def sharded_iterate_device(h, n_total, rank, world, dist=None, device=None, sync=True):
    """the same iteration without host round trips: the raw sums and counters stay on the device, the all-reduce runs
    on a device buffer (NCCL), everything is enqueued on torch's current stream; sync=False returns without waiting"""
    import torch
    first, n = shard_range(n_total, rank, world)
    h.zero_accum()
    h.vegas_accumulate(first, n, n_total)
    m = h.accum_len() + 2
    buf = getattr(h, "_exchange_buf", None)                  # one exchange buffer per handle, reused every iteration
    if buf is None or buf.numel() != m or buf.device != torch.device(device if device is not None else "cuda"):
        buf = h._exchange_buf = torch.empty(m, dtype=torch.float64, device=device)
    h.get_accum_device(buf.data_ptr())
    if dist is not None and dist.is_initialized():
        dist.all_reduce(buf, op=dist.ReduceOp.SUM)         # ordered after the pack kernel on the current stream
    h.set_accum_device(buf.data_ptr())
    return h.vegas_finalize(n_total, sync=sync)


def sharded_iterate(h, n_total, rank, world, dist=None, device=None, stream=None):
    """one iteration of n_total events split over `world` ranks; h has the C-ABI's method names
    (set_accum / vegas_accumulate / get_accum / vegas_finalize).  Host-staged exchange (works with any backend:
    the gloo test); device handles on NCCL use sharded_iterate_device"""
    first, n = shard_range(n_total, rank, world)
    zeros = np.zeros(h.accum_len() if hasattr(h, "accum_len") else 2 + h.d * h.n_bins)
    h.set_accum(zeros, np.zeros(2, np.uint64))
    h.vegas_accumulate(first, n, n_total, stream=stream)
    acc, counts = h.get_accum()
    acc, counts = allreduce_sums(acc, counts, dist, device)
    h.set_accum(acc, counts)
    return h.vegas_finalize(n_total, stream=stream)
