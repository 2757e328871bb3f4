"""World-size-2 gloo tests (CPU) of the sharded-iteration plumbing (paper_2105_10529_b200/sharding.py), in its host-staged
form and in the device-buffer form that bench.py --gpus N runs (here with a CPU tensor as the exchange buffer):
event ranges, the one all-reduce of the raw sums, identical grids on every rank.  The device handle is
replaced by an adapter over the oracle (same method names as the C-ABI binding)."""
import ctypes
import os
import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2105_10529_b200 import sharding, workloads as W


class OracleHandle:
    """binding.Vegas look-alike on host memory (tests only)"""

    def __init__(self, cfg):
        from oracle import mfo
        self.v = mfo.Vegas(cfg)
        self.d, self.n_bins = self.v.d, self.v.n_bins
        self.iteration = 0
        self.acc = np.zeros(2 + self.d * self.n_bins); self.cnt = np.zeros(2, np.uint64)

    def set_accum(self, acc, counts):
        self.acc = np.array(acc, dtype=np.float64); self.cnt = np.array(counts, dtype=np.uint64)

    def get_accum(self):
        return self.acc.copy(), self.cnt.copy()

    def vegas_accumulate(self, first, n, n_total, stream=None):
        acc, cnt = self.v.accumulate(self.iteration, first, n, n_total, n_threads=2, acc=self.acc.copy())
        self.acc = acc; self.cnt = self.cnt + cnt

    def vegas_finalize(self, n_total, stream=None, sync=True):
        self.iteration += 1
        return self.v.finalize(self.acc, n_total, self.cnt[0], self.cnt[1])

    # the device-side exchange of the C-ABI (mf_zero_accum / mf_get_accum_device / mf_set_accum_device) on host memory:
    # the "device buffer" is a CPU tensor, addressed by its data_ptr() like the real one
    def accum_len(self):
        return len(self.acc)

    def zero_accum(self, stream=None):
        self.acc[:] = 0.0; self.cnt[:] = 0

    def get_accum_device(self, ptr, stream=None):
        buf = np.concatenate([self.acc, self.cnt.astype(np.float64)])
        ctypes.memmove(ptr, buf.ctypes.data, buf.nbytes)

    def set_accum_device(self, ptr, stream=None):
        buf = np.zeros(len(self.acc) + 2)
        ctypes.memmove(buf.ctypes.data, ptr, buf.nbytes)
        self.acc = buf[:-2].copy(); self.cnt = np.rint(buf[-2:]).astype(np.uint64)


def test_shard_ranges_cover_the_iteration():
    for n, world in ((10, 3), (10_000_000, 8), (7, 8), (1, 2)):
        spans = [sharding.shard_range(n, r, world) for r in range(world)]
        assert spans[0][0] == 0 and sum(c for _, c in spans) == n
        for (f0, c0), (f1, _) in zip(spans, spans[1:]):
            assert f0 + c0 == f1


def _worker(rank, world, port, q, device_form=False):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    h = OracleHandle(W.config(W.GG_TT, seed=3))
    out = []
    for _ in range(2):
        if device_form:      # the function bench.py --gpus N runs, with a CPU tensor as the exchange buffer
            it = sharding.sharded_iterate_device(h, 6001, rank, world, dist, torch.device("cpu"))
        else:
            it = sharding.sharded_iterate(h, 6001, rank, world, dist)
        out.append((it["integral"], it["sigma"], it["n_pass"]))
    q.put((rank, out, h.v.get_grid()))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("device_form", [False, True])
def test_two_rank_iteration_matches_single_process(mfo, device_form):
    port = 29500 + (os.getpid() + 7 * device_form) % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q, device_form)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted([q.get(timeout=300) for _ in procs], key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    single = mfo.Vegas(W.config(W.GG_TT, seed=3))
    ref = [single.iterate(6001, n_threads=2) for _ in range(2)]
    for rank, out, grid in got:
        for (I, s, npass), r in zip(out, ref):
            assert abs(I / r["integral"] - 1) < 1e-12 and abs(s / r["sigma"] - 1) < 1e-9 and npass == r["n_pass"]
        np.testing.assert_allclose(grid, single.get_grid(), rtol=0, atol=1e-13)
    np.testing.assert_array_equal(got[0][2], got[1][2])      # every rank holds the same grid, bit for bit


# ---- bench.py's rank logic (the part in front of the first CUDA call) with world size 2 under gloo ------------------
def _bench_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    r, lr, w, d = bench.init_ranks("gloo")
    slow = bench.max_over_ranks(d, 10.0 + r)                     # the timing rule: max over ranks
    h = OracleHandle(W.config(W.GG_TT, seed=3))
    it = sharding.sharded_iterate_device(h, 4001, r, w, d, torch.device("cpu"))   # bench.py's step() at N > 1
    buf_id = id(h._exchange_buf)
    sharding.sharded_iterate_device(h, 4001, r, w, d, torch.device("cpu"))
    q.put((r, lr, w, d is not None, slow, it["integral"], buf_id == id(h._exchange_buf)))
    d.barrier()
    d.destroy_process_group()


def test_bench_rank_logic_world_size_2(mfo, monkeypatch):
    import bench
    port = 31500 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_bench_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted([q.get(timeout=300) for _ in procs])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    ref = mfo.Vegas(W.config(W.GG_TT, seed=3)).iterate(4001, n_threads=2)
    for r, (rank, local_rank, world, grouped, slow, integral, reused) in enumerate(got):
        assert (rank, local_rank, world, grouped) == (r, r, 2, True) and slow == 11.0 and reused   # one exchange buffer per handle
        assert abs(integral / ref["integral"] - 1) < 1e-12
    # without torchrun, `bench.py --gpus 2` starts the two ranks itself; inside torchrun (WORLD_SIZE set) it does not
    calls = []
    monkeypatch.setattr(os, "execvp", lambda exe, argv: calls.append(argv))
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    args = type("A", (), {"gpus": 2})()
    bench.launch_ranks_if_needed(args, ["--gpus", "2", "--steps", "3"])
    assert len(calls) == 1 and calls[0][1:4] == ["-m", "torch.distributed.run", "--nnodes=1"]
    assert calls[0][calls[0].index("--nproc-per-node") + 1] == "2" and calls[0][-4:] == ["--gpus", "2", "--steps", "3"]
    assert "127.0.0.1" in calls[0] and os.path.basename(calls[0][calls[0].index("--master-port") + 2]) == "bench.py"
    monkeypatch.setenv("WORLD_SIZE", "2")
    bench.launch_ranks_if_needed(args, ["--gpus", "2"])
    assert len(calls) == 1
    monkeypatch.delenv("WORLD_SIZE")
    assert bench.init_ranks("gloo") == (0, 0, 1, None)           # plain N = 1: no process group
