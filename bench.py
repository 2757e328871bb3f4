#!/usr/bin/env python
"""bench.py -- BASELINE.json metric: integrand events/s (fp64) for gg -> t t~ g at 1e7 events per
VEGAS iteration (configs[2], the configuration the metric is quoted on), one line of JSON.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one pass of the whole hot path (S1-S10: Philox -> VEGAS map -> x map -> RAMBO+Newton ->
cuts -> PDF -> |M|^2 -> weight -> reductions -> refine) over one batch of 1e7 events per GPU, i.e.
one mf_vegas_iterate; successive steps are successive iterations of one VEGAS run (the grid adapts,
as in config 2).  N > 1: every rank takes its own event range of an N*1e7-event iteration (weak
scaling) and the ranks exchange the 2+d*50 raw sums once per iteration (NCCL all-reduce).
`--impl reference` times the oracle (oracle/, plain CPU code, as it stands) on the host cores.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "integrand events/sec (fp64) gg->ttbar g, 1e7 events/iteration/GPU"
N_EVENTS = 10_000_000
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # SMs x DFMA lanes x 2 x max clock
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r2_ncu_traffic.json")   # dram bytes per passing event from the committed ncu capture


def ncu_traffic(kernel, n_pass):
    """roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel`, from the committed ncu
    --set full capture (profiles/r2_ncu_traffic.json: bytes per cut-passing event of that capture), scaled to the passing
    events of one launch of THIS run; (None, why) when no capture of that kernel is on file"""
    try:
        with open(TRAFFIC_FILE) as f:
            rec = json.load(f)[kernel]
    except (OSError, KeyError, ValueError):
        return None, "no ncu capture of %s in profiles/r2_ncu_traffic.json" % kernel
    return rec["dram_bytes_per_passing_event"] * n_pass, rec["source"]


def launch_ranks_if_needed(args, argv):
    """`python bench.py --gpus N` without torchrun: start N ranks (one per GPU) of this very command"""
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        port = str(29500 + os.getpid() % 400)
        os.execvp(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
                                   "--master-addr", "127.0.0.1", "--master-port", port, os.path.abspath(__file__)] + argv)


def init_ranks(backend="nccl", force_group=False):
    """(rank, local_rank, world, dist or None) from the torchrun environment; the process group exists iff world > 1 or
    force_group (the N > 1 code path at N = 1).  backend "gloo" runs the same logic on CPU (tests/test_sharding.py)."""
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world == 1 and not force_group:
        return rank, local_rank, world, None
    import torch
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29533")
    kw = {}
    if backend == "nccl":
        os.environ.setdefault("NCCL_DEBUG", "INFO")              # the communicator log (ranks, transport) goes to stderr:
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")       # stdout carries the one JSON line
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
        kw["device_id"] = torch.device("cuda", local_rank)
    dist.init_process_group(backend, rank=rank, world_size=world, **kw)
    return rank, local_rank, world, dist


def max_over_ranks(dist, value, device=None):
    """device time of the slowest rank (the contract's timing rule)"""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled every 50 ms while the warm-up, timed and e2e regions run"""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, uuid):
        self.rows, self.p = [], None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", uuid, "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                       "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.p = None

    def _read(self):
        for line in self.p.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        self.t.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        pw = [float(r[2]) for r in self.rows if len(r) >= 7 and r[2].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 7 and r[3 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def oracle_rate(n_threads, seconds):
    """the oracle as it stands (whole path, O1-O10) on a bounded sample of the workload"""
    from oracle import mfo
    from paper_2105_10529_b200 import workloads as W
    cfg = W.config(W.GG_TTG, seed=0)
    orc = mfo.Vegas(cfg)
    probe = 2000 * n_threads
    t0 = time.perf_counter(); orc.accumulate(0, 0, probe, N_EVENTS, n_threads=n_threads); dt = time.perf_counter() - t0
    n = max(probe, int(probe / dt * seconds))
    t0 = time.perf_counter(); orc.iterate(n, n_threads=n_threads); dt = time.perf_counter() - t0
    return n / dt, n, dt


def run_reference(args, rank):
    """--impl reference: the oracle on the host cores, rank 0 only"""
    if rank != 0:
        return
    from oracle import mfo
    from paper_2105_10529_b200 import workloads as W
    mfo.build()
    nt = mfo.max_threads()
    orc = mfo.Vegas(W.config(W.GG_TTG, seed=0))
    probe = 500 * nt
    t0 = time.perf_counter(); orc.accumulate(0, 0, probe, N_EVENTS, n_threads=nt); dt = time.perf_counter() - t0
    budget = 150.0 / max(1, args.steps + args.warmup)             # whole run within a few minutes
    n = max(2 * nt, int(probe / dt * min(budget, 20.0)))
    for _ in range(args.warmup):
        orc.iterate(n, n_threads=nt)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.iterate(n, n_threads=nt)
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    sample = "%d events per step (of the 1e7-event iteration), gg->ttg whole path, %d host threads" % (n, nt)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[2]: pp->tt~g via gg->tt~g, 7 dims x 50 bins, cuts pT>30 |eta|<2.5, seed 0 "
                               "(bounded sample per step)", "events_per_step": n},
        "cpu_baseline": {"value": value, "unit": "events/s", "cores": nt, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_ours(args, rank, local_rank, world, dist):
    import torch
    from paper_2105_10529_b200 import binding, sharding, workloads as W
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU path); use --impl reference for the oracle")
    binding.lib()
    sharded = dist is not None                                             # the N > 1 code path (also at N = 1 with --sharded)
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    n, n_total = args.events, args.events * world
    cfg = W.config(W.GG_TTG, seed=0, device=local_rank)
    h = binding.Vegas(cfg)
    staged = args.path == "staged"
    h.set_path(staged)
    flops = h.me_flops()
    bounds = h.me_flops_bounds()
    uuid = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid)
    peak_before = binding.fp64_peak(local_rank, 0.3)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)          # > 126 MB L2

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step(sync=False):
        flush.zero_()                                                      # L2 flush between iterations (both timed loops)
        if not sharded:
            return h.vegas_iterate(n, sync=sync)
        return sharding.sharded_iterate_device(h, n_total, rank, world, dist, dev, sync=sync)

    # clocks are sampled from the first warm-up step to the end of the end-to-end region (same load)
    sampler = ClockSampler(uuid) if rank == 0 else None
    for _ in range(args.warmup):
        step()
    barrier()
    if staged:
        h.stage_ms_sum()                                                   # forget the warm-up launches
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    fused_ms = []
    e0.record()
    for _ in range(args.steps):                                            # nothing synchronises inside the timed region
        step()
        if not staged:
            fused_ms.append(h.last_kernel_ms()[0])                         # (fused path: one event pair per handle -> waits per step)
    e1.record()
    barrier()
    ms = max_over_ranks(dist, e0.elapsed_time(e1), dev)
    if staged:                                                             # CUDA events the library recorded on the launching stream
        sums, launches = h.stage_ms_sum()                                  # around every stage of every timed launch
        stages = {k: v / launches for k, v in sums.items()}
        k_ms = stages["me"]
    else:
        stages, launches, k_ms = None, len(fused_ms), float(np.mean(fused_ms))
    its = h.get_iterations()
    pass_frac = float(np.mean([it["n_pass"] / it["n_events"] for it in its[-args.steps:]]))
    value = n_total * args.steps / (ms * 1e-3)

    # end to end through the C-ABI with host buffers: grid in from the host, record + grid back out, same L2 flush
    grid = h.get_grid()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        h.set_grid(grid)                                                   # H2D d*51 doubles
        rec = step(sync=True)                                              # D2H iteration record (40 B)
        grid = h.get_grid()                                                # D2H refined grid
    barrier()
    e2e_s = max_over_ranks(dist, time.perf_counter() - t0, dev)
    clocks = sampler.stop() if sampler else None
    peak_after = binding.fp64_peak(local_rank, 0.3)
    res = h.result()
    if rank != 0:
        return None
    n_pass = pass_frac * n                                                 # per launch (this rank's events)
    step_ms = ms / args.steps
    peak = max(peak_before, peak_after) / 1e12
    tf = lambda fl, t_ms: fl * n_pass / (t_ms * 1e-3) / 1e12               # TFLOP/s of `fl` flops per passing event over t_ms
    achieved = tf(flops["flops"], k_ms)
    kernel = "mf_me_kernel<2, double, 256>" if staged else "mf_iterate_compact_kernel<2>"
    traffic, traffic_src = ncu_traffic(kernel, n_pass) if staged else (None, "fused path: no per-event traffic")
    grid_bytes = int(grid.nbytes)
    out = {
        "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[2]: pp->tt~g via gg->tt~g (16 diagrams, 6x6 colour matrix), massive 3-body RAMBO + "
                               "Newton, cuts pT>30 |eta|<2.5, VEGAS 7 dims x 50 bins, seed 0, successive iterations of one run",
                   "events_per_step_per_gpu": n, "pass_fraction": pass_frac, "path": args.path,
                   "l2": "flushed before every step of both timed loops (256 MiB memset inside the timed region); inputs are 46 KB "
                         "of tables; the staged path passes ~1.0 GB of event records per step through HBM (> 126 MB L2)",
                   "parallelism": "event ranges over %d GPU(s), 1 NCCL all-reduce of 354 doubles on the device per iteration "
                                  "(no host round trip)" % world if sharded else "1 GPU",
                   "integral_pb": res["integral"], "sigma_pb": res["sigma"]},
        "clocks": clocks,
        "e2e": {"value": n_total * args.steps / e2e_s, "unit": "events/s", "h2d_bytes_per_step": grid_bytes,
                "d2h_bytes_per_step": grid_bytes + 40},
        "gpu_launches": ((5 if staged else 3) + (2 if sharded else 0)) * args.steps,   # + pack/unpack of the raw sums around the all-reduce
        "roofline": {
            "bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
            "traffic": traffic, "traffic_source": traffic_src,
            "algorithmic_bytes": 120.0 * n_pass if staged else 0.0,
            "kernel": kernel, "kernel_ms": k_ms, "kernel_launches_timed": launches, "kernel_share_of_step": k_ms / step_ms,
            "flops_per_event": flops["flops"], "fma_fraction_of_ops": flops["fma"] / (flops["add"] + flops["mul"] + flops["fma"]),
            "peak_source": "measured DFMA-chain microbenchmark (mf_fp64_peak), max of before/after the timed region; "
                           "MEASURED_PEAKS.json and the profiling guide have no fp64 entry",
            "peak_before": peak_before / 1e12, "peak_after": peak_after / 1e12, "peak_nominal": FP64_NOMINAL_TFLOPS,
            # the same algorithmic flops over the WHOLE step (front end, reductions, memsets, launch gaps included):
            # what north_star's "sustained in the integrand" asks; and both against the chip's nominal peak
            "frac_step": tf(flops["flops"], step_ms) / peak,
            "frac_nominal": achieved / FP64_NOMINAL_TFLOPS,
            "frac_step_nominal": tf(flops["flops"], step_ms) / FP64_NOMINAL_TFLOPS,
            # the leanest op list the generator knows for this amplitude (every helicity unrolled, everything shared)
            "flops_per_event_min": bounds["min"], "frac_min": tf(bounds["min"], k_ms) / peak,
            "frac_step_min": tf(bounds["min"], step_ms) / peak,
            "flops_per_event_executed": bounds["executed"],
            "note": "algorithmic flops = generator-counted |M|^2 add+mul+2*fma per passing event of the emitted organisation "
                    "(helicity loop: loop invariants counted once); front end, wavefunction ingredients and padding not counted"},
    }
    if staged:
        out["roofline"]["stages_ms"] = stages
        out["roofline"]["front_stage_hbm_gbps"] = 15 * 8 * n_pass / (stages["front"] * 1e-3) / 1e9   # 4*3+3 doubles per passing event
        out["roofline"]["reduce_stage_hbm_gbps"] = 16 * n_pass / (stages["reduce"] * 1e-3) / 1e9
    if world == 1 and not args.no_cpu_baseline:
        from oracle import mfo
        mfo.build()
        nt = mfo.max_threads()
        v, ns, dt = oracle_rate(nt, 12.0)
        v1, ns1, dt1 = oracle_rate(1, 6.0)
        out["cpu_baseline"] = {"value": v, "unit": "events/s", "cores": nt, "kind": "oracle",
                               "sample": "first %d events of the 1e7-event iteration, whole path, %.1f s" % (ns, dt),
                               "single_thread": {"value": v1, "unit": "events/s", "cores": 1,
                                                 "sample": "first %d events, whole path, %.1f s" % (ns1, dt1)}}
    return json.dumps(out)


def run_sweep(args):
    """BASELINE.json configs[4]: throughput sweep of the gg -> tt~g integrand of config 2 over events per
    launch (1e4 .. 1e8, 1e8 in slices of 2^24 events), uniform grid, single iteration, seed 1, in fp64 and
    with the fp32 variant of the |M|^2 stage.  One JSON line with one entry per size and precision."""
    import torch
    from paper_2105_10529_b200 import binding, workloads as W
    binding.lib()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    peak = binding.fp64_peak(0, 0.3) / 1e12
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    rows = []
    for n, prec in [(m, 64) for m in (10_000, 100_000, 1_000_000, 10_000_000, 100_000_000)] + \
                   ([(m, 32) for m in (10_000, 100_000, 1_000_000, 10_000_000, 100_000_000)] if args.path == "staged" else []):
        reps = 5 if n <= 10_000_000 else 2
        h = binding.Vegas(W.config(W.GG_TTG, seed=1, precision=prec))
        h.set_path(args.path == "staged")
        uniform = h.get_grid()
        h.vegas_accumulate(0, min(n, 1 << 24), n)                          # warm-up: allocates the staged workspace
        flops = h.me_flops()["flops"]
        best = None
        for _ in range(reps):
            h.set_grid(uniform)                                            # every repetition on the uniform grid
            flush.zero_()
            torch.cuda.synchronize()
            if args.path == "staged":
                h.stage_ms_sum()
            r = h.vegas_iterate(n, sync=True)
            k_ms, it_ms = h.last_kernel_ms()
            st, slices = h.stage_ms_sum() if args.path == "staged" else (None, 0)     # summed over the slices of <= 2^24 events
            if best is None or it_ms < best["iteration_ms"]:
                best = {"events": n, "me_precision": prec, "iteration_ms": it_ms, "events_per_s": n / (it_ms * 1e-3), "n_pass": r["n_pass"],
                        "integral_pb": r["integral"], "sigma_pb": r["sigma"], "stages_ms": st, "launches": slices,
                        "whole_path_tflops": flops * r["n_pass"] / (it_ms * 1e-3) / 1e12}
                if st:
                    best["me_tflops"] = flops * r["n_pass"] / (st["me"] * 1e-3) / 1e12
                    best["me_frac_of_peak"] = best["me_tflops"] / peak
                    best["reduce_stage_gbps"] = 16.0 * r["n_pass"] / (st["reduce"] * 1e-3) / 1e9
                    best["front_stage_gbps"] = 120.0 * r["n_pass"] / (st["front"] * 1e-3) / 1e9
        rows.append(best)
    print(json.dumps({"metric": "throughput sweep, gg->ttbar g integrand (configs[4])", "unit": "events/s", "dtype": "f64",
                      "path": args.path, "fp64_peak_tflops": peak, "fp32_variant": "me_precision 32 = |M|^2 stage in fp32, front end and reductions in fp64 (DESIGN.md A24); "
                                      "its TFLOP/s are fp32 operations against the same fp64 peak, for reference only", "sweep": rows}))


def run_processes(args):
    """Every process and generator selection at its config size (configs 0-3; the quark channel and the selectable
    generators of SURVEY 8(f)2/3 at the size of the process they vary): device time of whole iterations on the adapting
    grid (warm-up iterations first), L2 flushed before every timed iteration.  One JSON line."""
    import torch
    from paper_2105_10529_b200 import binding, workloads as W
    binding.lib()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    peak = binding.fp64_peak(0, 0.3) / 1e12
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    sizes = {W.EE_MUMU: 100_000, W.GG_TT: 1_000_000, W.GG_TTG: 10_000_000, W.GG_TTGG: 1_000_000, W.QQ_TT: 1_000_000, W.PP_TT: 1_000_000,
             W.QQ_TTG: 1_000_000, W.QG_TTQ: 1_000_000}
    cases = [(W.EE_MUMU, 0), (W.GG_TT, 0), (W.GG_TT, 1), (W.GG_TT, 2), (W.QQ_TT, 0), (W.QQ_TT, 1), (W.PP_TT, 0), (W.QQ_TTG, 0), (W.QG_TTQ, 0),
             (W.GG_TTG, 0), (W.GG_TTG, 1), (W.GG_TTG, 2), (W.GG_TTG, 3), (W.GG_TTGG, 0), (W.GG_TTGG, 1)]
    if args.only:
        cases = [c for c in cases if W.PROCESS_NAMES[c[0]] in args.only.split(",")]
    rows = []
    for proc, gen in cases:
        n = sizes[proc]
        h = binding.Vegas(W.config(proc, seed=0, generator=gen))
        for _ in range(3):
            h.vegas_iterate(n, sync=True)
        flops = h.me_flops()["flops"]
        ms, last = [], None
        for _ in range(5):
            flush.zero_()
            torch.cuda.synchronize()
            last = h.vegas_iterate(n, sync=True)
            ms.append(h.last_kernel_ms()[1])
        it_ms = sorted(ms)[len(ms) // 2]
        row = {"process": W.PROCESS_NAMES[proc], "generator": gen, "d": h.d, "events": n, "iteration_ms": it_ms,
               "events_per_s": n / (it_ms * 1e-3), "pass_fraction": last["n_pass"] / n,
               "me_flops_per_event": flops, "whole_path_tflops": flops * last["n_pass"] / (it_ms * 1e-3) / 1e12}
        row["whole_path_frac_of_fp64_peak"] = row["whole_path_tflops"] / peak
        try:
            st = h.last_stage_ms()
            row["stages_ms"] = st
        except binding.MfError:
            row["stages_ms"] = None                                         # fused path
        r = h.result()
        row["integral_pb"], row["sigma_pb"] = r["integral"], r["sigma"]
        rows.append(row)
    print(json.dumps({"metric": "events/s of whole VEGAS iterations, every process and generator selection", "unit": "events/s",
                      "dtype": "f64", "fp64_peak_tflops": peak, "timing": "median of 5 iterations after 3 warm-up iterations, "
                      "CUDA events around mf_vegas_iterate, 256 MiB L2 flush before each", "rows": rows}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--events", type=int, default=N_EVENTS, help="events per iteration per GPU")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="configs[4]: events-per-launch sweep of the gg->tt~g integrand (1 GPU)")
    ap.add_argument("--sharded", action="store_true", help="run the multi-GPU code path (device-side all-reduce of the raw sums) even at N = 1")
    ap.add_argument("--processes", action="store_true", help="every process / generator selection at its config size (1 GPU)")
    ap.add_argument("--only", default="", help="with --processes: comma-separated process names (ee_mumu, gg_tt, qq_tt, pp_tt, qq_ttg, qg_ttq, gg_ttg, gg_ttgg)")
    ap.add_argument("--path", default="staged", choices=["staged", "fused"],
                    help="staged: front end / |M|^2 / reductions as three kernels (default); fused: one kernel")
    args = ap.parse_args()
    if args.impl == "ours" and not (args.sweep or args.processes):
        launch_ranks_if_needed(args, sys.argv[1:])         # --gpus N without torchrun: N ranks of this command
    if args.impl == "reference":
        run_reference(args, int(os.environ.get("RANK", "0")))
        return
    if args.sweep or args.processes:
        if int(os.environ.get("RANK", "0")) == 0:
            (run_sweep if args.sweep else run_processes)(args)
        return
    # stdout carries the one JSON line: anything a library prints there (NCCL's version banner and communicator log at
    # NCCL_DEBUG=INFO) is sent to stderr, the line itself goes to the saved descriptor
    sys.stdout.flush()
    out_fd = os.dup(1)
    os.dup2(2, 1)
    rank, local_rank, world, dist = init_ranks("nccl", force_group=args.sharded)
    try:
        line = run_ours(args, rank, local_rank, world, dist)
    finally:
        if dist is not None:
            dist.destroy_process_group()
    sys.stdout.flush()
    if line:
        os.write(out_fd, (line + "\n").encode())


if __name__ == "__main__":
    main()
