"""Text summary of an ncu report (`ncu --set full ... -o report`) for profiles/: per captured launch the counters the
design arguments rest on (duration, DRAM bytes, local- and shared-memory traffic, FP64 pipe, issue activity, stall
reasons per issue).  Optionally records the DRAM bytes per cut-passing event of one kernel in a JSON file that
bench.py reads for `roofline.traffic`.

    python -m paper_2105_10529_b200.profile_summary report.ncu-rep [--traffic-json profiles/r2_ncu_traffic.json
        --kernel "mf_me_kernel<2, double, 256>" --passing 8480000 --source profiles/r2_ttg_ncu.md]

Needs the `ncu` command line tool (reads the report; no GPU)."""
import argparse
import csv
import json
import os
import subprocess

WANT = ["dram__bytes_read.sum", "dram__bytes_write.sum", "gpu__time_duration.sum", "launch__registers_per_thread", "launch__grid_size",
        "launch__block_size", "launch__occupancy_limit_registers", "launch__occupancy_limit_shared_mem",
        "sass__inst_executed_local_loads", "sass__inst_executed_local_stores", "sass__inst_executed_shared_loads",
        "sass__inst_executed_shared_stores", "l1tex__t_sector_pipe_lsu_mem_local_op_ld_hit_rate.pct", "lts__t_sector_hit_rate.pct",
        "l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum", "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum",
        "l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed",
        "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_elapsed", "sm__warps_active.avg.pct_of_peak_sustained_active",
        "smsp__issue_active.avg.pct_of_peak_sustained_active", "sm__icc_request_hit_rate.pct", "smsp__inst_executed.sum",
        "sm__cycles_elapsed.avg", "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum.per_cycle_elapsed",
        "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum.per_cycle_elapsed",
        "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum.per_cycle_elapsed"]
TO_BYTES = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def launches(report):
    raw = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
    rows = list(csv.reader(raw.splitlines()))
    hdr, units = rows[0], rows[1]
    return [({h: v for h, v in zip(hdr, vals)}, dict(zip(hdr, units))) for vals in rows[2:]]


def dram_bytes(d, units):
    return sum(float(d[k].replace(",", "")) * TO_BYTES[units[k]] for k in ("dram__bytes_read.sum", "dram__bytes_write.sum"))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--traffic-json")
    ap.add_argument("--kernel", help="demangled kernel name (prefix) whose DRAM bytes go to the JSON file")
    ap.add_argument("--passing", type=float, help="cut-passing events of the captured launch")
    ap.add_argument("--source", default="", help="the profiles/ file that holds this summary")
    args = ap.parse_args()
    first = None
    for d, units in launches(args.report):
        name = d.get("Kernel Name", "")
        print("== " + name[:110])
        for k in WANT:
            if k in d:
                print("  %-76s %-16s %s" % (k, units[k], d[k]))
        st = {k: float(v.replace(",", "")) for k, v in d.items()
              if k.startswith("smsp__average_warps_issue_stalled") and k.endswith("per_issue_active.ratio")}
        top = sorted(st.items(), key=lambda x: -x[1])[:9]
        try:      # executed fp64 flops of the launch = (dadd + dmul + 2 dfma thread-instructions per cycle) x elapsed cycles
            f = lambda k: float(d["smsp__sass_thread_inst_executed_op_%s_pred_on.sum.per_cycle_elapsed" % k].replace(",", ""))
            cyc = float(d["sm__cycles_elapsed.avg"].replace(",", ""))
            ms = float(d["gpu__time_duration.sum"].replace(",", "")) * {"ms": 1.0, "us": 1e-3, "s": 1e3}[units["gpu__time_duration.sum"]]
            fl = (f("dadd") + f("dmul") + 2.0 * f("dfma")) * cyc
            print("  executed fp64: %.4e flops per launch (%.4e thread-instructions) = %.2f TFLOP/s over the profiled launch"
                  % (fl, (f("dadd") + f("dmul") + f("dfma")) * cyc, fl / (ms * 1e-3) / 1e12))
        except (KeyError, ValueError):
            pass
        print("  stalls/issue: " + " ".join("%s=%.2f" % (k.replace("smsp__average_warps_issue_stalled_", "").replace("_per_issue_active.ratio", ""), v)
                                            for k, v in top))
        if args.kernel and first is None and args.kernel in name.replace("(int)", "").replace("void ", ""):
            first = dram_bytes(d, units)
    if args.traffic_json and first is not None and args.passing:
        rec = {}
        if os.path.exists(args.traffic_json):
            with open(args.traffic_json) as f:
                rec = json.load(f)
        rec[args.kernel] = {"dram_bytes_per_launch": first, "events_passing": args.passing,
                            "dram_bytes_per_passing_event": first / args.passing, "source": args.source}
        with open(args.traffic_json, "w") as f:
            json.dump(rec, f, indent=1, sort_keys=True)
            f.write("\n")


if __name__ == "__main__":
    main()
