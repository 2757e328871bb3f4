"""python -m paper_2105_10529_b200.gen [outdir] -- write the generated |M|^2 device code
(csrc/generated/mf_me2_*.cuh) and print the exact per-event operation counts."""
import os
import sys
from . import amplitudes as A
from . import lanes as L
from . import quarks as Q


def _write(path, text):
    old = open(path).read() if os.path.exists(path) else None
    if old != text:
        with open(path, "w") as f:
            f.write(text)


def lean_flops(ng):
    """flops of the leanest form the generator knows: every helicity configuration unrolled, everything shared"""
    gen = A.Gen(ng, loop_legs=(), parity=True, basis="linear")
    gen.build()
    c = gen.g.counts([gen.out])
    return c["add"] + c["mul"] + 2 * c["fma"]


def main(outdir=None):
    here = os.path.dirname(os.path.abspath(__file__))
    outdir = outdir or os.path.join(os.path.dirname(here), "csrc", "generated")
    os.makedirs(outdir, exist_ok=True)
    for fname in A.PROCESSES:
        gen = A.generate(fname)
        text, tot = A.emit_function(gen, fname)
        if fname == "mf_me2_gg_ttg":
            text += "#define MF_ME2_GG_TTG_NFLOPS_MIN %dull\n" % lean_flops(3)
            text += A.emit_function_smem(A.generate_smem(fname), fname, A.SMEM_CLOBBER_EVERY, A.SMEM_HOIST_COST, A.SMEM_RCP_LEAF)
        _write(os.path.join(outdir, fname + ".cuh"), text)
        print("%-22s add %7d mul %7d fma %7d rcp %3d  flops/event %8d  inputs %d" % (
            fname, tot["add"], tot["mul"], tot["fma"], tot["rcp"],
            tot["add"] + tot["mul"] + 2 * tot["fma"], len(gen.input_names)))
    for fname, make in Q.PROCESSES_2Q.items():          # q q~ -> t t~ g, q g -> t t~ q
        gen = make()
        gen.build()
        text, tot = A.emit_function(gen, fname)
        _write(os.path.join(outdir, fname + ".cuh"), text)
        print("%-22s add %7d mul %7d fma %7d rcp %3d  flops/event %8d  inputs %d" % (
            fname, tot["add"], tot["mul"], tot["fma"], tot["rcp"],
            tot["add"] + tot["mul"] + 2 * tot["fma"], len(gen.input_names)))
    # gg -> tt~gg: one event over four lanes.  ALGORITHMIC counts (mf_me_flops) = the one-thread organisation with
    # every current and spinor shared (the 16 gluon polarisations as a loop): what the lanes compute without
    # their redundancy; executed = 4 x the per-lane counts.
    fname = "mf_me2_gg_ttgg_lanes"
    gen = L.GenLanes()
    gen.build()
    text, tot, _parts = L.emit_lanes(gen, fname)
    one = A.Gen(4, loop_legs=(0, 1, 2, 3), parity=True, basis="linear")
    one.build()
    p0, b0, _h = one.g.plan([one.out], None)
    c0, c1 = one.g.count_list(p0), one.g.count_list(b0)
    alg = {k: c0[k] + 16 * (c1[k] + (1 if k == "add" else 0)) for k in c0}
    text += "// algorithmic (one thread per event, everything shared): %d add, %d mul, %d fma  (flops = %d)\n" % (
        alg["add"], alg["mul"], alg["fma"], alg["add"] + alg["mul"] + 2 * alg["fma"])
    text += "#define MF_ME2_GG_TTGG_NADD %dull\n#define MF_ME2_GG_TTGG_NMUL %dull\n#define MF_ME2_GG_TTGG_NFMA %dull\n" % (
        alg["add"], alg["mul"], alg["fma"])
    text += "#define MF_ME2_GG_TTGG_NFLOPS_MIN %dull\n" % lean_flops(4)
    _write(os.path.join(outdir, fname + ".cuh"), text)
    print("%-22s add %7d mul %7d fma %7d rcp %3d  flops/event %8d  (per lane x 4; algorithmic %d)  inputs %d" % (
        fname, 4 * tot["add"], 4 * tot["mul"], 4 * tot["fma"], 4 * tot["rcp"],
        4 * (tot["add"] + tot["mul"] + 2 * tot["fma"]), alg["add"] + alg["mul"] + 2 * alg["fma"], len(gen.input_names)))


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else None)
