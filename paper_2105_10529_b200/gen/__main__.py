"""python -m paper_2105_10529_b200.gen [outdir] -- write the generated |M|^2 device code
(csrc/generated/mf_me2_*.cuh) and print the exact per-event operation counts."""
import os
import sys
from . import amplitudes as A


def main(outdir=None):
    here = os.path.dirname(os.path.abspath(__file__))
    outdir = outdir or os.path.join(os.path.dirname(here), "csrc", "generated")
    os.makedirs(outdir, exist_ok=True)
    for fname in A.PROCESSES:
        gen = A.generate(fname)
        text, tot = A.emit_function(gen, fname)
        path = os.path.join(outdir, fname + ".cuh")
        old = open(path).read() if os.path.exists(path) else None
        if old != text:
            with open(path, "w") as f:
                f.write(text)
        print("%-16s add %7d mul %7d fma %7d rcp %3d  flops/event %8d  inputs %d" % (
            fname, tot["add"], tot["mul"], tot["fma"], tot["rcp"],
            tot["add"] + tot["mul"] + 2 * tot["fma"], len(gen.input_names)))


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else None)
