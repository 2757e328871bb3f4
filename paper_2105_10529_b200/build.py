"""In-tree build of libmadflow_b200.so for sm_100a: run the amplitude generator, compile the C-ABI,
the no-alloc reduction and the eight per-process kernel objects in parallel with nvcc, link.  `python -m
paper_2105_10529_b200.build [--force]`."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libmadflow_b200.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _newer(target, deps):
    return os.path.exists(target) and all(os.path.getmtime(target) >= os.path.getmtime(d) for d in deps)


def build(force=False, verbose=False):
    obj_dir, lib = OBJ, LIB
    from .gen.__main__ import main as gen_main
    gen_main()
    os.makedirs(obj_dir, exist_ok=True)
    gen = [os.path.join(CSRC, "generated", f) for f in os.listdir(os.path.join(CSRC, "generated"))]
    kern = gen + [os.path.join(CSRC, f) for f in ("mf_device.cuh", "mf_event.cuh", "mf_kernels.cuh", "mf_proc.h")]
    api = kern + [os.path.join(CSRC, f) for f in ("mf_small_kernels.cuh", "mf_params.h")]
    api += [os.path.join(os.path.dirname(HERE), "include", "madflow_b200.h")]
    jobs = [("mf_api.o", os.path.join(CSRC, "mf_api.cu"), [])]
    jobs += [("mf_noalloc.o", os.path.join(CSRC, "mf_noalloc.cu"), [])]      # mf_reduce_weights_noalloc (static device scratch)
    jobs += [("mf_proc%d.o" % p, os.path.join(CSRC, "mf_proc.cu"), ["-DMF_PROC=%d" % p]) for p in range(8)]

    def compile_one(job):
        obj, src, extra = job
        out = os.path.join(obj_dir, obj)
        if not force and _newer(out, (api if obj in ("mf_api.o", "mf_noalloc.o") else kern) + [src]):
            return obj, "up to date"
        r = subprocess.run(["nvcc"] + NVCC_FLAGS + extra + ["-c", src, "-o", out], capture_output=True, text=True)
        with open(out + ".log", "w") as f:
            f.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed for %s:\n%s" % (obj, (r.stdout + r.stderr)[-4000:]))
        return obj, "compiled"

    with ThreadPoolExecutor(max_workers=8) as ex:
        results = list(ex.map(compile_one, jobs))
    objs = [os.path.join(obj_dir, j[0]) for j in jobs]
    if force or not _newer(lib, objs):
        subprocess.check_call(["nvcc", "-shared", "-o", lib] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"])
    if verbose:
        for obj, what in results:
            print(obj, what)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
