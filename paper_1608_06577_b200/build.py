"""In-tree build of the CUDA C-ABI library (libvh.so) for sm_100a with nvcc.

    python -m paper_1608_06577_b200.build [--force] [--verbose]

vh_api.cu and twelve launch units (vh_launch.cu compiled with -DVH_COMBO=0..11, one per EOS / viscous / Milne combination) are
compiled in parallel to objects under csrc/build/<precision>/ and linked into libvh.so (real = double) and libvh_f32.so
(real = float, -DVH_REAL=float; `--f64` / `--f32` build only one of them).  The built .so is git-ignored but travels with the
source tree; nothing is JIT-compiled at import time."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
SO = os.path.join(HERE, "libvh.so")
# real = double: libvh.so (the product, everything BASELINE.json measures); real = float: libvh_f32.so
LIBS = {"f64": (SO, []), "f32": (os.path.join(HERE, "libvh_f32.so"), ["-DVH_REAL=float"])}
N_COMBO = 12
HEADERS = ["vh_real.cuh", "vh_peaks.cuh", "vh_device.cuh", "vh_math.cuh", "vh_kernels.cuh", "vh_kernels2.cuh", "vh_kernels3.cuh", "vh_kernels4.cuh", "vh_kernels5.cuh", "vh_internal.cuh", "vh_eos_lattice.hpp",
           os.path.join("..", "..", "include", "vh.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC"]


def units():
    """(source, object, extra flags) of every translation unit."""
    out = [("vh_api.cu", "vh_api.o", []), ("vh_launch_reduced.cu", "vh_launch_reduced.o", [])]
    for k in range(N_COMBO):
        out.append(("vh_launch.cu", "vh_launch_%d.o" % k, ["-DVH_COMBO=%d" % k]))
    return out


def up_to_date(so) -> bool:
    if not os.path.exists(so):
        return False
    t = os.path.getmtime(so)
    deps = [os.path.join(CSRC, f) for f in ["vh_api.cu", "vh_launch.cu", "vh_launch_reduced.cu"] + HEADERS] + [os.path.abspath(__file__)]
    return all(os.path.getmtime(d) <= t for d in deps)


def build(force: bool = False, verbose: bool = False, precisions=("f64", "f32")) -> str:
    """Builds the library of every requested precision that is out of date; returns the path of libvh.so."""
    todo = [p for p in precisions if force or not up_to_date(LIBS[p][0])]
    if not todo:
        return SO
    nvcc = os.environ.get("NVCC", "nvcc")
    extra = ["-Xptxas", "-v"] if verbose else []
    jobs = []
    for p in todo:
        os.makedirs(os.path.join(OBJ, p), exist_ok=True)
        for src, obj, flags in units():
            jobs.append((p, src, os.path.join(OBJ, p, obj), flags + LIBS[p][1]))

    def compile_one(j):
        p, src, obj, flags = j
        cmd = [nvcc] + NVCC_FLAGS + extra + flags + ["-c", "-o", obj, os.path.join(CSRC, src)]
        return j, subprocess.run(cmd, capture_output=True, text=True)

    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as ex:
        results = list(ex.map(compile_one, jobs))
    for (p, src, obj, flags), r in results:
        if verbose or r.returncode != 0:
            sys.stderr.write("---- %s %s\n%s%s" % (src, " ".join(flags), r.stdout, r.stderr))
        if r.returncode != 0:
            raise RuntimeError("nvcc failed on %s %s" % (src, " ".join(flags)))
    for p in todo:
        objs = [os.path.join(OBJ, p, u[1]) for u in units()]
        subprocess.check_call([nvcc, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIBS[p][0]] + objs)
    return SO


if __name__ == "__main__":
    only = [p for p in LIBS if "--" + p in sys.argv]
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, precisions=tuple(only) or tuple(LIBS)))
