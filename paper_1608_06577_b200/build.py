"""In-tree build of the CUDA C-ABI library (libvh.so) for sm_100a with nvcc.

    python -m paper_1608_06577_b200.build [--force] [--verbose]

vh_api.cu and twelve launch units (vh_launch.cu compiled with -DVH_COMBO=0..11, one per EOS / viscous / Milne combination) are
compiled in parallel to objects under csrc/build/ and linked into libvh.so.  The built .so is git-ignored but travels with the
source tree; nothing is JIT-compiled at import time."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
SO = os.path.join(HERE, "libvh.so")
N_COMBO = 12
HEADERS = ["vh_device.cuh", "vh_math.cuh", "vh_kernels.cuh", "vh_kernels2.cuh", "vh_kernels3.cuh", "vh_kernels4.cuh", "vh_internal.cuh", "vh_eos_lattice.hpp",
           os.path.join("..", "..", "include", "vh.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC"]


def units():
    """(source, object, extra flags) of every translation unit."""
    out = [("vh_api.cu", "vh_api.o", [])]
    for k in range(N_COMBO):
        out.append(("vh_launch.cu", "vh_launch_%d.o" % k, ["-DVH_COMBO=%d" % k]))
    return out


def up_to_date() -> bool:
    if not os.path.exists(SO):
        return False
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, f) for f in ["vh_api.cu", "vh_launch.cu"] + HEADERS] + [os.path.abspath(__file__)]
    return all(os.path.getmtime(d) <= t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and up_to_date():
        return SO
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []

    def compile_one(u):
        src, obj, flags = u
        cmd = [nvcc] + NVCC_FLAGS + extra + flags + ["-c", "-o", os.path.join(OBJ, obj), os.path.join(CSRC, src)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        return u, r

    with ThreadPoolExecutor(max_workers=min(len(units()), os.cpu_count() or 1)) as ex:
        results = list(ex.map(compile_one, units()))
    for (src, obj, flags), r in results:
        if verbose or r.returncode != 0:
            sys.stderr.write("---- %s %s\n%s%s" % (src, " ".join(flags), r.stdout, r.stderr))
        if r.returncode != 0:
            raise RuntimeError("nvcc failed on %s %s" % (src, " ".join(flags)))
    cmd = [nvcc, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a", "-o", SO] + [os.path.join(OBJ, u[1]) for u in units()]
    subprocess.check_call(cmd)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
