"""TEST INFRASTRUCTURE ONLY: builds oracle/libvh_oracle.so (serial CPU oracle, g++ -O2, no CUDA).

Run as `python oracle/build.py`; also called by __graft_entry__.build() ("building the checker is not using it").
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SO = os.path.join(HERE, "libvh_oracle.so")
SRCS = [os.path.join(HERE, "vh_oracle_capi.cpp"), os.path.join(HERE, "vh_oracle_count.cpp")]
DEPS = SRCS + [os.path.join(HERE, "vh_oracle.hpp"), os.path.join(HERE, "vh_oracle_lattice.hpp")]


def build(force: bool = False) -> str:
    if not force and os.path.exists(SO) and all(os.path.getmtime(SO) >= os.path.getmtime(d) for d in DEPS):
        return SO
    cmd = ["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-Wall", "-o", SO] + SRCS
    subprocess.check_call(cmd)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
