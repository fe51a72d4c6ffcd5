"""Build the C / OpenMP oracle twin (oracle/oracle_c.c -> oracle/liboracle_c.so) with gcc.
Test infrastructure only; `__graft_entry__.build()` calls this so the checker exists on the GPU
box (building the checker is not using it).

    python -m oracle.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "oracle_c.c")
LIB = os.path.join(HERE, "liboracle_c.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    # the image has several gcc front ends and not all of them find libgomp: try them in turn,
    # and fall back to a single-threaded build (same results, one core) if none does
    tried = []
    cands = [os.environ.get("CC"), "/usr/bin/gcc-13", "/usr/bin/gcc", "gcc", "cc"]
    for omp in (["-fopenmp"], []):
        for cc in [c for c in cands if c]:
            cmd = [cc, "-O2", *omp, "-shared", "-fPIC", "-std=c11", SRC, "-o", LIB, "-lm"]
            try:
                res = subprocess.run(cmd, capture_output=True, text=True)
            except OSError as e:
                tried.append(f"{cc}: {e}")
                continue
            if res.returncode == 0:
                return LIB
            tried.append(f"{' '.join(cmd)}: {res.stderr.strip()[:200]}")
    sys.stderr.write("\n".join(tried) + "\n")
    raise RuntimeError("could not build liboracle_c.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
