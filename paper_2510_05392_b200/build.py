"""In-tree build of the CUDA library (libmg5_b200.so) for sm_100a.

  python -m paper_2510_05392_b200.build        # generate the diagram programs, compile, link

Steps: (1) gen/emit_cuda.py writes csrc/generated/*; (2) every .cu is compiled to an object with
`nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo` (in parallel); (3) objects are linked into
paper_2510_05392_b200/libmg5_b200.so.  Objects are rebuilt only when a source or header is newer.
"""
from __future__ import annotations

import concurrent.futures as cf
import glob
import os
import subprocess
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
GEN = os.path.join(CSRC, "generated")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libmg5_b200.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]

# per-file extra flags (none at present: the all-fp32 instantiation of the 1240-diagram process is a translation unit of
# its own, generated/proc_gg_ttxggg_f32.cu, so that it compiles in parallel with the fp64 one)
EXTRA = {}


import re

_INC = re.compile(r'^\s*#\s*include\s+"([^"]+)"', re.M)


def _deps(path, seen=None):
    """the file and every header it includes with "..." (recursively)"""
    seen = set() if seen is None else seen
    path = os.path.normpath(path)
    if path in seen or not os.path.exists(path):
        return seen
    seen.add(path)
    for inc in _INC.findall(open(path).read()):
        _deps(os.path.join(os.path.dirname(path), inc), seen)
    return seen


def _compile(src, verbose):
    base = os.path.basename(src)
    obj = os.path.join(OBJ, base.replace(".cu", ".o"))
    dep_m = max(os.path.getmtime(d) for d in _deps(src))
    if os.path.exists(obj) and os.path.getmtime(obj) >= dep_m:
        return obj, 0.0, ""
    t = time.time()
    cmd = ["nvcc"] + NVCC_FLAGS + EXTRA.get(base, []) + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed for {src}:\n{r.stdout}\n{r.stderr}")
    return obj, time.time() - t, r.stderr


def build(verbose: bool = False, jobs: int | None = None) -> str:
    from .gen import emit_cuda, emit_hs, emit_hsg
    emit_cuda.generate_all(GEN)
    emit_hs.emit(GEN)
    emit_hsg.emit(GEN)
    os.makedirs(OBJ, exist_ok=True)
    srcs = sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(GEN, "*.cu")))
    # biggest first
    srcs.sort(key=lambda s: -os.path.getsize(s.replace("proc_", "").replace(".cu", "_jamps.cuh"))
              if os.path.exists(s.replace("proc_", "").replace(".cu", "_jamps.cuh")) else 0)
    objs = []
    with cf.ThreadPoolExecutor(max_workers=jobs or os.cpu_count()) as ex:
        for obj, dt, log in ex.map(lambda s: _compile(s, verbose), srcs):
            objs.append(obj)
            if dt and verbose:
                print(f"[build] {os.path.basename(obj)} {dt:.1f}s")
                if log:
                    with open(obj + ".ptxas.log", "w") as f:
                        f.write(log)
    if not os.path.exists(LIB) or any(os.path.getmtime(o) > os.path.getmtime(LIB) for o in objs):
        subprocess.check_call(["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    t0 = time.time()
    print(build(verbose=True), f"{time.time() - t0:.1f}s")
