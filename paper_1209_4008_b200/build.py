"""Build libgf.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1209_4008_b200.build [--force] [--verbose]

Objects go to paper_1209_4008_b200/_build/, the library to paper_1209_4008_b200/libgf.so.  The instances of the
sweep kernels are twelve translation units ((precision, reals-per-link) x {relaxation, monitored, heatbath}) and
compile in parallel.  A unit is rebuilt when any source or header is newer than its object.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
OBJ = os.path.join(HERE, "_build")
LIB = os.path.join(HERE, "libgf.so")

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]
FLAGS += os.environ.get("GF_NVCC_EXTRA", "").split()  # tuning experiments: extra -D switches (none in a normal build)

# (object name, source, extra defines).  The sweep kernels of one (precision, reals-per-link) are three units
# (gf_sweep_inst.cu: relaxation + launcher, monitored relaxation, heatbath), twelve in all.
UNITS = [
    ("gf_api.o", "gf_api.cu", []),
    ("gf_aux.o", "gf_aux.cu", []),
]
for _fp64, _R in ((0, 12), (0, 18), (1, 12), (1, 18)):
    for _part in range(3):
        UNITS.append((f"gf_sweep_f{64 if _fp64 else 32}_r{_R}_p{_part}.o", "gf_sweep_inst.cu",
                      [f"-DGF_INST_FP64={_fp64}", f"-DGF_INST_R={_R}", f"-DGF_INST_PART={_part}"]))


def _deps():
    out = [os.path.join(INCLUDE, "gf.h"), os.path.abspath(__file__)]
    for name in os.listdir(CSRC):
        if name.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, name))
    return out


def _stale(target: str, newest_dep: float) -> bool:
    return not os.path.exists(target) or os.path.getmtime(target) < newest_dep


def _compile(unit, verbose: bool):
    obj, src, defs = unit
    cmd = [NVCC, *ARCH, *FLAGS, *defs, "-I", INCLUDE, "-c", os.path.join(CSRC, src), "-o", os.path.join(OBJ, obj)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = os.path.join(OBJ, obj + ".ptxas.txt")
    with open(log, "w") as fh:  # registers / spills per kernel (-Xptxas -v)
        fh.write(" ".join(cmd) + "\n" + res.stderr)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed for {obj}:\n{res.stdout}\n{res.stderr}")
    if verbose:
        print(res.stderr)
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    newest = max(os.path.getmtime(p) for p in _deps())
    todo = [u for u in UNITS if force or _stale(os.path.join(OBJ, u[0]), newest)]
    if todo:
        with ThreadPoolExecutor(max_workers=min(len(todo), os.cpu_count() or 1)) as pool:
            list(pool.map(lambda u: _compile(u, verbose), todo))
    if todo or _stale(LIB, newest):
        tmp = LIB + f".{os.getpid()}.tmp"
        cmd = [NVCC, *ARCH, "-shared", "-o", tmp, *[os.path.join(OBJ, u[0]) for u in UNITS]]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
