"""Build libbang.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2205_06819_b200.build [--force]

The fused kernel is instantiated per (precision, supersampling) in separate translation units
(csrc/bang_fused_inst.cu compiled eight times) so that they build in parallel.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
SO = os.path.join(HERE, "libbang.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
         "--expt-relaxed-constexpr", "-Xptxas", "-v"]


def _sources():
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "bang.h")]
    return deps


def _units():
    units = [("bang_api.o", os.path.join(CSRC, "bang_api.cu"), [])]
    for tn in ("float", "double"):
        for s in (1, 2, 3, 4):
            units.append((f"bang_fused_{tn}_{s}.o", os.path.join(CSRC, "bang_fused_inst.cu"),
                          [f"-DBANG_INST_T={tn}", f"-DBANG_INST_TN={tn}", f"-DBANG_INST_S={s}"]))
    return units


def _compile(unit):
    obj, src, defs = unit
    out = os.path.join(OBJ, obj)
    cmd = [NVCC, *FLAGS, *os.environ.get("BANG_NVCC_EXTRA", "").split(), *defs, "-c", src, "-o", out]
    r = subprocess.run(cmd, capture_output=True, text=True)
    with open(out + ".log", "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed for {obj}:\n{r.stderr[-4000:]}")
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(p) for p in _sources())
    if not force and os.path.exists(SO) and os.path.getmtime(SO) >= newest:
        return SO
    os.makedirs(OBJ, exist_ok=True)
    units = _units()
    with ThreadPoolExecutor(max_workers=min(len(units), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(_compile, units))
    cmd = [NVCC, "-shared", "-o", SO, *objs, "-gencode", "arch=compute_100a,code=sm_100a", "-lcudart"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + r.stderr[-4000:])
    if verbose:
        print("built", SO)
    return SO


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
