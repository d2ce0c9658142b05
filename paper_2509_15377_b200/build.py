"""Builds libavm.so (the C-ABI CUDA library of include/avm.h) in-tree with nvcc for sm_100a.

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the snapshot.
Translation units: csrc/avm.cu (C ABI, host side, the small kernels and the parity hooks) and csrc/avm_transport_inst.cu
compiled once per (field kind, B) pair — the persistent transport kernel's instantiations — in parallel.
"""
from __future__ import annotations

import glob
import os
import shutil
import subprocess
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(_HERE)
SO = os.path.join(_HERE, "libavm.so")
SO_DEBUG = os.path.join(_HERE, "libavm_debug.so")      # build(defines=["-DAVM_DEBUG"]); loaded when AVM_LIBRARY points at it
OBJ_DIR = os.path.join(_HERE, "build")
CSRC = os.path.join(_HERE, "csrc")
DEPS = sorted(glob.glob(os.path.join(CSRC, "*"))) + [os.path.join(ROOT, "include", "avm.h"), os.path.abspath(__file__)]   # every file the build reads
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]
# (object name, source, extra defines)
UNITS = [("avm", "avm.cu", [])] + [(f"transport_fk{fk}_b{b}", "avm_transport_inst.cu", [f"-DAVM_INST_FK={fk}", f"-DAVM_INST_B={b}"])
                                   for fk in (0, 1, 2) for b in (0, 1)]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: libavm.so cannot be built")
    return exe


def is_fresh() -> bool:
    return os.path.exists(SO) and os.path.getmtime(SO) >= max(os.path.getmtime(p) for p in DEPS)


def build(force: bool = False, verbose: bool = False, defines=()) -> str:
    """defines: extra -D flags for every unit (e.g. ["-DAVM_DEBUG"]: bounds checks that __trap())."""
    if not force and not defines and is_fresh():
        return SO
    so = SO_DEBUG if defines else SO
    obj_dir = OBJ_DIR + ("_debug" if defines else "")
    os.makedirs(obj_dir, exist_ok=True)
    exe = nvcc()

    def compile_unit(u):
        name, src, defs = u
        obj = os.path.join(obj_dir, name + ".o")
        cmd = [exe] + NVCC_FLAGS + list(defs) + list(defines) + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, os.path.join(CSRC, src)]
        r = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src} {defs}:\n{r.stdout}\n{r.stderr}")
        return obj, r.stderr

    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 1)) as ex:
        results = list(ex.map(compile_unit, UNITS))
    if verbose:
        for _, log in results:
            print(log)
    subprocess.run([exe, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", so] + [o for o, _ in results], check=True, cwd=ROOT)
    return so


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, defines=[a for a in sys.argv[1:] if a.startswith("-D")]))
