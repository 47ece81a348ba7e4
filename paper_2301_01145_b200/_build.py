"""Build libsailffish_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

The kernel instantiations are spread over eight translation units (precision x kernel family), the
fp32 fast-path unit and the API unit; they are compiled in parallel and linked into one shared library that depends on the
CUDA runtime only.  Run as ``python -m paper_2301_01145_b200._build`` or through
``__graft_entry__.build()``.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
OBJ = HERE / "build"
LIB = HERE / "libsailffish_b200.so"

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-std=c++17", "-O3", "-lineinfo", "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"] + ARCH + os.environ.get("SF_NVCC_EXTRA", "").split()

UNITS = [("sf_api", "sf_api.cu", []), ("sf_fast", "sf_fast.cu", []), ("sf_static", "sf_static.cu", [])]
for kind in range(4):
    for tname, t in (("f32", "float"), ("f64", "double")):
        UNITS.append((f"sf_inst_k{kind}_{tname}", "sf_inst.cu", [f"-DSF_INST_KIND={kind}", f"-DSF_INST_T={t}"]))


def _sources_mtime() -> float:
    files = list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")) + [HERE.parent / "include" / "sailffish.h", Path(__file__)]
    return max(f.stat().st_mtime for f in files)


def _compile(unit) -> str:
    name, src, defs = unit
    obj = OBJ / f"{name}.o"
    cmd = [NVCC] + COMMON + defs + ["-c", str(CSRC / src), "-o", str(obj)]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed for {name}:\n{' '.join(cmd)}\n{r.stdout}\n{r.stderr}")
    return str(obj)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and LIB.exists() and LIB.stat().st_mtime >= _sources_mtime():
        return LIB
    OBJ.mkdir(exist_ok=True)
    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(_compile, UNITS))
    tmp = LIB.with_suffix(f".{os.getpid()}.tmp.so")
    cmd = [NVCC, "-shared", "--cudart", "static", "-o", str(tmp)] + ARCH + objs
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{' '.join(cmd)}\n{r.stdout}\n{r.stderr}")
    os.replace(tmp, LIB)
    if verbose:
        print(f"built {LIB}")
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
