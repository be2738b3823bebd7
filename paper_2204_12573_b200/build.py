"""Build libflare_b200.so (and the bench hooks libflare_probes.so) in-tree with nvcc for sm_100a (no torch
extension machinery needed: plain C-ABI shared objects).  `python -m paper_2204_12573_b200.build [--force]`."""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libflare_b200.so")
PROBES_LIB = os.path.join(HERE, "libflare_probes.so")  # bench hooks (include/flare_probes.h), a library of their own
SOURCES = ["flare_api.cu", "neighbor.cu", "descriptor.cu", "qform.cu", "force.cu", "integrate.cu", "analysis.cu", "domain.cu", "virial_static.cu"]
HEADERS = ["common.cuh", "basis.cuh", "kernels.cuh", os.path.join("..", "..", "include", "flare_b200.h"),
           os.path.join("..", "..", "include", "flare_probes.h")]
NVCC = os.environ.get("NVCC", "nvcc")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


def _stale(target: str, deps: list[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(src: str, verbose: bool) -> str:
    obj = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
    deps = [os.path.join(CSRC, src)] + [os.path.join(CSRC, h) for h in HEADERS]
    if _stale(obj, deps):
        cmd = [NVCC, *NVCC_FLAGS, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {src}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            sys.stderr.write(r.stderr)
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    if force:
        for f in os.listdir(OBJ):
            os.remove(os.path.join(OBJ, f))
        for lib in (LIB, PROBES_LIB):
            if os.path.exists(lib):
                os.remove(lib)
    with cf.ThreadPoolExecutor(max_workers=min(8, len(SOURCES) + 1)) as ex:
        objs = list(ex.map(lambda s: _compile(s, verbose), SOURCES + ["probes.cu"]))
    for lib, lib_objs in ((LIB, objs[:-1]), (PROBES_LIB, objs[-1:])):
        if _stale(lib, lib_objs):
            cmd = [NVCC, "-shared", "-o", lib, *lib_objs, "-gencode", "arch=compute_100a,code=sm_100a", "-lcudart"]
            r = subprocess.run(cmd, capture_output=True, text=True)
            if r.returncode != 0:
                raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
