"""Build the C-ABI CUDA library (include/sph.h) for sm_100a with nvcc, in-tree.

    python -m paper_2511_11425_b200.build [--force]

Produces paper_2511_11425_b200/libsph_b200.so.  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_OBJ = os.path.join(_HERE, "build")
LIB = os.path.join(_HERE, "libsph_b200.so")
SOURCES = ["sph_api.cu", "sph_build.cu", "sph_density.cu", "sph_forces.cu", "sph_misc.cu",
           "sph_integrate.cu", "sph_interface.cu", "sph_rungs.cu", "sph_active.cu", "sph_tile_density.cu", "sph_tile_forces.cu", "sph_forces_list.cu", "sph_forces_tlist.cu", "sph_static.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-ftz=true",
              "--expt-extended-lambda", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _deps():
    d = [os.path.join(_CSRC, f) for f in os.listdir(_CSRC)]
    d.append(os.path.join(os.path.dirname(_HERE), "include", "sph.h"))
    return d


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    os.makedirs(_OBJ, exist_ok=True)
    nvcc = _nvcc()

    def one(src):
        obj = os.path.join(_OBJ, src.replace(".cu", ".o"))
        cmd = [nvcc, *NVCC_FLAGS, *os.environ.get("SPH_NVCC_EXTRA", "").split(), "-c", os.path.join(_CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {src}:\n{r.stdout}\n{r.stderr}")
        with open(obj + ".ptxas.txt", "w") as f:
            f.write(" ".join(cmd) + "\n" + r.stderr)
        if verbose:
            print(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(one, SOURCES))
    tmp = LIB + f".{os.getpid()}.tmp"
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp,
                           *objs, "-lcudart"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
