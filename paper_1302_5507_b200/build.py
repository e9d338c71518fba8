"""Build libsdp.so (hand-written sm_100a kernels + C ABI) in-tree with nvcc.

``python -m paper_1302_5507_b200.build`` or ``build()`` from ``__graft_entry__``. Objects are
compiled in parallel; the score and traceback-DP kernels are instantiated for 32 column counts x
{forward, reverse, traceback} x {exact, padded}, split over sixteen translation units by ``-DSDP_K_LO/-DSDP_K_HI``.
"""
from __future__ import annotations

import hashlib
import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libsdp.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--expt-relaxed-constexpr"]
K_RANGES = [(2 * r + 1, 2 * r + 2) for r in range(16)]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if c and os.path.exists(c):
            return c
    raise RuntimeError("nvcc not found: libsdp needs the CUDA toolkit (there is no CPU fallback)")


def _deps_hash(extra: str) -> str:
    h = hashlib.sha256(extra.encode())
    for root in (CSRC, os.path.join(os.path.dirname(HERE), "include")):
        for fn in sorted(os.listdir(root)):
            if fn.endswith((".cu", ".cuh", ".h")):
                with open(os.path.join(root, fn), "rb") as f:
                    h.update(fn.encode())
                    h.update(f.read())
    return h.hexdigest()


def _units():
    units = [("sdp_api", "sdp_api.cu", []), ("bucket", "bucket.cu", []), ("traceback", "traceback.cu", []), ("thin_kernel", "thin_kernel.cu", []),
             ("microbench", "microbench.cu", []), ("best_read", "best_read.cu", []), ("mate", "mate.cu", [])]
    for r, (lo, hi) in enumerate(K_RANGES):
        units.append((f"score_r{r}", "score_inst.cu",
                      [f"-DSDP_K_LO={lo}", f"-DSDP_K_HI={hi}", f"-DSDP_K_FN=launch_score_r{r}",
                       f"-DSDP_T_FN=launch_trace_r{r}"]))
    return units


def build(force: bool = False, verbose: bool = False, jobs: int | None = None) -> str:
    nvcc = _nvcc()
    os.makedirs(OBJ, exist_ok=True)
    stamp = os.path.join(OBJ, "stamp.txt")
    want = _deps_hash(" ".join(NVCC_FLAGS))
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read() == want:
        return LIB

    def compile_one(unit):
        name, src, defs = unit
        obj = os.path.join(OBJ, name + ".o")
        cmd = [nvcc, *NVCC_FLAGS, *defs, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {name}:\n{r.stdout}\n{r.stderr}")
        with open(os.path.join(OBJ, name + ".ptxas.txt"), "w") as f:
            f.write(r.stderr)
        if verbose:
            sys.stderr.write(r.stderr)
        return obj

    jobs = jobs or min(12, (os.cpu_count() or 4))
    units = _units()
    only = os.environ.get("SDP_BUILD_UNITS")          # development: recompile just these units, reuse the other objects
    if only:
        names = set(only.split(","))
        todo = [u for u in units if u[0] in names or not os.path.exists(os.path.join(OBJ, u[0] + ".o"))]
    else:
        todo = units
    with ThreadPoolExecutor(max_workers=jobs) as ex:
        list(ex.map(compile_one, todo))
    objs = [os.path.join(OBJ, u[0] + ".o") for u in units]
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp, *objs]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    os.replace(tmp, LIB)
    with open(stamp, "w") as f:
        f.write(want if not only else "partial build")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
