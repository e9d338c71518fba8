"""Build libsdp.so (hand-written sm_100a kernels + C ABI) in-tree with nvcc.

``python -m paper_1302_5507_b200.build`` or ``build()`` from ``__graft_entry__``. Objects are
compiled in parallel; the score and traceback-DP kernels are instantiated for 32 column counts x
{forward, reverse, traceback} x {exact, padded}, split over sixteen K ranges by ``-DSDP_K_LO/-DSDP_K_HI``.
They (``score_cubin.cu``) are compiled to cubins whose scoring constants are sentinel immediates;
the cubins are embedded in the library as data (``.incbin``) and patched per context at load time
(``score_modules.cu``). The build checks that every sentinel sits only where the loader looks for it.
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


SENTINELS = {"negOc": 0x5D1A37C2, "negO": 0x2B6E4A91, "c2": 0x63C5195D, "Cd": 0x39E2746B, "e2": 0x1F83528E,   # score_kernel.cuh
             "t_negOf": 0x4E2B7D13, "t_negOe": 0x2D9C51E6, "t_c8": 0x35A8C6F1, "t_Cd8": 0x3B5E92A7}              # trace_kernel.cuh


def _units():
    units = [("sdp_api", "sdp_api.cu", []), ("bucket", "bucket.cu", []), ("traceback", "traceback.cu", []), ("thin_kernel", "thin_kernel.cu", []),
             ("microbench", "microbench.cu", []), ("best_read", "best_read.cu", []), ("best_read_static", "best_read_static.cu", []),
             ("mate", "mate.cu", []),
             ("score_modules", "score_modules.cu", []), ("slow_lane", "slow_lane.cu", [])]
    for r, (lo, hi) in enumerate(K_RANGES):
        units.append((f"cubin_r{r}", "score_cubin.cu", [f"-DSDP_K_LO={lo}", f"-DSDP_K_HI={hi}"]))
    return units


SCORE_SENTINELS = ("negOc", "negO", "c2", "Cd", "e2")
TRACE_SENTINELS = ("t_negOf", "t_negOe", "t_c8", "t_Cd8")


def check_cubin_sentinels(path: str) -> dict:
    """Every sentinel must occur in the cubin, and only as the 32-bit immediate of an instruction: bytes 4..7 of a
    16-byte slot of an executable section. Every kernel must use every sentinel of its family at least once (a score
    kernel the five of score_kernel.cuh, a traceback DP kernel the four of trace_kernel.cuh): a kernel in which ptxas
    derived a constant some other way would otherwise hide behind the hits of its neighbours in the same image.
    Returns the hit counts per sentinel, which the build embeds next to the image and score_modules.cu compares with
    what it patches at load time. (Same walk as patch_score_image in score_modules.cu.)"""
    import struct
    img = open(path, "rb").read()
    assert img[:4] == b"\x7fELF" and img[4] == 2 and img[5] == 1, f"{path}: not a little-endian ELF64"
    shoff, = struct.unpack_from("<Q", img, 0x28)
    shentsize, shnum, shstrndx = struct.unpack_from("<HHH", img, 0x3A)
    assert shentsize == 64
    str_off, = struct.unpack_from("<Q", img, shoff + 64 * shstrndx + 0x18)
    hits = {k: 0 for k in SENTINELS}
    by_val = {v: k for k, v in SENTINELS.items()}
    kernels = 0
    for s in range(shnum):
        name_off, typ, flags, _, off, size = struct.unpack_from("<IIQQQQ", img, shoff + 64 * s)
        if typ != 1 or not (flags & 4):
            continue
        assert off % 16 == 0
        name = img[str_off + name_off:img.index(b"\0", str_off + name_off)].decode()
        mine = {k: 0 for k in SENTINELS}
        for at in range(off, off + size - 15, 16):
            w, = struct.unpack_from("<I", img, at + 4)
            if w in by_val:
                mine[by_val[w]] += 1
        family = SCORE_SENTINELS if name.startswith(".text.sdp_score_k") else \
            TRACE_SENTINELS if name.startswith(".text.sdp_trace_k") else None
        if family is None:
            if any(mine.values()):
                raise RuntimeError(f"{path}: sentinel immediates in unexpected section {name}")
            continue
        kernels += 1
        for k in SENTINELS:
            if (mine[k] == 0) != (k not in family):
                raise RuntimeError(f"{path}: kernel {name[6:]} uses sentinel {k} {mine[k]} times: each kernel must use "
                                   "exactly the sentinels of its family, each at least once")
            hits[k] += mine[k]
    if kernels != 12:
        raise RuntimeError(f"{path}: {kernels} score / traceback kernels found, 12 expected (2 K x 6 variants)")
    for name, v in SENTINELS.items():
        total = img.count(struct.pack("<I", v))
        if hits[name] == 0 or total != hits[name]:
            raise RuntimeError(f"{path}: sentinel {name} found {total} times in the file but {hits[name]} times as an "
                               "instruction immediate: the immediate patching of score_modules.cu would miss a use")
    return hits


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
        if name.startswith("cubin_"):
            # device code only -> cubin -> checked -> wrapped into an object file as read-only data
            cubin = os.path.join(OBJ, name + ".cubin")
            flags = [f for f in NVCC_FLAGS if f not in ("-Xcompiler", "-fPIC")]
            cmd = [nvcc, *flags, *defs, "-cubin", os.path.join(CSRC, src), "-o", cubin]
        else:
            cmd = [nvcc, *NVCC_FLAGS, *defs, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {name}:\n{r.stdout}\n{r.stderr}")
        with open(os.path.join(OBJ, name + ".ptxas.txt"), "w") as f:
            f.write(r.stderr)
        if verbose:
            sys.stderr.write(r.stderr)
        if name.startswith("cubin_"):
            hits = check_cubin_sentinels(cubin)
            sym = "sdp_" + name                       # sdp_cubin_r<r>_start / _end / _hits
            asm = os.path.join(OBJ, name + ".S")
            with open(asm, "w") as f:
                # _hits: how often each sentinel occurs in this image, in SENTINELS order (= ScorePatch order)
                f.write(f'.section .rodata\n.balign 64\n.global {sym}_start\n.global {sym}_end\n.global {sym}_hits\n'
                        f'{sym}_start:\n.incbin "{cubin}"\n{sym}_end:\n.balign 4\n{sym}_hits:\n.long '
                        + ", ".join(str(hits[k]) for k in SENTINELS)
                        + '\n.section .note.GNU-stack,"",@progbits\n')
            r2 = subprocess.run(["gcc", "-c", "-fPIC", asm, "-o", obj], capture_output=True, text=True)
            if r2.returncode != 0:
                raise RuntimeError(f"embedding {cubin} failed:\n{r2.stderr}")
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
