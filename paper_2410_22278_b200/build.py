"""Builds libpbc_jk.so (the C-ABI library of include/pbc_jk.h) in-tree with nvcc for sm_100a.

    python -m paper_2410_22278_b200.build [--force] [-j N]

One object per instantiation unit (the real-space kernel families are compiled once per
angular-momentum class group so the classes build in parallel); objects are cached under
csrc/build/ keyed by the hash of the sources and flags.
"""
from __future__ import annotations

import argparse
import concurrent.futures as cf
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libpbc_jk.so")
PEAKS_LIB = os.path.join(HERE, "libpbc_jk_benchpeaks.so")     # bench.py's roofline denominators; not part of the product ABI
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-fopenmp,-O2", "-I", INCLUDE, "-I", OBJ]

# headers each source includes (directly or not): a change recompiles only the units that see it
_SR_H = ["pbcjk_common.h", "pbcjk_md.cuh", "pbcjk_sr.cuh"]
_SRK_H = _SR_H + ["pbcjk_srk.cuh", "gen_sr_k.py"]     # the K evaluators are generated into csrc/build/gen
HEADERS = {"pbcjk_api.cu": _SR_H + ["pbcjk_lr.cuh", "pbcjk_1e.cuh", os.path.join(INCLUDE, "pbc_jk.h")],
           "pbcjk_lr.cu": ["pbcjk_common.h", "pbcjk_md.cuh", "pbcjk_lr.cuh"],
           "pbcjk_1e.cu": _SR_H + ["pbcjk_lr.cuh", "pbcjk_1e.cuh"],
           "sr_dispatch.cu": _SR_H, "sr_j_inst.cu": _SR_H, "sr_k_inst.cu": _SRK_H, "bench_peaks.cu": []}


def _units():
    """(object name, source, extra defines)"""
    u = [("api", "pbcjk_api.cu", []), ("lr", "pbcjk_lr.cu", []), ("one_electron", "pbcjk_1e.cu", []),
         ("sr_dispatch", "sr_dispatch.cu", [])]
    for lb in range(5):
        u.append((f"sr_j_{lb}", "sr_j_inst.cu", [f"-DJ_LB={lb}"]))
    for la in range(3):
        for ld in range(la + 1):
            for lb in range(3):
                for mixed in (0, 1):     # fp64 kernels, and fp64+fp32 kernels of the mixed-precision mode
                    u.append((f"sr_k_{la}{lb}{ld}_{mixed}", "sr_k_inst.cu",
                              [f"-DK_LA={la}", f"-DK_LB={lb}", f"-DK_LD={ld}", f"-DK_MIXED={mixed}"]))
    return u


def _digest(src: str, defs) -> str:
    h = hashlib.sha256()
    for f in [os.path.join(CSRC, src)] + [f if os.path.isabs(f) else os.path.join(CSRC, f) for f in HEADERS[src]]:
        with open(f, "rb") as fh:
            h.update(fh.read())
    # flags enter the key with the checkout path stripped: the objects built here stay valid on the GPU box
    h.update(" ".join(NVCC_FLAGS + list(defs)).replace(os.path.dirname(HERE), ".").encode())
    return h.hexdigest()[:16]


def _compile(unit, force: bool, verbose: bool) -> str:
    name, src, defs = unit
    obj = os.path.join(OBJ, name + ".o")
    stamp = obj + ".hash"
    dig = _digest(src, defs)
    if not force and os.path.exists(obj) and os.path.exists(stamp) and open(stamp).read() == dig:
        return obj
    cmd = ["nvcc"] + NVCC_FLAGS + defs + ["-c", os.path.join(CSRC, src), "-o", obj]
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed for {name}:\n{r.stdout}\n{r.stderr}")
    if verbose:
        with open(obj + ".ptxas.txt", "w") as fh:
            fh.write(r.stderr)
    with open(stamp, "w") as fh:
        fh.write(dig)
    return obj


def build(force: bool = False, jobs: int = 0, verbose: bool = False, only=None) -> str:
    """only: optional list of unit-name prefixes to (re)compile (development aid; no link unless all objects exist)"""
    os.makedirs(OBJ, exist_ok=True)
    sys.path.insert(0, CSRC)
    import gen_sr_k                                   # straight-line K quartet evaluators, one header per unit
    sys.path.pop(0)
    gen_sr_k.main(os.path.join(OBJ, "gen"))
    units = _units()
    if only:
        units = [u for u in units if any(u[0].startswith(p) for p in only)]
    jobs = jobs or max(1, min(len(units), (os.cpu_count() or 2)))
    # heaviest units first so the long compiles overlap with everything else
    heavy = ["sr_k_222_1", "sr_k_221_1", "sr_k_212_1", "sr_k_222_0", "sr_k_220_1", "sr_k_221_0", "sr_k_212_0", "sr_k_211_1",
             "sr_k_220_0", "sr_j_4", "sr_j_3"]
    units.sort(key=lambda u: heavy.index(u[0]) if u[0] in heavy else len(heavy))
    with cf.ThreadPoolExecutor(max_workers=jobs) as ex:
        objs = list(ex.map(lambda u: _compile(u, force, verbose), units))
    if only:
        return ""
    newest = max(os.path.getmtime(o) for o in objs)
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < newest:
        cmd = ["nvcc", "-shared", "-o", LIB] + objs + ["-Xcompiler", "-fopenmp", "-lgomp"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    pk = _compile(("bench_peaks", "bench_peaks.cu", []), force, verbose)
    if force or not os.path.exists(PEAKS_LIB) or os.path.getmtime(PEAKS_LIB) < os.path.getmtime(pk):
        r = subprocess.run(["nvcc", "-shared", "-o", PEAKS_LIB, pk], capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return LIB


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--force", action="store_true")
    ap.add_argument("-j", type=int, default=0)
    ap.add_argument("-v", action="store_true", help="keep ptxas -v output next to each object")
    ap.add_argument("--only", nargs="*", help="compile only the units whose name starts with one of these (no link)")
    a = ap.parse_args()
    print(build(a.force, a.j, a.v, a.only))
    sys.exit(0)
