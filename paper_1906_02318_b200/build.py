"""Builds paper_1906_02318_b200/libmpmi.so (sm_100a only) from csrc/ with nvcc, in-tree.

    python -m paper_1906_02318_b200.build [--force]

One translation unit per (lifted dim D, kernel mode) so that the heavily unrolled kernels compile
in parallel; nvcc cross-compiles without a GPU.
"""
import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libmpmi.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v"] + os.environ.get("MPMI_NVCC_EXTRA", "").split()     # e.g. -DMPMI_TC_DEBUG: in-kernel clock64 timelines

UNITS = [("api", "mpmi_api.cu", []), ("noalloc", "noalloc.cu", [])]
UNITS += [(f"reg{d}_{m}", "inst_reg.cu", [f"-DMPMI_D={d}", f"-DMPMI_MODE={m}"]) for d in (32, 16, 8) for m in (0, 1)]
UNITS += [(f"lat{d}", "inst_lat.cu", [f"-DMPMI_D={d}"]) for d in (32, 16, 8)]
UNITS += [(f"regn{d}_{m}", "inst_reg.cu", [f"-DMPMI_D={d}", f"-DMPMI_MODE={m}", "-DMPMI_NOISE=1"]) for d in (32, 16, 8) for m in (0, 1)]
UNITS += [(f"tilen{d}_{m}", "inst_tile.cu", [f"-DMPMI_D={d}", f"-DMPMI_MODE={m}", "-DMPMI_NOISE=1"]) for d in (128, 64) for m in (0, 1)]
UNITS += [("relift", "inst_relift.cu", []), ("affine", "inst_affine.cu", [])]
UNITS += [("split", "inst_split.cu", []), ("splitn", "inst_split.cu", ["-DMPMI_NOISE=1"])]
UNITS += [(f"tc_{m}", "inst_tc.cu", [f"-DMPMI_MODE={m}"]) for m in (0, 1)]
UNITS += [(f"tile{d}_{m}", "inst_tile.cu", [f"-DMPMI_D={d}", f"-DMPMI_MODE={m}"]) for d in (128, 64) for m in (0, 1)]


def _source_hash():
    h = hashlib.sha256()
    for root in (CSRC, os.path.join(os.path.dirname(HERE), "include")):
        for f in sorted(os.listdir(root)):
            if f.endswith((".cu", ".cuh", ".h")):
                h.update(f.encode())
                h.update(open(os.path.join(root, f), "rb").read())
    h.update(" ".join(FLAGS).encode())
    return h.hexdigest()


def _compile(unit):
    name, src, defs = unit
    obj = os.path.join(OBJ, name + ".o")
    log = os.path.join(OBJ, name + ".ptxas.log")
    cmd = [NVCC, *FLAGS, *defs, "-c", os.path.join(CSRC, src), "-o", obj]
    p = subprocess.run(cmd, capture_output=True, text=True)
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + p.stdout + p.stderr)
    if p.returncode != 0:
        raise RuntimeError(f"nvcc failed for {name}:\n{p.stderr[-4000:]}")
    return obj


def build(force=False, verbose=False):
    os.makedirs(OBJ, exist_ok=True)
    stamp = os.path.join(OBJ, "stamp")
    h = _source_hash()
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read() == h:
        return LIB
    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(_compile, UNITS))
    p = subprocess.run([NVCC, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a"],
                       capture_output=True, text=True)
    if p.returncode != 0:
        raise RuntimeError("link failed:\n" + p.stderr[-4000:])
    with open(stamp, "w") as f:
        f.write(h)
    if verbose:
        print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
