"""Build the sm_100a C-ABI library in-tree: paper_2111_07396_b200/libss_b200.so.

nvcc cross-compiles without a GPU.  The kernels are spread over translation units that compile in parallel
(csrc/ss_warp_tu.cu is compiled once per mode and variant group).  -ffp-contract=off on the host side keeps the
window half-width arithmetic (csrc/ss_planner.h) un-fused; device-side the fold uses explicit __dmul_rn/__dsub_rn
(R2).  A hash of the sources is stored beside the library: load() rebuilds when it no longer matches.
"""
from __future__ import annotations

import glob
import hashlib
import os
import subprocess
import sys
import time
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libss_b200.so")
STAMP = LIB + ".srchash"
OBJ = os.path.join(HERE, "build")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "--extended-lambda", "-Xcompiler", "-fPIC", "-Xcompiler", "-ffp-contract=off"]


def units():
    """(object name, source, extra defines) of every translation unit."""
    u = []
    for src in sorted(glob.glob(os.path.join(CSRC, "*.cu"))):
        base = os.path.splitext(os.path.basename(src))[0]
        if base == "ss_warp_tu":
            for gv in (0, 1):
                for grp in (0, 1, 2):
                    for sh in (0, 1, 2, 3):
                        u.append((f"{base}_{gv}_{grp}_{sh}.o", src,
                                  [f"-DSS_TU_GV={gv}", f"-DSS_TU_GROUP={grp}", f"-DSS_TU_SHARED={sh}"]))
        elif base == "ss_group_tu":
            for gv in (0, 1):
                for g in (4, 8, 16):
                    for f32 in (0, 1, 2, 3):
                        u.append((f"{base}_{gv}_{g}_{f32}.o", src, [f"-DSS_TU_GV={gv}", f"-DSS_TU_G={g}", f"-DSS_TU_F32={f32}"]))
        elif base == "ss_cluster_tu":
            for gv in (0, 1):
                for c in (3, 4, 5):
                    u.append((f"{base}_{gv}_{c}.o", src, [f"-DSS_TU_GV={gv}", f"-DSS_TU_C={c}"]))
        elif base == "ss_block_tu":
            for part in range(14):
                u.append((f"{base}_{part}.o", src, [f"-DSS_TU_PART={part}"]))
        else:
            u.append((base + ".o", src, []))
    return u


def _deps():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh"))
                  + glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(HERE, "..", "include", "*.h"))
                  + [os.path.abspath(__file__)])


EXTRA = os.environ.get("SS_EXTRA_NVCC_FLAGS", "").split()      # experiments (-D switches); part of the source hash


def source_hash() -> str:
    h = hashlib.sha256()
    h.update(" ".join(EXTRA).encode())
    for d in _deps():
        h.update(os.path.basename(d).encode())
        with open(d, "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def is_fresh() -> bool:
    try:
        with open(STAMP) as f:
            return os.path.exists(LIB) and f.read().strip() == source_hash()
    except OSError:
        return False


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and is_fresh():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []

    def compile_one(u):
        obj, src, defs = u
        out = os.path.join(OBJ, obj)
        t0 = time.time()
        r = subprocess.run([NVCC] + FLAGS + EXTRA + extra + defs + ["-c", "-o", out, src], capture_output=True, text=True)
        if os.environ.get("SS_BUILD_TIMES"):
            sys.stderr.write(f"{obj}: {time.time() - t0:.1f} s\n")
        return out, r

    objs = []
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        for out, r in ex.map(compile_one, units()):
            if verbose or r.returncode != 0:
                sys.stderr.write(r.stdout + r.stderr)
            if r.returncode != 0:
                raise subprocess.CalledProcessError(r.returncode, r.args)
            objs.append(out)
    subprocess.run([NVCC, "-shared", "-o", LIB] + objs + ["-lcudart"], check=True)
    with open(STAMP, "w") as f:
        f.write(source_hash())
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
