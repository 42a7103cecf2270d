"""Builds ``libbiobeam_b200.so`` in-tree with nvcc for sm_100a (no GPU needed to compile).

``python -m paper_1706_02261_b200.build [--force]`` or :func:`build_library`.  The kernels
are instantiated per line length (``bb_inst.cu`` compiled once per TX = Nx/32); the objects
are compiled in parallel and linked into one shared library next to this file.
"""
from __future__ import annotations

import concurrent.futures
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "_build")
LIB = os.path.join(HERE, "libbiobeam_b200.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
TXS = (1, 2, 4, 8, 16, 32)
PXS = (1, 2, 4, 8)

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-I", INCLUDE]


def _nvcc() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def _sources():
    deps = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC))] + [os.path.join(INCLUDE, "bb.h")]
    return deps


def _digest(deps) -> str:
    """Content hash of the sources: a copy of the tree (fresh mtimes, e.g. on the GPU box) must not
    trigger a rebuild of an up-to-date library."""
    h = hashlib.sha256()
    for d in deps:
        h.update(os.path.basename(d).encode())
        with open(d, "rb") as f:
            h.update(f.read())
    h.update(" ".join(NVCC_FLAGS[:-1]).encode())
    return h.hexdigest()


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("command failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return r.stdout + r.stderr


def build_library(force: bool = False, verbose: bool = False) -> str:
    deps = _sources()
    stamp = LIB + ".sha256"
    digest = _digest(deps)
    if not force and os.path.exists(LIB) and os.path.exists(stamp):
        with open(stamp) as f:
            if f.read().strip() == digest:
                return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()
    jobs = []
    for tx in TXS:
        obj = os.path.join(OBJ, "bb_inst_tx%d.o" % tx)
        jobs.append((obj, [nvcc, *NVCC_FLAGS, "-DBB_TX=%d" % tx, "-c", os.path.join(CSRC, "bb_inst.cu"), "-o", obj]))
    for px in PXS:
        for cw in (4, 8):
            for bt in (0, 1):
                obj = os.path.join(OBJ, "bb_inst16_px%d_cw%d_b%d.o" % (px, cw, bt))
                jobs.append((obj, [nvcc, *NVCC_FLAGS, "-DBB_PX=%d" % px, "-DBB_CW=%d" % cw, "-DBB_BATCH=%d" % bt, "-c",
                                   os.path.join(CSRC, "bb_inst16.cu"), "-o", obj]))
    for px in (1, 2, 4, 8):
        for cw in (4, 8):
            for bt in (0, 1):
                obj = os.path.join(OBJ, "bb_inst8_px%d_cw%d_b%d.o" % (px, cw, bt))
                jobs.append((obj, [nvcc, *NVCC_FLAGS, "-DBB_PX=%d" % px, "-DBB_CW=%d" % cw, "-DBB_BATCH=%d" % bt, "-c",
                                   os.path.join(CSRC, "bb_inst8.cu"), "-o", obj]))
    obj_c = os.path.join(OBJ, "bb_instc.o")
    jobs.append((obj_c, [nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, "bb_instc.cu"), "-o", obj_c]))
    obj_api = os.path.join(OBJ, "bb_api.o")
    jobs.append((obj_api, [nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, "bb_api.cu"), "-o", obj_api]))
    obj_probe = os.path.join(OBJ, "bb_probe.o")
    jobs.append((obj_probe, [nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, "bb_probe.cu"), "-o", obj_probe]))
    obj_na = os.path.join(OBJ, "bb_noalloc.o")
    jobs.append((obj_na, [nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, "bb_noalloc.cu"), "-o", obj_na]))
    todo = [(o, c) for o, c in jobs if force or _stale(o, deps)]          # objects newer than every source are kept
    with concurrent.futures.ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        for out in ex.map(lambda oc: _run(oc[1]), todo):
            if verbose and out.strip():
                print(out)
    tmp = LIB + ".tmp%d" % os.getpid()
    _run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp, *[o for o, _ in jobs],
          "-lcudart_static", "-ldl", "-lrt", "-lpthread"])
    os.replace(tmp, LIB)
    with open(stamp, "w") as f:
        f.write(digest + "\n")
    return LIB


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose=True))
