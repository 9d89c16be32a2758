"""Builds libmvd.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1308_0730_b200.build [-j N] [--force]

One object per supported pencil length (csrc/lengths.def x csrc/inst.cu) plus csrc/mvd.cu and csrc/reduce_static.cu, compiled
in parallel, cached by modification time under csrc/build/<hash of the compiler flags>/ (so objects of an
experiment build are never linked into a normal one), linked into
paper_1308_0730_b200/libmvd.so.  Nothing here runs at import time of the package.
"""
from __future__ import annotations

import argparse
import hashlib
import os
import re
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libmvd.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "-Xfatbin=-compress-all"]
if os.environ.get("MVD_SKIP_MATH"):   # experiment: memory traffic only (results are wrong)
    FLAGS += ["-DMVD_SKIP_MATH"]
if os.environ.get("MVD_TMA_TILE"):   # experiment: tile width of the TMA-staged y/z passes
    FLAGS += ["-DMVD_TMA_TILE=" + os.environ["MVD_TMA_TILE"]]


def lengths():
    out = []
    for line in open(os.path.join(CSRC, "lengths.def")):
        m = re.match(r"\s*MVD_LEN\((\d+),\s*(\d+)\)", line)
        if m:
            out.append((int(m.group(1)), int(m.group(2))))
    return out


def _newer(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("command failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout[-4000:], r.stderr[-4000:]))
    return r


def build(jobs=None, force=False, verbose=True):
    global OBJ
    tag = hashlib.sha1(" ".join([NVCC] + FLAGS).encode()).hexdigest()[:10]
    OBJ = os.path.join(CSRC, "build", tag)
    os.makedirs(OBJ, exist_ok=True)
    stamp = os.path.join(CSRC, "build", "linked_flags")
    relink = not os.path.exists(stamp) or open(stamp).read() != tag
    hdr = [os.path.join(CSRC, f) for f in ("fft_reg.cuh", "pass_kernels.cuh", "pass_tma.cuh", "async_copy.cuh", "fft_ops.h")]
    tasks = []
    objs = []
    for a, b in lengths():
        o = os.path.join(OBJ, "inst_%d_%d.o" % (a, b))
        objs.append(o)
        src = os.path.join(CSRC, "inst.cu")
        if force or _newer(o, hdr + [src]):
            tasks.append([NVCC, *FLAGS, "-DMVD_INST_A=%d" % a, "-DMVD_INST_B=%d" % b, "-c", src, "-o", o])
    host_deps = hdr[4:] + [os.path.join(CSRC, f) for f in ("mvd.cu", "misc_kernels.cuh", "lengths.def")] + \
        [os.path.join(os.path.dirname(HERE), "include", "mvd.h")]
    # reduce_static.cu is self-contained (the no-allocation sum with its file-scope device array): it depends on mvd.h only
    for name, deps in (("mvd", host_deps), ("reduce_static", [os.path.join(CSRC, "reduce_static.cu"), host_deps[-1]])):
        o = os.path.join(OBJ, name + ".o")
        objs.append(o)
        src = os.path.join(CSRC, name + ".cu")
        if force or _newer(o, [d for d in deps if os.path.exists(d)]):
            tasks.append([NVCC, *FLAGS, "-c", src, "-o", o])
    jobs = jobs or max(1, len(os.sched_getaffinity(0)))
    if verbose:
        print("[mvd build] %d objects to compile, %d jobs" % (len(tasks), jobs), flush=True)
    with ThreadPoolExecutor(max_workers=jobs) as ex:
        list(ex.map(_run, tasks))
    if tasks or relink or not os.path.exists(LIB):
        _run([NVCC, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a", "-lcudart"])
        open(stamp, "w").write(tag)
    if verbose:
        print("[mvd build] %s" % LIB, flush=True)
    return LIB


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("-j", type=int, default=None)
    ap.add_argument("--force", action="store_true")
    a = ap.parse_args()
    build(a.j, a.force)
    sys.exit(0)
