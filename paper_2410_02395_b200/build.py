"""Builds libmbs_b200.so (the C-ABI library of include/mbs.h) in-tree with nvcc for sm_100a.

    python -m paper_2410_02395_b200.build [--force]

One translation unit per FFT size (csrc/fft_inst.cu with -DMBS_FFT_SIZE=M) so the sizes compile in
parallel.  Objects go to <repo>/build/, the library next to this file.
"""
from __future__ import annotations

import concurrent.futures
import hashlib
import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJDIR = os.path.join(ROOT, "build", "obj")
LIB = os.path.join(HERE, "libmbs_b200.so")

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3",
         "--expt-relaxed-constexpr", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


def fft_sizes():
    text = open(os.path.join(CSRC, "fft_plans.h")).read()
    body = text.split("#define MBS_FOR_EACH_FFT_SIZE(X)")[1]
    return [int(m) for m in re.findall(r"X\((\d+)\)", body)]


def _source_digest():
    h = hashlib.sha256()
    for d in (CSRC, os.path.join(ROOT, "include")):
        for name in sorted(os.listdir(d)):
            if name.endswith((".cu", ".cuh", ".h")):
                h.update(name.encode())
                h.update(open(os.path.join(d, name), "rb").read())
    h.update(" ".join(FLAGS).encode())
    return h.hexdigest()


def _compile(job):
    src, obj, extra = job
    cmd = [NVCC] + FLAGS + extra + ["-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJDIR, exist_ok=True)
    stamp = os.path.join(OBJDIR, "digest.txt")
    digest = _source_digest()
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read() == digest:
        return LIB
    jobs = []
    for name in ("api.cu", "kernels.cu", "fft_registry.cu"):
        jobs.append((os.path.join(CSRC, name), os.path.join(OBJDIR, name[:-3] + ".o"), []))
    for m in fft_sizes():
        jobs.append((os.path.join(CSRC, "fft_inst.cu"), os.path.join(OBJDIR, "fft_%d.o" % m),
                     ["-DMBS_FFT_SIZE=%d" % m]))
    with concurrent.futures.ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        objs = list(ex.map(_compile, jobs))
    cmd = [NVCC, "-shared", "-o", LIB] + objs + ["-Xcompiler", "-fPIC", "-lcudart"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    with open(stamp, "w") as f:
        f.write(digest)
    if verbose:
        print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
