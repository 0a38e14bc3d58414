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
    body = text.split("#define MBS_FOR_EACH_FFT_SIZE(X)")[-1].split("#endif")[0]
    return [int(m) for m in re.findall(r"X\((\d+)\)", body)]


_INC = re.compile(r'^\s*#\s*include\s*"([^"]+)"', re.M)


def _deps(path, seen=None):
    """The file and every header it includes with quotes, recursively (paths relative to the including file)."""
    seen = set() if seen is None else seen
    path = os.path.normpath(path)
    if path in seen or not os.path.exists(path):
        return seen
    seen.add(path)
    for inc in _INC.findall(open(path).read()):
        _deps(os.path.join(os.path.dirname(path), inc), seen)
    return seen


def _job_digest(src, extra):
    h = hashlib.sha256()
    for dep in sorted(_deps(src)):
        h.update(os.path.relpath(dep, ROOT).encode())
        h.update(open(dep, "rb").read())
    h.update(" ".join(FLAGS + extra).encode())
    return h.hexdigest()


def _compile(job):
    src, obj, extra = job
    cmd = [NVCC] + FLAGS + extra + ["-c", src, "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return obj


def build(force: bool = False, verbose: bool = False, sizes=None) -> str:
    """Compiles what changed (one digest per object over the source, the headers it includes and the flags) and links.
    `sizes` (kernel development only: `--sizes 256,512`) links a library that knows just those subdomain lengths."""
    os.makedirs(OBJDIR, exist_ok=True)
    jobs = []
    for name in ("api.cu", "kernels.cu", "refine_f64.cu"):
        jobs.append((os.path.join(CSRC, name), os.path.join(OBJDIR, name[:-3] + ".o"), []))
    if sizes:
        tag = "_".join(str(m) for m in sizes)
        jobs.append((os.path.join(CSRC, "fft_registry.cu"), os.path.join(OBJDIR, "fft_registry_dev_%s.o" % tag),
                     ["-DMBS_DEV_SIZES(X)=" + " ".join("X(%d)" % m for m in sizes)]))
    else:
        jobs.append((os.path.join(CSRC, "fft_registry.cu"), os.path.join(OBJDIR, "fft_registry.o"), []))
    for m in (sizes or fft_sizes()):
        jobs.append((os.path.join(CSRC, "fft_inst.cu"), os.path.join(OBJDIR, "fft_%d.o" % m),
                     ["-DMBS_FFT_SIZE=%d" % m]))
    stale, digests = [], {}
    for src, obj, extra in jobs:
        digests[obj] = _job_digest(src, extra)
        stamp = obj + ".digest"
        if force or not os.path.exists(obj) or not os.path.exists(stamp) or open(stamp).read() != digests[obj]:
            stale.append((src, obj, extra))
    marker = os.path.join(OBJDIR, "linked.txt")
    linked = " ".join(obj for _, obj, _ in jobs)
    if not stale and os.path.exists(LIB) and os.path.exists(marker) and open(marker).read() == linked:
        return LIB
    with concurrent.futures.ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
        list(ex.map(_compile, stale))
    for _, obj, _ in stale:
        with open(obj + ".digest", "w") as f:
            f.write(digests[obj])
    objs = [obj for _, obj, _ in jobs]
    cmd = [NVCC, "-shared", "-o", LIB] + objs + ["-Xcompiler", "-fPIC", "-lcudart"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    with open(marker, "w") as f:
        f.write(linked)
    if verbose:
        print("built %s (%d of %d objects recompiled)" % (LIB, len(stale), len(jobs)))
    return LIB


if __name__ == "__main__":
    _sizes = None
    if "--sizes" in sys.argv:
        _sizes = [int(v) for v in sys.argv[sys.argv.index("--sizes") + 1].split(",")]
    build(force="--force" in sys.argv, verbose=True, sizes=_sizes)
