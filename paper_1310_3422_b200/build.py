"""In-tree build of libge.so for sm_100a (nvcc cross-compiles without a GPU).

    python -m paper_1310_3422_b200.build [--force] [--verbose]

The shared object lands next to this file (paper_1310_3422_b200/lib/libge.so); it is
git-ignored but travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "lib", "libge.so")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-fmad=false",            # every fma in the kernels is written out; no implicit contraction
    "-Xcompiler", "-fPIC",
]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static", "-ldl"]
OBJ = os.path.join(_HERE, "lib", "obj")


def _sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers():
    return glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(INCLUDE, "*.h"))


def _deps():
    return _sources() + _headers()


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    """Every .cu of csrc/ is a translation unit of its own (the kernel families compile in parallel); objects are
    cached under lib/obj and recompiled when the source, any header or the flags changed."""
    nvcc = os.environ.get("NVCC", "nvcc")
    extra = os.environ.get("GE_NVCC_EXTRA", "").split()        # e.g. -DGE_STRIP_MINB_F32=4 for tuning sweeps
    libtag = LIB + ".flags"
    same_flags = os.path.exists(libtag) and open(libtag).read() == " ".join(NVCC_FLAGS + extra)
    if not force and same_flags and not needs_build():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    hdr_time = max(os.path.getmtime(f) for f in _headers())
    flags_tag = " ".join(NVCC_FLAGS + extra)
    jobs, objs = [], []
    for src in _sources():
        obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
        tag = obj + ".flags"
        objs.append(obj)
        fresh = (not force and os.path.exists(obj) and os.path.exists(tag) and open(tag).read() == flags_tag
                 and os.path.getmtime(obj) > max(hdr_time, os.path.getmtime(src)))
        if fresh:
            continue
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-I", INCLUDE, "-c", "-o", obj, src]
        jobs.append((src, tag, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for src, tag, proc in jobs:
        out, _ = proc.communicate()
        if verbose or proc.returncode != 0:
            sys.stderr.write(out)
        if proc.returncode != 0:
            failed = True
        else:
            with open(tag, "w") as f:
                f.write(flags_tag)
    if failed:
        raise RuntimeError("nvcc failed building libge.so")
    tmp = LIB + ".tmp.%d" % os.getpid()
    proc = subprocess.run([nvcc] + LINK_FLAGS + ["-o", tmp] + objs, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if proc.returncode != 0:
        sys.stderr.write(proc.stdout)
        if os.path.exists(tmp):
            os.remove(tmp)
        raise RuntimeError("nvcc failed linking libge.so (exit %d)" % proc.returncode)
    os.replace(tmp, LIB)
    with open(libtag, "w") as f:
        f.write(flags_tag)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
