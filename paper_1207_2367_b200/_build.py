"""In-tree build of libnb.so: nvcc, sm_100a only, no torch headers, no JIT cache.

`python -m paper_1207_2367_b200._build` (or __graft_entry__.build()) compiles every .cu under
csrc/ to an object and links them into paper_1207_2367_b200/libnb.so.  nvcc cross-compiles
without a GPU.  The shared library travels to the GPU box with the source tree.
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libnb.so")
OBJDIR = os.path.join(HERE, "build")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]
# The evaluation kernels are compiled with ptxas -O1: its scheduler keeps close to the statement order of the
# pair body, which is arranged so that FP64 instructions with three register sources find one of them in the
# operand-reuse cache (csrc/nb_force_dev.cuh); -O3 interleaves the unrolled pairs for
# latency and loses that (measured on B200: 121.9 cycles per warp-pair at -O3, 118.7 at -O1 with the round-1 body).
PTXAS_LEVEL = {"nb_force.cu": "-O1", "nb_static.cu": "-O1"}


def sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cu"))


def _deps_mtime():
    files = sources() + [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cuh")]
    files.append(os.path.join(os.path.dirname(HERE), "include", "nb.h"))
    return max(os.path.getmtime(f) for f in files)


def _compile(src: str) -> tuple[str, str]:
    obj = os.path.join(OBJDIR, os.path.basename(src)[:-3] + ".o")
    level = PTXAS_LEVEL.get(os.path.basename(src))
    cmd = [NVCC, *ARCH, *FLAGS, *(["-Xptxas", level] if level else []), "-c", src, "-o", obj]
    p = subprocess.run(cmd, capture_output=True, text=True)
    if p.returncode != 0:
        raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), p.stdout, p.stderr))
    return obj, p.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _deps_mtime():
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    with cf.ThreadPoolExecutor(max_workers=4) as ex:
        res = list(ex.map(_compile, sources()))
    if verbose:
        for _, log in res:
            sys.stderr.write(log)
    cmd = [NVCC, *ARCH, "-shared", "-o", LIB, *[o for o, _ in res]]
    p = subprocess.run(cmd, capture_output=True, text=True)
    if p.returncode != 0:
        raise RuntimeError("link failed: %s\n%s\n%s" % (" ".join(cmd), p.stdout, p.stderr))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
