"""Build the C-ABI CUDA library paper_2605_03563_b200/libpoisson_b200.so for sm_100a (in-tree, nvcc).

    python -m paper_2605_03563_b200.build [--force] [--verbose]
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpoisson_b200.so")
OBJ = os.path.join(HERE, "build")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++20", "-fmad=false", "-lineinfo",
         "--extended-lambda", "-Xcompiler", "-fPIC"]


# Files whose results are compared with the oracle at a tolerance (1e-12 for the multipole sums), not bit for bit: the
# compiler may contract a * b + c into fma there.  Everything else keeps -fmad=false (explicit fma only, C1b).  C++20: `requires` in plane.cuh.
CONTRACT_OK = {"k_multipole.cu"}


def sources():
    return sorted(f for f in os.listdir(CSRC) if f.endswith(".cu"))


def _deps_mtime():
    files = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "poisson.h"),
                                                                  os.path.abspath(__file__)]
    return max(os.path.getmtime(f) for f in files)


def needs_build():
    return not os.path.exists(LIB) or os.path.getmtime(LIB) < _deps_mtime()


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []

    hdr_mtime = max(os.path.getmtime(os.path.join(CSRC, f)) for f in os.listdir(CSRC) if not f.endswith(".cu"))
    hdr_mtime = max(hdr_mtime, os.path.getmtime(os.path.join(HERE, "..", "include", "poisson.h")),
                    os.path.getmtime(os.path.abspath(__file__)))

    def compile_one(src):
        obj = os.path.join(OBJ, src[:-3] + ".o")
        if not force and not verbose and os.path.exists(obj) and \
                os.path.getmtime(obj) > max(hdr_mtime, os.path.getmtime(os.path.join(CSRC, src))):
            return obj  # up to date
        flags = [f for f in FLAGS if not (src in CONTRACT_OK and f == "-fmad=false")]
        cmd = [NVCC] + flags + extra + ["-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, r.stdout, r.stderr))
        if verbose:
            print(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=8) as ex:
        objs = list(ex.map(compile_one, sources()))
    subprocess.check_call([NVCC, "-shared", "-o", LIB] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
