"""Builds libpyjac_b200.so in-tree with nvcc for sm_100a.  `python -m paper_1809_01029_b200.build [--force] [-v]`.

Every source is compiled to an object file under csrc/build/ (git-ignored; recompiled only when it or a header is
newer) and the objects are linked into the shared library."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libpyjac_b200.so")
SOURCES = ["pyjac_host.cpp", "pyjac_plan.cpp", "pyjac_kernels.cu", "pyjac_jacobian.cu", "pyjac_jacobian_ls1.cu", "pyjac_jacobian_ls2.cu",
           "pyjac_jacobian_ls4.cu", "pyjac_capi.cu", "pyjac_peaks.cu"]
HEADERS = [os.path.join(CSRC, "pyjac_internal.h"), os.path.join(CSRC, "pyjac_jacobian.cuh"), os.path.join(CSRC, "pyjac_jacobian_launch.cuh"), os.path.join(CSRC, "pyjac_math.cuh"),
           os.path.join(ROOT, "include", "pyjac.h")]


def _newer(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.exists(f) and os.path.getmtime(f) > t for f in deps)


def build(force=False, verbose=False):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    flags = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC",
             "-I", os.path.join(ROOT, "include"), "-I", CSRC]
    if verbose:
        flags += ["-Xptxas", "-v"]
    sources = [s for s in SOURCES if os.path.exists(os.path.join(CSRC, s))]
    objs = [os.path.join(OBJ, s.rsplit(".", 1)[0] + ".o") for s in sources]
    todo = [(s, o) for s, o in zip(sources, objs) if force or _newer(o, [os.path.join(CSRC, s)] + HEADERS)]

    def compile_one(so):
        subprocess.run([nvcc] + flags + ["-c", os.path.join(CSRC, so[0]), "-o", so[1]], check=True)

    with ThreadPoolExecutor(max_workers=max(1, min(len(todo), os.cpu_count() or 1))) as ex:
        list(ex.map(compile_one, todo))
    if todo or _newer(LIB, objs):
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
