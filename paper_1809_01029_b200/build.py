"""Builds libpyjac_b200.so in-tree with nvcc for sm_100a.  `python -m paper_1809_01029_b200.build`."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpyjac_b200.so")
SOURCES = ["pyjac_host.cpp", "pyjac_kernels.cu", "pyjac_capi.cu"]
DEPS = SOURCES + ["pyjac_internal.h"]


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    files = [os.path.join(CSRC, f) for f in DEPS] + [os.path.join(ROOT, "include", "pyjac.h")]
    return any(os.path.getmtime(f) > t for f in files)


def build(force=False, verbose=False, out=None, defines=()):
    """out / defines: build a variant (e.g. defines=['PYJAC_NT=512']) to another path (tuning experiments)."""
    if out is None and not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(ROOT, "include"), "-I", CSRC,
           "-o", out or LIB] + ["-D" + d for d in defines] + [os.path.join(CSRC, f) for f in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas"); cmd.insert(2, "-v")
    subprocess.run(cmd, check=True)
    return out or LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
