"""Build libmc.so (the C-ABI CUDA library, include/mc.h) in-tree with nvcc for sm_100a.

    python -m paper_2607_02954_b200.build [--force]

The .so is git-ignored but travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmc.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
         "-Xptxas", "-v"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return (sources() + glob.glob(os.path.join(CSRC, "*.cuh"))
            + [os.path.join(os.path.dirname(HERE), "include", "mc.h"), os.path.abspath(__file__)])


def csrc_sha() -> str:
    """Hash of the CUDA sources (names and contents of csrc/*.cu, *.cuh): ties a built library and an
    ncu capture to the sources they were made from."""
    import hashlib
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh"))):
        h.update(os.path.basename(f).encode())
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


SHA_FILE = os.path.join(HERE, "libmc.csrc_sha")   # written beside libmc.so by build()


def built_sha() -> str:
    try:
        with open(SHA_FILE) as fh:
            return fh.read().strip()
    except OSError:
        return ""


def build(force: bool = False, verbose: bool = False) -> str:
    if (not force and os.path.exists(LIB) and built_sha() == csrc_sha()
            and os.path.getmtime(LIB) >= max(os.path.getmtime(p) for p in _deps())):
        return LIB
    cmd = [NVCC] + FLAGS + sources() + ["-o", LIB]
    r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libmc.so")
    with open(os.path.join(HERE, "libmc.ptxas.log"), "w") as fh:
        fh.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    with open(SHA_FILE, "w") as fh:
        fh.write(csrc_sha() + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
