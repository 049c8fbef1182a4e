"""Build librs.so (the C-ABI library of include/rs.h) in-tree with nvcc for sm_100a.

    python -m paper_1306_2953_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so lands next to this file so that it travels with the
repository snapshot to the GPU box; it is git-ignored.
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(ROOT, "include")
SO = os.path.join(HERE, "librs.so")

SOURCES = ["rs_api.cu", "rs_mesh.cu", "rs_kernels.cu", "rs_sweep.cu", "rs_blas.cu", "rs_overlap.cu", "rs_nonlocal.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-O3",
    "-shared",
]


def _deps() -> list[str]:
    d = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".h", ".cuh"))]
    d += [os.path.join(INCLUDE, f) for f in os.listdir(INCLUDE) if f.endswith(".h")]
    d.append(os.path.abspath(__file__))
    return d


def _digest() -> str:
    h = hashlib.sha256()
    for p in sorted(_deps()):
        h.update(os.path.basename(p).encode())
        h.update(open(p, "rb").read())
    return h.hexdigest()


def needs_build() -> bool:
    """True when librs.so is missing or was built from other sources (content hash, not mtime:
    the snapshot that carries the tree to the GPU box does not promise to keep mtimes)."""
    if not os.path.exists(SO) or not os.path.exists(SO + ".sha256"):
        return True
    return open(SO + ".sha256").read().strip() != _digest()


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return SO
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc, *NVCC_FLAGS, "-I", INCLUDE, "-I", CSRC, "-o", SO]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    if verbose:
        sys.stderr.write(r.stderr)
    with open(SO + ".sha256", "w") as f:
        f.write(_digest())
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
