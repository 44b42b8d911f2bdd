"""Build librealfast_b200.so in-tree with nvcc for sm_100a (no JIT cache, no torch extension).

Whether a build is needed is decided by CONTENT, not by file times: the SHA-256 of every source, header, this
file and the nvcc command line is stored beside the library (``librealfast_b200.so.srchash``) when it is linked.
A library that travels to another machine with its sources (built ``*.so`` files are kept out of the history but
do ship to the GPU box) is reused only if that hash still matches the sources it arrived with; otherwise nvcc
runs there.  ``build()`` reports which of the two happened (``last_action``), so a log shows it.
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librealfast_b200.so")
STAMP = LIB + ".srchash"
SOURCES = ["rf_api.cu", "rf_tables.cu", "rf_search.cu", "rf_prep.cu", "rf_cutout.cu", "rf_static.cu"]
HEADERS = ["rf_internal.h", "rf_fft.cuh", "rf_kernels.cuh", "rf_tree_kernels.cuh",
           os.path.join("..", "..", "include", "realfast.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-O2", "-DNDEBUG",
]
last_action = "none"     # "compiled" | "reused" after build()


def _nvcc() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def _extra_flags() -> list:
    return os.environ.get("RF_NVCC_EXTRA", "").split()


def source_hash() -> str:
    """SHA-256 over the contents of every dependency and the compile flags."""
    h = hashlib.sha256()
    for name in SOURCES + HEADERS:
        with open(os.path.join(CSRC, name), "rb") as fh:
            h.update(name.encode() + b"\0" + fh.read() + b"\0")
    with open(os.path.abspath(__file__), "rb") as fh:
        h.update(fh.read())
    h.update(" ".join(NVCC_FLAGS + _extra_flags()).encode())
    return h.hexdigest()


def needs_build() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(STAMP):
        return True
    with open(STAMP) as fh:
        return fh.read().strip() != source_hash()


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every CUDA source into one shared library; returns its path."""
    global last_action
    if not force and not needs_build():
        last_action = "reused"
        return LIB
    want = source_hash()
    if os.path.exists(STAMP):
        os.remove(STAMP)
    objs = []
    procs = []
    for s in SOURCES:
        obj = os.path.join(CSRC, s.replace(".cu", ".o"))
        cmd = [_nvcc(), *NVCC_FLAGS, *_extra_flags(), "-c", os.path.join(CSRC, s), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for cmd, pr in procs:
        out, _ = pr.communicate()
        if verbose or pr.returncode:
            sys.stderr.write(out)
        if pr.returncode:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    link = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB, *objs]
    subprocess.run(link, check=True)
    with open(STAMP, "w") as fh:
        fh.write(want + "\n")
    last_action = "compiled"
    return LIB


def describe() -> str:
    """One line for logs: what build() did and which sources the library corresponds to."""
    return f"{LIB}: {last_action} (source hash {source_hash()[:16]})"


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="-v" in sys.argv)
    print(describe())
