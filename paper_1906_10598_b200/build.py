"""In-tree nvcc build of ``libpt.so`` for sm_100a (B200).

``python -m paper_1906_10598_b200.build`` or ``build()``; nvcc cross-compiles without a GPU.  The built
library stays next to this file (git-ignored, but it travels to the GPU box with the tree).
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpt.so")
STAMP = os.path.join(HERE, ".libpt.stamp")
SOURCES = ["pt_api.cu", "pt_doppler.cu", "pt_acquire.cu", "pt_retry.cu", "pt_noalloc.cu"]
# bench-only micro-benchmarks (measured FFMA / MUFU stream rates): their own library, not part of the product ABI
PROBE_LIB = os.path.join(HERE, "libpt_probe.so")
PROBE_STAMP = os.path.join(HERE, ".libpt_probe.stamp")
PROBE_SOURCES = ["pt_probe.cu"]
NVCC_FLAGS = [
    "-O3",
    "-std=c++17",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo",
    "-Xcompiler", "-fPIC",
    "-Xcompiler", "-fvisibility=hidden",
    "--shared",
]


def _nvcc() -> str:
    cand = os.environ.get("NVCC") or "/usr/local/cuda/bin/nvcc"
    return cand if os.path.exists(cand) else "nvcc"


def _fingerprint() -> str:
    h = hashlib.sha256()
    root = os.path.dirname(HERE)
    files = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC))] + [os.path.join(root, "include", "pt.h")]
    for f in files:
        with open(f, "rb") as fh:
            h.update(f.encode())
            h.update(fh.read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()


def _build(lib: str, stamp: str, sources, force: bool, verbose: bool, extra_flags) -> str:
    fp = _fingerprint()
    if not force and not extra_flags and os.path.exists(lib) and os.path.exists(stamp):
        with open(stamp) as fh:
            if fh.read().strip() == fp:
                return lib
    tmp = lib + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + list(extra_flags) + ["-o", tmp] + [os.path.join(CSRC, s) for s in sources]
    if verbose:
        print(" ".join(cmd), file=sys.stderr)
    subprocess.run(cmd, check=True)
    os.replace(tmp, lib)
    with open(stamp, "w") as fh:
        fh.write(fp)
    return lib


def build(force: bool = False, verbose: bool = False, extra_flags=()) -> str:
    """Compile csrc/*.cu into libpt.so; a no-op when sources and flags are unchanged (fingerprint stamp)."""
    return _build(LIB, STAMP, SOURCES, force, verbose, extra_flags)


def build_probe(force: bool = False, verbose: bool = False) -> str:
    """Compile the bench-only peak probes into libpt_probe.so."""
    return _build(PROBE_LIB, PROBE_STAMP, PROBE_SOURCES, force, verbose, ())


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True,
                extra_flags=["-Xptxas", "-v"] if "--ptxas-v" in sys.argv else ()))
    print(build_probe(force="--force" in sys.argv, verbose=True))
