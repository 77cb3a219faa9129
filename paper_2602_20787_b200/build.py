"""Build libsteps_cyl.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2602_20787_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with
the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsteps_cyl.so")
SOURCES = [os.path.join(CSRC, "steps_cyl.cu")]
SASSMIX = os.path.join(HERE, "libsteps_cyl.sassmix.json")


def _deps() -> list:
    """Everything the library is compiled from: all of csrc/ plus the public header (content-hashed)."""
    files = sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC)
                   if f.endswith((".cu", ".cuh", ".h")) and not f.startswith("ubench_"))
    return files + [os.path.join(os.path.dirname(HERE), "include", "steps_cyl.h"),
                    os.path.join(HERE, "sassmix.py")]


NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC",
              "--fmad=true", "-cudart", "static"]


def nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    raise RuntimeError("nvcc not found")


def _extra() -> list:
    return os.environ.get("STEPS_NVCC_EXTRA", "").split()


def _source_hash() -> str:
    import hashlib
    h = hashlib.sha256(" ".join(NVCC_FLAGS + _extra()).encode())
    for d in _deps():
        h.update(open(d, "rb").read())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if the library is missing or its sources changed (content hash, not mtime: the
    gpurun snapshot does not preserve mtimes)."""
    stamp = LIB + ".hash"
    want = _source_hash()
    fresh = os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read().strip() == want
    if force or not fresh:
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = [nvcc(), *NVCC_FLAGS, *_extra(), *(["-Xptxas", "-v"] if verbose else []), *SOURCES, "-o", tmp]
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
        if os.path.exists(SASSMIX):
            os.unlink(SASSMIX)
        with open(stamp, "w") as f:
            f.write(want + "\n")
    # instruction tally of the pair loops of THIS binary (bench.py's roofline numerator): the file records the
    # library's SHA-256, so a tally left behind by another build of the library is noticed and retaken
    from . import sassmix
    if not sassmix.is_current(LIB, SASSMIX):
        sassmix.write(LIB, SASSMIX)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
