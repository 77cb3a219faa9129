"""Compile and run the FP64-pipe microbenchmark (csrc/ubench_fp64_pipe.cu) on cuda:0.

    python -m paper_2602_20787_b200.ubench

Prints a markdown table (profiles/r2_fp64_pipe_microbench.md is its output).  Design evidence, not part of the
library: it measures what an FP64 instruction costs on this GPU depending on its operand forms and on what is
issued beside it, which is what the pair kernels' instruction selection follows.
"""
from __future__ import annotations

import os
import subprocess
import sys
import tempfile

from .build import CSRC, nvcc


def main() -> int:
    src = os.path.join(CSRC, "ubench_fp64_pipe.cu")
    with tempfile.TemporaryDirectory() as d:
        exe = os.path.join(d, "ubench_fp64_pipe")
        subprocess.run([nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", src, "-o", exe],
                       check=True)
        return subprocess.run([exe]).returncode


if __name__ == "__main__":
    sys.exit(main())
