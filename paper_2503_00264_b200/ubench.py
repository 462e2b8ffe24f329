"""Builds and runs csrc/ubench_fp64.cu: the DFMA / DMMA throughput of the FP64 pipe on this GPU.

    python -m paper_2503_00264_b200.ubench

The output is the denominator of bench.py's "alu" roofline and the evidence for the DMMA decision.
Needs a CUDA device; nothing here is on the product path."""
from __future__ import annotations

import subprocess
import sys
import tempfile
from pathlib import Path

from .build import _nvcc

SRC = Path(__file__).resolve().parent / "csrc" / "ubench_fp64.cu"


def main() -> int:
    with tempfile.TemporaryDirectory() as d:
        exe = Path(d) / "ubench_fp64"
        subprocess.run([_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", str(exe), str(SRC)], check=True)
        return subprocess.run([str(exe)]).returncode


if __name__ == "__main__":
    sys.exit(main())
