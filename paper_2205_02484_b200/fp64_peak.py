"""Builds and runs csrc/fp64_peak.cu, the DFMA micro-benchmark behind the "alu" roofline.

    python -m paper_2205_02484_b200.fp64_peak

Needs a GPU.  Prints the program's table (cycles per warp-level DFMA per SM sub-partition and device-wide rate for
ILP x resident-warps combinations).  A measurement aid: nothing in the library or bench.py depends on it.
"""
import os
import subprocess
import sys
import tempfile

HERE = os.path.dirname(os.path.abspath(__file__))


def main() -> int:
    src = os.path.join(HERE, "csrc", "fp64_peak.cu")
    with tempfile.TemporaryDirectory() as tmp:
        exe = os.path.join(tmp, "fp64_peak")
        subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", exe, src], check=True)
        return subprocess.run([exe]).returncode


if __name__ == "__main__":
    sys.exit(main())
