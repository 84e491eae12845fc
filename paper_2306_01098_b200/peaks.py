"""`python -m paper_2306_01098_b200.peaks` -- build and run csrc/peaks.cu: the measured read-only / copy HBM
bandwidth and fp32 / fp64 FMA peaks of this GPU (roofline context; SURVEY.md 8(d) asks for all denominators)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
EXE = os.path.join(HERE, "build", "peaks")


def build() -> str:
    os.makedirs(os.path.dirname(EXE), exist_ok=True)
    src = os.path.join(HERE, "csrc", "peaks.cu")
    if not os.path.exists(EXE) or os.path.getmtime(EXE) < os.path.getmtime(src):
        subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", EXE, src], check=True)
    return EXE


if __name__ == "__main__":
    sys.exit(subprocess.run([build()]).returncode)
