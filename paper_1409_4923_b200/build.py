"""Builds the C-ABI library (csrc/ -> libbm.so) in-tree with nvcc for sm_100a only."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libbm.so")


def build(verbose=False, jobs=None):
    """make -C csrc (nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo).  Cross-compiles without a GPU."""
    jobs = jobs or max(1, min(16, os.cpu_count() or 1))
    r = subprocess.run(["make", "-C", CSRC, f"-j{jobs}"], capture_output=not verbose, text=True)
    if r.returncode != 0:
        raise RuntimeError("building libbm.so failed:\n" + (r.stdout or "") + (r.stderr or ""))
    if not os.path.exists(LIB):
        raise RuntimeError("make succeeded but libbm.so is missing")
    return LIB


if __name__ == "__main__":
    print(build(verbose=True))
