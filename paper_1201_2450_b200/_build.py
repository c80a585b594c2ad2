"""Build paper_1201_2450_b200/libtnlm.so in-tree with nvcc for sm_100a (no torch headers involved)."""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtnlm.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-shared", "--use_fast_math", "-Xptxas", "-v", "-cudart", "static"]
# --use_fast_math applies to the whole library (flush-to-zero, approximate division and sqrt, also in the
# metric kernels), "Arithmetic flags", states what depends on it.


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _newest_src():
    files = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "tnlm.h")]
    return max(os.path.getmtime(f) for f in files)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_src():
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = [NVCC] + FLAGS + sources() + ["-o", tmp]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libtnlm.so")
    os.replace(tmp, LIB)
    with open(os.path.join(HERE, "build_ptxas.log"), "w") as fh:
        log = (" ".join(cmd) + "\n" + res.stdout + res.stderr).replace(tmp, LIB).replace(HERE + os.sep, "")
        fh.write("".join(ln for ln in log.splitlines(True) if "Compile time" not in ln))   # registers and spills, no timings
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
