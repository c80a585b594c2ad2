"""Build oracle/libtnlm_oracle.so from tnlm_oracle.c and oracle/libtnlmr_oracle.so from tnlmr_oracle.c with gcc
(C11, OpenMP, -O2, no fast-math).

Test infrastructure only.  ``python oracle/build_oracle.py`` or ``build()`` from Python.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "tnlm_oracle.c")
LIB = os.path.join(HERE, "libtnlm_oracle.so")


SRC_R = os.path.join(HERE, "tnlmr_oracle.c")
LIB_R = os.path.join(HERE, "libtnlmr_oracle.so")


def _build_one(src: str, lib: str, force: bool) -> str:
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= os.path.getmtime(src):
        return lib
    tmp = lib + f".tmp{os.getpid()}"
    cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-fno-fast-math", "-ffp-contract=off", src, "-o", tmp, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, lib)
    return lib


def build(force: bool = False) -> str:
    """The TNLM-E oracle (returns its path); also keeps the TNLM-R oracle up to date."""
    _build_one(SRC_R, LIB_R, force)
    return _build_one(SRC, LIB, force)


def build_r(force: bool = False) -> str:
    """The TNLM-R oracle (projector pair + CGLS)."""
    return _build_one(SRC_R, LIB_R, force)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
