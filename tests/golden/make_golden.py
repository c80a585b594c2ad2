"""Writes tests/golden/tiny_enhance.txt by calling ONLY the CPU oracle (never the CUDA path).

The paper prints no worked numeric example of Eq. 3 / Eq. 8, so this
fixture is not a paper value: it freezes the pinned oracle's output on a tiny seeded stack so
that any later change of the oracle's arithmetic shows up in review (tests/test_golden.py).

Run from the repo root:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import tnlm_oracle as O            # noqa: E402
from tnlm_inputs import CONFIGS, make_stack    # noqa: E402

CFG = CONFIGS["config1"].scaled(n_phase=3, nz=4, ny=6, nx=7)


def main():
    g = make_stack(CFG)
    f = O.enhance(g, CFG.patch_radius, CFG.search_radius, np.float32(CFG.h), np.float32(CFG.mu), 2)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_enhance.txt")
    with open(path, "w") as fh:
        fh.write("# TNLM-E (PAPER.md:204-211, Eq. 8/9) by oracle/tnlm_oracle.c on config1 scaled to "
                 "3x4x6x7, d=1 M=1 h=0.1 mu=1.0, 2 iterations, seed 0\n")
        fh.write("# written by tests/golden/make_golden.py; columns: flat_index g f_out (float32, %.9g)\n")
        for i, (a, b) in enumerate(zip(g.reshape(-1), f.reshape(-1))):
            fh.write(f"{i} {a:.9g} {b:.9g}\n")
    print(path)


if __name__ == "__main__":
    main()
