"""Writes the stored expected values under tests/golden/ that come from the ORACLE.

Calls only oracle/ (never the CUDA path).  Run from the repo root:
    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle as o  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))


def main():
    W = o.build_tensor_ewald(8)
    np.savetxt(os.path.join(HERE, "w_L8_oracle.txt"), W.reshape(4 * 8, 8), fmt="%.17e",
               header="oracle.build_tensor_ewald(8): W[c][rho_y][rho_x], c = xx, xy, yy, zz; 32 rows of 8")


if __name__ == "__main__":
    main()
