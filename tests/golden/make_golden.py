"""Write tests/golden/poly_default.txt.  Calls only oracle/ (never the CUDA path)."""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle.fit_poly import fit_default_poly  # noqa: E402


def main():
    c, err = fit_default_poly()
    with open(os.path.join(HERE, "poly_default.txt"), "w") as f:
        f.write("# Default P(s) = sum c_k s^k: least-squares fit of PAPER.md Eq. 8 (line 179)\n"
                "# by DESIGN.md reading S3; written by tests/golden/make_golden.py\n"
                "# k  double  float32\n")
        for k, v in enumerate(c):
            f.write(f"{k} {v:.12e} {float(np.float32(v))!r}\n")
        f.write(f"# max |r P(r^2) - f_grid(r)| on (0,3) = {err:.4e}\n")


if __name__ == "__main__":
    main()
