"""Derive the default 5th-order polynomial P(s) from PAPER.md Eq. 8.  TEST INFRASTRUCTURE.

The paper says f_grid(s) in Eq. 12 "is a 5-th order polynomial in s" and
that the short matching scale "enables the use of a fifth-order polynomial approximation"
(PAPER.md:189), but it never prints the coefficients.  DESIGN.md readings S1-S4:

* the coefficients are an INPUT of the path; the default set is derived from Eq. 8 here;
* Eq. 8 is a force MAGNITUDE (-> 1/r^2) while Eq. 12's term sits beside (s+eps)^(-3/2)
  (-> 1/r^3) and multiplies the separation vector, so P(s) ~ f_grid(sqrt s)/sqrt s (S2);
* fit (S3): least squares of r*P(r^2) against Eq. 8's f_grid(r) at 4096 Chebyshev-Gauss
  nodes r_k = 1.5*(1 + cos(pi*(k+1/2)/4096)) in (0, 3), columns scaled to unit max, FP64
  lstsq; degree 5 in s (S4).

`python -m oracle.fit_poly` prints the six coefficients in double and rounded to float32;
the float32 values are what paper_1410_2805_b200/workloads.py stores as DEFAULT_POLY and
what tests/golden/poly_default.txt records.
"""
from __future__ import annotations

import numpy as np

from . import sr_oracle

R_S = 3.0  # force-matching scale, PAPER.md:132-136 (Fig. 3): 3 grid cells
N_NODES = 4096


def fit_default_poly():
    k = np.arange(N_NODES)
    r = 0.5 * R_S * (1.0 + np.cos(np.pi * (k + 0.5) / N_NODES))
    target = sr_oracle.fgrid_eq8(r)
    s = r * r
    cols = np.stack([r * s ** p for p in range(6)], axis=1)
    scale = np.abs(cols).max(axis=0)
    sol, *_ = np.linalg.lstsq(cols / scale, target, rcond=None)
    c = sol / scale
    resid = cols @ c - target
    return c, float(np.abs(resid).max())


def main():
    c, err = fit_default_poly()
    print("double :", ", ".join(f"{v:.10e}" for v in c))
    print("float32:", ", ".join(repr(float(np.float32(v))) for v in c))
    print(f"max |r*P(r^2) - f_grid(r)| on (0,3): {err:.3e}")


if __name__ == "__main__":
    main()
