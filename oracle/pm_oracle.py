"""Oracle of HACC's long-range (particle-mesh) force.  TEST INFRASTRUCTURE ONLY: only tests/ may
import this; it shares nothing with paper_1410_2805_b200/csrc.

PAPER.md:124-159 (section 2.3), plain numpy in FP64, every step in the paper's order:

  1. "CIC mass deposition": rho(g) = sum_p m_p W(x_p - g) / Delta^3, W the product of the three
     1-D triangles max(0, 1 - |d|/Delta), periodic.
  2. one forward FFT of rho.
  3. "The 'Poisson-solve' in the HACC code is the composition of all the kernels above in one
     single Fourier transform": for every component i
         a_i(k) = -D_i(k) * 4 pi G6(k) * S(k) * rho(k)                         (G = 1)
     with the sixth-order influence function G6 of Eq. 5, the sinc-Gaussian
     filter S of Eq. 6 (sigma = 0.8 grid cells, n_s = 3) and the fourth-order
     Super-Lanczos spectral derivative of Eq. 7.
  4. "each component of the field gradient requires an independent FFT": three
     inverse FFTs.
  5. "CIC ... force interpolation" with the same W.

Readings (S25-S28): theta_i = 2 pi k_i Delta / L is the argument of every
cosine and sine; Eq. 6's vector expression is the product over the three dimensions of
[(2/theta_i) sin(theta_i/2)]^n_s, its Gaussian exp(-|theta|^2 sigma^2 / 4) with sigma in grid
cells; Eq. 7 (whose exponent lost its i in PAPER.md) is the multiplier
D(theta) = i [ (4/3) sin(theta) - (1/6) sin(2 theta) ] / Delta; the k = 0 mode is dropped (mean
density exerts no force); a = -grad phi, laplace phi = 4 pi rho.

Pins (tests/test_pm_oracle.py): the orientation-averaged force between two particles equals
the paper's own fit Eq. 8 (oracle_fgrid_eq8, written from PAPER.md:179 independently of this
file) to a few parts in a thousand of its peak, approaches 1/r^2 beyond the matching scale of
three cells (Fig. 3), momentum is conserved to round-off, a lattice feels no force, and
PM + short-range force closes to Newton's 1/r^2 below the matching scale.
"""
from __future__ import annotations

import numpy as np


def _cic(pos_cells):
    """Lower grid index and the two 1-D weights per dimension: (i0 (n,3), w (2, n, 3))."""
    i0 = np.floor(pos_cells).astype(np.int64)
    d = pos_cells - i0
    return i0, np.stack([1.0 - d, d])


def influence_g6(theta_x, theta_y, theta_z, delta):
    """Eq. 5.  theta_i = 2 pi k_i Delta / L.  Zero where the bracket vanishes."""
    c = lambda m: np.cos(m * theta_x) + np.cos(m * theta_y) + np.cos(m * theta_z)
    den = c(1) - (5.0 / 64.0) * c(2) + (1.0 / 1024.0) * c(4) - 2835.0 / 1024.0
    g = np.zeros_like(den)
    ok = np.abs(den) > 1e-14
    g[ok] = (45.0 / 128.0) * delta * delta / den[ok]
    return g


def filter_s(theta_x, theta_y, theta_z, sigma, ns):
    """Eq. 6."""
    def sinc(t):
        out = np.ones_like(t)
        m = np.abs(t) > 1e-12
        out[m] = (2.0 / t[m]) * np.sin(t[m] / 2.0)
        return out
    t2 = theta_x ** 2 + theta_y ** 2 + theta_z ** 2
    return np.exp(-t2 * sigma * sigma / 4.0) * (sinc(theta_x) * sinc(theta_y) * sinc(theta_z)) ** ns


def lanczos_d(theta, delta):
    """Eq. 7: multiplier of the fourth-order Super-Lanczos derivative."""
    return 1j * ((4.0 / 3.0) * np.sin(theta) - (1.0 / 6.0) * np.sin(2.0 * theta)) / delta


def pm_accel(x, y, z, m, box_l, ng, sigma=0.8, ns=3):
    """Long-range acceleration at the particles: dict(ax, ay, az) in FP64."""
    n = len(x)
    delta = float(box_l) / ng
    pos = np.stack([np.asarray(x, np.float64), np.asarray(y, np.float64),
                    np.asarray(z, np.float64)], 1) / delta
    mass = np.ones(n) if m is None else np.asarray(m, np.float64)
    i0, w = _cic(pos)
    rho = np.zeros((ng, ng, ng))
    for a in (0, 1):
        for b in (0, 1):
            for c in (0, 1):
                np.add.at(rho, ((i0[:, 0] + a) % ng, (i0[:, 1] + b) % ng, (i0[:, 2] + c) % ng),
                          mass * w[a, :, 0] * w[b, :, 1] * w[c, :, 2] / delta ** 3)
    rho_k = np.fft.fftn(rho)
    t1 = 2.0 * np.pi * np.fft.fftfreq(ng)
    tx, ty, tz = np.meshgrid(t1, t1, t1, indexing="ij")
    phi_k = 4.0 * np.pi * influence_g6(tx, ty, tz, delta) * filter_s(tx, ty, tz, sigma, ns) * rho_k
    out = {}
    for name, t in (("ax", tx), ("ay", ty), ("az", tz)):
        g = np.real(np.fft.ifftn(-lanczos_d(t, delta) * phi_k))
        v = np.zeros(n)
        for a in (0, 1):
            for b in (0, 1):
                for c in (0, 1):
                    v += w[a, :, 0] * w[b, :, 1] * w[c, :, 2] * \
                        g[(i0[:, 0] + a) % ng, (i0[:, 1] + b) % ng, (i0[:, 2] + c) % ng]
        out[name] = v
    return out
