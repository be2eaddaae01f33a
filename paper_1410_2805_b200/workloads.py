"""Seeded synthetic particle sets for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle, so it holds none of the
method's arithmetic: no force law, no cell index, no polynomial evaluation. It only
draws random particles (numpy PCG64, seed = 14102805 + config index) and names the
parameters of each config.

The paper's runs are LambdaCDM particle distributions with 32-64.5 M particles per GPU
node (section 6); those snapshots are not available, so uniform +
Plummer-halo mixtures (BASELINE.json `configs`) stand in for them.  Recipe (stated in
DESIGN.md section 4):

* background: uniform in [0, L)^3;
* halo particle counts: truncated Pareto N(>n) ~ 1/n on [n_min, n_max], drawn by
  inverse CDF until the halo budget floor(f_halo * N) is used up (last halo truncated);
* halo centres uniform; Plummer scale radius a = 0.2 * 10**u, u ~ U(0,1), i.e.
  log-uniform in [0.2, 2.0] grid units;
* Plummer radii r = a / sqrt(u**(-2/3) - 1) with u ~ U(0, u_max), u_max chosen so that
  r <= 10 a (truncation; BASELINE.json is silent on it), isotropic directions,
  periodic wrap into [0, L);
* unit masses; velocities zero (configs 0-3) or Gaussian sigma = 0.5 (config 4);
* everything sampled in float64, cast to float32, values that round up to L are set
  to 0, then one seeded random permutation of the particle order so that the first
  binning is a genuine unsorted scatter.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

BASE_SEED = 14102805

# The default polynomial P(s) = sum_k c_k s^k standing for the filtered grid force of
# PAPER.md Eq. 8 divided by r (reading S2/S3).  The paper never prints its
# coefficients; these six float32 numbers are INPUT DATA, written by
# `python -m oracle.fit_poly` (which calls only oracle/ code) and checked against that
# fitter in tests/test_oracle_pins.py.  Both the oracle and the CUDA path receive them
# as the `poly` argument.
DEFAULT_POLY = (
    0.26908568,
    -0.07422199,
    0.010907516,
    -0.0009488722,
    4.4874712e-05,
    -8.5389166e-07,
)


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config: box, mesh, mixture and step parameters."""

    index: int
    name: str
    n_side: int  # N = n_side**3 particles
    box_l: float  # periodic box length, grid units
    nc: int  # chaining-mesh cells per dimension
    f_halo: float  # fraction of particles in Plummer halos
    halo_n_min: int
    halo_n_max: int
    sigma_v: float  # Gaussian velocity sigma per component (0 = zero velocities)
    n_sub: int  # sub-cycles (config 4: 5 x [drift, bin, force+kick])
    r_max: float = 3.0
    eps: float = 0.1
    dt: float = 0.01

    @property
    def n(self) -> int:
        return self.n_side**3

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index


CONFIGS = (
    Config(0, "uniform-32^3", 32, 32.0, 10, 0.0, 32, 20000, 0.0, 1),
    Config(1, "halos30-128^3", 128, 128.0, 42, 0.30, 32, 20000, 0.0, 1),
    Config(2, "halos50-256^3", 256, 256.0, 85, 0.50, 32, 20000, 0.0, 1),
    Config(3, "halos40-512^3", 512, 512.0, 170, 0.40, 32, 200000, 0.0, 1),
    Config(4, "halos50-256^3-subcycle5", 256, 256.0, 85, 0.50, 32, 20000, 0.5, 5),
)


def scaled_config(cfg: Config, n_side: int) -> Config:
    """Same mixture at a smaller particle count and the same mean cell occupancy.

    Box and mesh shrink with n_side so that density (1 particle per unit volume) and
    the cell width stay as in `cfg`.  Used by parity tests that need an oracle-sized
    problem with the clustered structure of the big configs.
    """
    box_l = float(n_side)
    nc = int(box_l * cfg.nc / cfg.box_l)
    nc = max(nc, 3)
    while box_l / nc < cfg.r_max:
        nc -= 1
    return replace(cfg, n_side=n_side, box_l=box_l, nc=nc,
                   name=f"{cfg.name}@{n_side}^3")


def _halo_sizes(rng: np.random.Generator, budget: int, n_min: int, n_max: int) -> np.ndarray:
    """Truncated alpha=1 Pareto counts by inverse CDF until `budget` is used up."""
    sizes = []
    left = budget
    # mean of the truncated Pareto = n_min*ln(n_max/n_min)/(1-n_min/n_max)
    mean = n_min * np.log(n_max / n_min) / (1.0 - n_min / n_max)
    while left > 0:
        k = max(16, int(1.2 * left / mean) + 16)
        u = rng.random(k)
        n = np.floor(n_min / (1.0 - u * (1.0 - n_min / n_max))).astype(np.int64)
        n = np.clip(n, n_min, n_max)
        c = np.cumsum(n)
        m = int(np.searchsorted(c, left, side="left"))
        if m < k:  # budget reached inside this batch: truncate the last halo
            n = n[: m + 1].copy()
            n[m] -= c[m] - left
            sizes.append(n)
            left = 0
        else:
            sizes.append(n)
            left -= int(c[-1])
    out = np.concatenate(sizes) if sizes else np.zeros(0, np.int64)
    return out[out > 0]


_U_MAX = float((1.0 + 1.0 / 100.0) ** -1.5)  # r <= 10 a  <=>  u <= 1.01^-1.5


def _wrap32(p64: np.ndarray, box_l: float) -> np.ndarray:
    p64 -= box_l * np.floor(p64 / box_l)
    p = p64.astype(np.float32)
    p[p >= np.float32(box_l)] = 0.0
    p[p < 0] = 0.0
    return p


def make_particles(cfg: Config):
    """Return dict with float32 arrays x, y, z, vx, vy, vz, m (length cfg.n)."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed))
    n = cfg.n
    box_l = cfg.box_l
    n_halo_p = int(np.floor(cfg.f_halo * n))
    n_bg = n - n_halo_p
    pos = np.empty((3, n), dtype=np.float32)

    # background, in chunks to bound float64 temporaries
    chunk = 1 << 24
    for d in range(3):
        for s in range(0, n_bg, chunk):
            e = min(n_bg, s + chunk)
            pos[d, s:e] = _wrap32(rng.random(e - s) * box_l, box_l)

    n_halos = 0
    if n_halo_p > 0:
        sizes = _halo_sizes(rng, n_halo_p, cfg.halo_n_min, cfg.halo_n_max)
        n_halos = len(sizes)
        centres = rng.random((n_halos, 3)) * box_l
        a = 0.2 * 10.0 ** rng.random(n_halos)
        starts = np.concatenate(([0], np.cumsum(sizes)))
        # per-particle halo index, processed in chunks of halos
        h0 = 0
        while h0 < n_halos:
            h1 = int(np.searchsorted(starts, starts[h0] + chunk, side="right")) - 1
            h1 = min(max(h1, h0 + 1), n_halos)
            cnt = sizes[h0:h1]
            k = int(cnt.sum())
            hid = np.repeat(np.arange(h0, h1), cnt)
            u = rng.random(k) * _U_MAX
            u = np.maximum(u, 1e-300)
            r = a[hid] / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
            ct = 2.0 * rng.random(k) - 1.0
            st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
            ph = 2.0 * np.pi * rng.random(k)
            o = n_bg + int(starts[h0])
            pos[0, o:o + k] = _wrap32(centres[hid, 0] + r * st * np.cos(ph), box_l)
            pos[1, o:o + k] = _wrap32(centres[hid, 1] + r * st * np.sin(ph), box_l)
            pos[2, o:o + k] = _wrap32(centres[hid, 2] + r * ct, box_l)
            h0 = h1

    if cfg.sigma_v > 0:
        vel = np.empty((3, n), dtype=np.float32)
        for d in range(3):
            for s in range(0, n, chunk):
                e = min(n, s + chunk)
                vel[d, s:e] = (rng.standard_normal(e - s) * cfg.sigma_v).astype(np.float32)
    else:
        vel = np.zeros((3, n), dtype=np.float32)

    perm = rng.permutation(n)
    out = {}
    for i, k in enumerate("xyz"):
        out[k] = np.ascontiguousarray(pos[i][perm])
    for i, k in enumerate(("vx", "vy", "vz")):
        out[k] = np.ascontiguousarray(vel[i][perm]) if cfg.sigma_v > 0 else vel[i]
    out["m"] = np.ones(n, dtype=np.float32)
    out["n_halos"] = n_halos
    return out


def lattice_particles(n_side: int, spacing: float = 1.0, offset: float = 0.0):
    """Simple-cubic lattice, n_side^3 particles (DESIGN.md pin P3); box = n_side*spacing."""
    g = (np.arange(n_side, dtype=np.float64) * spacing + offset)
    zz, yy, xx = np.meshgrid(g, g, g, indexing="ij")
    f = lambda a: np.ascontiguousarray(a.ravel().astype(np.float32))
    return f(xx), f(yy), f(zz)


def dyadic_particles(n: int, box_l: float, bits: int, seed: int):
    """Uniform particles on a 2^-bits lattice: d, d^2 and s are then exact in float32
    for box_l <= 32 and bits <= 9 (reading S11 test fixture)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    k = int(round(box_l * (1 << bits)))
    p = rng.integers(0, k, size=(3, n)).astype(np.float64) / (1 << bits)
    return tuple(np.ascontiguousarray(p[i].astype(np.float32)) for i in range(3))
