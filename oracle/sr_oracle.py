"""ctypes front end of oracle/sr_oracle.c.  TEST INFRASTRUCTURE ONLY (see sr_oracle.c header).

Every function here is a thin call into the FP64 C oracle; the arithmetic lives in the C
file, each routine citing the PAPER.md passage it follows.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        fp = C.POINTER(C.c_float)
        dp = C.POINTER(C.c_double)
        u32p = C.POINTER(C.c_uint32)
        i64p = C.POINTER(C.c_int64)
        L.oracle_num_threads.restype = C.c_int
        L.oracle_fgrid_eq8.restype = C.c_double
        L.oracle_fgrid_eq8.argtypes = [C.c_double]
        L.oracle_fsr.restype = C.c_double
        L.oracle_fsr.argtypes = [C.c_double, C.c_double, dp]
        L.oracle_sr_brute.restype = C.c_uint64
        L.oracle_sr_brute.argtypes = [C.c_int64, fp, fp, fp, fp, C.c_double, C.c_float,
                                      C.c_float, fp, C.c_int64, i64p, dp, dp, dp, u32p, dp]
        L.oracle_mesh.restype = None
        L.oracle_mesh.argtypes = [C.c_int64, fp, fp, fp, C.c_double, C.c_int, u32p, u32p, u32p]
        L.oracle_sr_celllist.restype = C.c_uint64
        L.oracle_sr_celllist.argtypes = [C.c_int64, fp, fp, fp, fp, C.c_double, C.c_int,
                                         C.c_float, C.c_float, fp, C.c_int, C.c_int64, i64p,
                                         dp, dp, dp, u32p, C.POINTER(C.c_uint64), dp]
        L.oracle_kick.restype = None
        L.oracle_kick.argtypes = [C.c_int64, fp, dp, C.c_float, dp]
        L.oracle_drift.restype = None
        L.oracle_drift.argtypes = [C.c_int64, fp, fp, C.c_float, C.c_double, dp]
        _lib = L
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(C.POINTER(C.c_float))


def _ptr(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def fgrid_eq8(r):
    """PAPER.md Eq. 8 (line 179) evaluated in double."""
    r = np.atleast_1d(np.asarray(r, dtype=np.float64))
    return np.array([lib().oracle_fgrid_eq8(float(v)) for v in r])


def fsr(s, eps, poly):
    """PAPER.md Eq. 12 (line 337): (s+eps)^(-3/2) - P(s), double."""
    c = np.ascontiguousarray(np.asarray(poly, dtype=np.float32).astype(np.float64))
    s = np.atleast_1d(np.asarray(s, dtype=np.float64))
    return np.array([lib().oracle_fsr(float(v), float(eps), _ptr(c, C.c_double)) for v in s])


def sr_brute(x, y, z, m, box_l, r_max, eps, poly, targets=None):
    """Plain all-pairs sum.  Returns dict(ax, ay, az (float64), nbr (uint32), C, min_gap)."""
    x, px = _f32(x)
    y, py = _f32(y)
    z, pz = _f32(z)
    n = len(x)
    if m is None:
        pm = None
    else:
        m, pm = _f32(m)
    poly, pp = _f32(poly)
    if targets is None:
        nt, pt = n, None
    else:
        targets = np.ascontiguousarray(targets, dtype=np.int64)
        nt, pt = len(targets), _ptr(targets, C.c_int64)
    ax = np.zeros(nt)
    ay = np.zeros(nt)
    az = np.zeros(nt)
    nbr = np.zeros(nt, dtype=np.uint32)
    gap = C.c_double(0.0)
    tot = lib().oracle_sr_brute(n, px, py, pz, pm, float(box_l), float(r_max), float(eps), pp,
                                nt, pt, _ptr(ax, C.c_double), _ptr(ay, C.c_double),
                                _ptr(az, C.c_double), _ptr(nbr, C.c_uint32), C.byref(gap))
    return dict(ax=ax, ay=ay, az=az, nbr=nbr, C=int(tot), min_gap=gap.value)


def sr_celllist(x, y, z, m, box_l, nc, r_max, eps, poly, want_force=True, targets=None):
    """Independent linked-list chaining-mesh evaluation (all particles, or `targets`).

    Returns dict(nbr, C, n_eval[, ax, ay, az], seconds=(list build, evaluation))."""
    x, px = _f32(x)
    y, py = _f32(y)
    z, pz = _f32(z)
    n = len(x)
    if m is None:
        pm = None
    else:
        m, pm = _f32(m)
    poly, pp = _f32(poly)
    assert nc >= 3 and box_l / nc >= r_max
    if targets is None:
        nt, pt = n, None
    else:
        targets = np.ascontiguousarray(targets, dtype=np.int64)
        nt, pt = len(targets), _ptr(targets, C.c_int64)
    ax = np.zeros(nt if want_force else 1)
    ay = np.zeros(nt if want_force else 1)
    az = np.zeros(nt if want_force else 1)
    nbr = np.zeros(nt, dtype=np.uint32)
    nev = C.c_uint64(0)
    sec = np.zeros(2)
    tot = lib().oracle_sr_celllist(n, px, py, pz, pm, float(box_l), int(nc), float(r_max),
                                   float(eps), pp, int(bool(want_force)), nt, pt,
                                   _ptr(ax, C.c_double), _ptr(ay, C.c_double),
                                   _ptr(az, C.c_double), _ptr(nbr, C.c_uint32), C.byref(nev),
                                   _ptr(sec, C.c_double))
    out = dict(nbr=nbr, C=int(tot), n_eval=int(nev.value), seconds=(float(sec[0]), float(sec[1])))
    if want_force:
        out.update(ax=ax, ay=ay, az=az)
    return out


def mesh(x, y, z, box_l, nc):
    """Chaining mesh: dict(cid uint32[n], count uint32[nc^3], cell_start uint32[nc^3+1])."""
    x, px = _f32(x)
    y, py = _f32(y)
    z, pz = _f32(z)
    n = len(x)
    ncell = nc ** 3
    cid = np.zeros(n, dtype=np.uint32)
    count = np.zeros(ncell, dtype=np.uint32)
    start = np.zeros(ncell + 1, dtype=np.uint32)
    lib().oracle_mesh(n, px, py, pz, float(box_l), int(nc), _ptr(cid, C.c_uint32),
                      _ptr(count, C.c_uint32), _ptr(start, C.c_uint32))
    return dict(cid=cid, count=count, cell_start=start)


def kick(v, a, dt):
    v, pv = _f32(v)
    a = np.ascontiguousarray(a, dtype=np.float64)
    out = np.zeros(len(v))
    lib().oracle_kick(len(v), pv, _ptr(a, C.c_double), float(dt), _ptr(out, C.c_double))
    return out


def drift(x, v, dt, box_l):
    x, px = _f32(x)
    v, pv = _f32(v)
    out = np.zeros(len(x))
    lib().oracle_drift(len(x), px, pv, float(dt), float(box_l), _ptr(out, C.c_double))
    return out


def subcycle_sks(x, y, z, vx, vy, vz, m, box_l, nc, r_max, eps, poly, dt, n_sub):
    """The short-range map of PAPER.md Eq. 9 (line 207-212): n_sub sub-cycles of the symplectic
    SKS map of PAPER.md:205 (stream dt/2, kick dt with the force at the streamed positions,
    stream dt/2), composed in the paper's order with nothing merged or reordered:

        for each sub-cycle:  x <- S(dt/2) x;  a <- force(x);  v <- v + dt a;  x <- S(dt/2) x.

    The state arrays are float32 (they are float32 arrays in the path's interface); every map
    is evaluated in FP64 by the C oracle on the float32 state and rounded once.  Returns the
    final float32 state and the FP64 accelerations of the last kick."""
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    pos = [f32(x).copy(), f32(y).copy(), f32(z).copy()]
    vel = [f32(vx).copy(), f32(vy).copy(), f32(vz).copy()]
    acc = None
    for _ in range(int(n_sub)):
        pos = [_wrap32(drift(p, v, 0.5 * dt, box_l), box_l) for p, v in zip(pos, vel)]
        r = sr_celllist(pos[0], pos[1], pos[2], m, box_l, nc, r_max, eps, poly)
        acc = [r["ax"], r["ay"], r["az"]]
        vel = [kick(v, a, dt).astype(np.float32) for v, a in zip(vel, acc)]
        pos = [_wrap32(drift(p, v, 0.5 * dt, box_l), box_l) for p, v in zip(pos, vel)]
    return pos, vel, acc


def _wrap32(p64, box_l):
    """Round a position in [0, L) to float32; a value that rounds up to L becomes 0 (S16)."""
    p = p64.astype(np.float32)
    p[p >= np.float32(box_l)] = 0.0
    return p


# ---------------------------------------------------------------------------------------------
# Multi-level (density-adaptive) time stepping, PAPER.md:214-216 (section 2.5) and 315-325
# (section 3.1, Eq. 11).  Readings (S21-S23):
#   * the density estimate is the occupancy of the particle's chaining-mesh cell at the
#     BEGINNING of the long step ("fixed when the tree is constructed"); rho0 = N / nc^3 is the
#     mean occupancy, so rho/rho0 = n_c nc^3 / N;
#   * Eq. 11 (its floor brackets are garbled in PAPER.md:321): l = floor((rho/rho0) / d) + 1
#     kicks, raised to at least l_min ("at least 2 sub-cycles") and capped at l_max ("the
#     maximum level is capped");
#   * "to ensure time synchronization" the kick counts are powers of two: a particle takes
#     2^k kicks, 2^k the largest power of two <= l, k = its LEVEL; l_min, l_max powers of two;
#   * a particle with n kicks is evolved by n SKS maps S(T/2n) K(T/n) S(T/2n), "these stream
#     operators are further split such that all particles are acted on by the same number of
#     stream operators": everybody takes 2 l_max half streams S(T / (2 l_max)), and after half
#     stream h = 1 .. 2 l_max the particles of level k with h an odd multiple of l_max / 2^k are
#     kicked by T / 2^k with the force of ALL particles at the current positions -- that is
#     exactly level k = log2(l_max) - v2(h), v2 the number of trailing zero bits of h.
def kick_counts(count_of_cell, n_total, n_cells, d, l_min, l_max):
    """Eq. 11 per cell occupancy -> (kicks l, level k = floor(log2 l)) as integer arrays."""
    c = np.asarray(count_of_cell, dtype=np.float64)
    ratio = c * float(n_cells) / float(n_total)
    l = np.floor(ratio / float(d)).astype(np.int64) + 1
    l = np.clip(l, int(l_min), int(l_max))
    k = np.floor(np.log2(l.astype(np.float64)) + 1e-12).astype(np.int64)
    return l, k


def assign_levels(x, y, z, box_l, nc, d, l_min, l_max):
    """Level of every particle from the occupancy of its cell (oracle mesh)."""
    m = mesh(x, y, z, box_l, nc)
    _, k = kick_counts(m["count"], len(x), nc ** 3, d, l_min, l_max)
    return k[m["cid"].astype(np.int64)].astype(np.uint8)


def subcycle_multilevel(x, y, z, vx, vy, vz, m, box_l, nc, r_max, eps, poly, T, d, l_min, l_max,
                        levels=None):
    """One long step T of the multi-level short-range map, composed step by step in the order
    stated above.  float32 state, every map evaluated in FP64 by the C oracle and rounded once
    (as subcycle_sks).  Returns (pos, vel, levels, evaluated candidate pairs)."""
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    pos = [f32(x).copy(), f32(y).copy(), f32(z).copy()]
    vel = [f32(vx).copy(), f32(vy).copy(), f32(vz).copy()]
    lm = int(round(np.log2(l_max)))
    assert 2 ** lm == l_max and 2 ** int(round(np.log2(l_min))) == l_min and l_min <= l_max
    if levels is None:
        levels = assign_levels(pos[0], pos[1], pos[2], box_l, nc, d, l_min, l_max)
    levels = np.asarray(levels, dtype=np.uint8)
    half = 0.5 * T / l_max
    evals = 0
    for h in range(1, 2 * l_max + 1):
        pos = [_wrap32(drift(p, v, half, box_l), box_l) for p, v in zip(pos, vel)]
        v2 = (h & -h).bit_length() - 1
        k = lm - v2
        if k < 0:
            continue
        t = np.nonzero(levels == k)[0]
        if len(t) == 0:
            continue
        r = sr_celllist(pos[0], pos[1], pos[2], m, box_l, nc, r_max, eps, poly, targets=t)
        evals += r["n_eval"]
        dt = T / float(2 ** k)
        for c, a in zip(vel, (r["ax"], r["ay"], r["az"])):
            c[t] = kick(c[t], a, dt).astype(np.float32)
    return pos, vel, levels, evals
