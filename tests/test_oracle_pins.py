"""Pins for the CPU oracle (no GPU): closed forms, invariants, textbook reductions, brute force.

Each test is chosen so that a plausible mistake in oracle/sr_oracle.c (a dropped term, a
wrong sign or index, a transposed operand, <= instead of <) fails at least one of them.
Pin numbers P1..P10 follow SURVEY.md section 8(c) / DESIGN.md section 5.
"""
import os

import numpy as np
import pytest

from oracle import sr_oracle as orc
from oracle.fit_poly import fit_default_poly
from paper_1410_2805_b200 import workloads as wl

POLY = np.asarray(wl.DEFAULT_POLY, dtype=np.float32)
ZERO_POLY = np.zeros(6, dtype=np.float32)
EPS = 0.1
RMAX = 3.0


def _golden(golden_dir, kind):
    rows = []
    with open(os.path.join(golden_dir, "fsr_spot_values.txt")) as f:
        for line in f:
            t = line.split()
            if t and t[0] == kind:
                rows.append((float(t[1]), float(t[2])))
    return rows


def _arr(*v):
    return np.asarray(v, dtype=np.float32)


# ----------------------------------------------------------------------------- Eq. 8 / fit
def test_eq8_asymptotics():
    """Eq. 8 'has the correct asymptotic behaviors at small and large
    separation': Newtonian 1/r^2 at large r, and -> 0 linearly ((2/3) b^3 r + (c+e...)) at
    small r; a wrong sign on the second term would diverge like 2b/r."""
    r = np.array([10.0, 12.0, 20.0])
    np.testing.assert_allclose(orc.fgrid_eq8(r) * r * r, 1.0, atol=5e-5)
    r0 = np.array([1e-3, 2e-3])
    f = orc.fgrid_eq8(r0)
    # leading terms: (2/3) b^3 r + c r + e*(1 + ...) ; e = 1e-4 is the r -> 0 limit
    np.testing.assert_allclose(f, 1e-4 + (2.0 / 3.0 * 0.72 ** 3 + 0.01) * r0, rtol=0, atol=2e-7)


def test_eq8_matches_newtonian_at_three_cells(golden_dir):
    """Fig. 3 caption: the PM force matches 1/r^2 at ~3 grid cells; survey
    values of f_grid*r^2 (independent of this oracle)."""
    for r, v in _golden(golden_dir, "eq8r2"):
        assert abs(orc.fgrid_eq8(r)[0] * r * r - v) < 6e-5
    assert abs(orc.fgrid_eq8(3.0)[0] * 9.0 - 1.0) < 0.01


def test_default_poly_is_the_fit_of_eq8(golden_dir):
    c, err = fit_default_poly()
    assert np.array_equal(np.float32(c), POLY)
    assert err < 8e-4                                      # P9, second half
    for (k, v) in _golden(golden_dir, "coef"):
        assert abs(c[int(k)] - v) <= 2e-6 * abs(v)         # survey's independent fit
    # stored golden file is what the fitter writes
    rows = [l.split() for l in open(os.path.join(golden_dir, "poly_default.txt"))
            if not l.startswith("#")]
    assert np.array_equal(np.float32([float(r[2]) for r in rows]), POLY)


def test_force_matching_p9():
    """P9: with eps = 0 the short-range kernel vanishes at the matching scale r_s = 3
    (PAPER.md:132, 175): |f_SR(9)| <= 2e-4 against r^-3 = 0.037."""
    assert abs(orc.fsr(9.0, 0.0, POLY)[0]) <= 2e-4
    r = np.linspace(0.05, 3.0, 60)
    p = (1.0 / r ** 3) - orc.fsr(r * r, 0.0, POLY)           # = P(r^2)
    assert np.max(np.abs(r * p - orc.fgrid_eq8(r))) <= 8e-4


def test_fsr_spot_values_p1(golden_dir):
    for s, v in _golden(golden_dir, "fsr"):
        assert abs(orc.fsr(s, EPS, POLY)[0] - v) <= 2e-7 * max(1.0, abs(v))
    (s, v), = _golden(golden_dir, "poly")
    p1 = (s + EPS) ** -1.5 - orc.fsr(s, EPS, POLY)[0]
    assert abs(p1 - v) < 1e-8


# ----------------------------------------------------------------------------- two particles
@pytest.mark.parametrize("d", [(1.0, 0.0, 0.0), (0.5, -0.75, 1.25), (-1.5, 2.0, 0.25)])
def test_two_particle_plummer_closed_form_p1_p8(d):
    """poly = 0 -> textbook Plummer-softened Newtonian pair force, attractive (S5), with the
    neighbour's mass."""
    L = 32.0
    x = _arr(10.0, 10.0 + d[0]); y = _arr(12.0, 12.0 + d[1]); z = _arr(7.0, 7.0 + d[2])
    m = _arr(2.0, 3.0)
    o = orc.sr_brute(x, y, z, m, L, RMAX, EPS, ZERO_POLY)
    dv = np.array(d, dtype=np.float64)
    s = float(dv @ dv)
    w = (s + np.float64(np.float32(EPS))) ** -1.5
    a0 = 3.0 * w * dv          # on particle 0, towards particle 1, mass of particle 1
    a1 = -2.0 * w * dv
    got0 = np.array([o["ax"][0], o["ay"][0], o["az"][0]])
    got1 = np.array([o["ax"][1], o["ay"][1], o["az"][1]])
    np.testing.assert_allclose(got0, a0, rtol=1e-14, atol=1e-300)
    np.testing.assert_allclose(got1, a1, rtol=1e-14, atol=1e-300)
    assert list(o["nbr"]) == [1, 1] and o["C"] == 2


@pytest.mark.parametrize("k", range(6))
def test_polynomial_term_index_and_sign(k):
    """poly = e_k isolates -m d s^k (Eq. 12's minus sign, power k of s = r.r).  Dyadic
    coordinates make s^k exact, so the comparison is to rounding."""
    L = 32.0
    d = np.array([0.5, 1.0, -0.25])
    x = _arr(4.0, 4.0 + d[0]); y = _arr(4.0, 4.0 + d[1]); z = _arr(4.0, 4.0 + d[2])
    e = np.zeros(6, dtype=np.float32); e[k] = 1.0
    base = orc.sr_brute(x, y, z, None, L, RMAX, EPS, ZERO_POLY)
    o = orc.sr_brute(x, y, z, None, L, RMAX, EPS, e)
    s = float(d @ d)
    for c, name in enumerate(("ax", "ay", "az")):
        assert abs((o[name][0] - base[name][0]) - (-(s ** k) * d[c])) < 1e-13
        assert abs((o[name][1] - base[name][1]) - (+(s ** k) * d[c])) < 1e-13


def test_minimum_image_across_boundary():
    """S10: particle at 0.5 and particle at L-0.5 are 1 apart through the boundary; the
    force on the first points in -x."""
    L = 32.0
    for axis in range(3):
        p = [np.full(2, 5.0, np.float32) for _ in range(3)]
        p[axis] = _arr(0.5, L - 0.5)
        o = orc.sr_brute(p[0], p[1], p[2], None, L, RMAX, EPS, ZERO_POLY)
        a = np.array([o["ax"], o["ay"], o["az"]])          # [comp, particle]
        w = (1.0 + np.float64(np.float32(EPS))) ** -1.5
        expect = np.zeros((3, 2)); expect[axis] = [-w, +w]
        np.testing.assert_allclose(a, expect, atol=1e-15)
        assert o["C"] == 2


def test_cutoff_is_strict_p2():
    """S9: interact iff s < r_max^2."""
    L = 32.0
    y = _arr(3.0, 3.0); z = _arr(3.0, 3.0)
    o = orc.sr_brute(_arr(1.0, 4.0), y, z, None, L, RMAX, EPS, POLY)
    assert o["C"] == 0 and o["ax"][0] == 0.0 and o["min_gap"] == 0.0
    below = np.nextafter(np.float32(4.0), np.float32(0.0))
    o = orc.sr_brute(_arr(1.0, below), y, z, None, L, RMAX, EPS, POLY)
    assert o["C"] == 2 and o["ax"][0] != 0.0
    o = orc.sr_brute(_arr(1.0, 4.5), y, z, None, L, RMAX, EPS, POLY)
    assert o["C"] == 0 and o["ax"][0] == 0.0 and o["ax"][1] == 0.0


def test_self_and_coincident_particles_s8():
    """j == i excluded; distinct coincident particles count as a pair and add zero force."""
    L = 32.0
    x = _arr(5.0, 5.0, 6.0); y = _arr(5.0, 5.0, 5.0); z = _arr(5.0, 5.0, 5.0)
    o = orc.sr_brute(x, y, z, None, L, RMAX, EPS, POLY)
    assert list(o["nbr"]) == [2, 2, 2]
    assert o["ax"][0] == o["ax"][1] and o["ax"][0] > 0
    one = orc.sr_brute(_arr(5.0), _arr(5.0), _arr(5.0), None, L, RMAX, EPS, POLY)
    assert one["C"] == 0 and one["ax"][0] == 0.0


# ----------------------------------------------------------------------------- lattice, P3
def test_cubic_lattice_92_neighbours_zero_force_p3():
    """Unit simple-cubic lattice: #{k in Z^3 : 0 < |k|^2 < 9} = 6+12+8+6+24+24+0+12 = 92
    (sum of r_3(k), k = 1..8); with <= it would be 122.  Force zero by symmetry."""
    x, y, z = wl.lattice_particles(16, 1.0, 0.25)
    o = orc.sr_brute(x, y, z, None, 16.0, RMAX, EPS, POLY)
    assert np.all(o["nbr"] == 92) and o["C"] == 92 * 16 ** 3
    amax = max(np.abs(o[k]).max() for k in ("ax", "ay", "az"))
    assert amax < 1e-12
    c = orc.sr_celllist(x, y, z, None, 16.0, 5, RMAX, EPS, POLY)
    assert np.all(c["nbr"] == 92)


# ----------------------------------------------------------------------------- invariants
@pytest.fixture(scope="module")
def small_set():
    rng = np.random.default_rng(7)
    n, L = 3000, 16.0
    x, y, z = (rng.random(n) * L).astype(np.float32), (rng.random(n) * L).astype(np.float32), \
        (rng.random(n) * L).astype(np.float32)
    # a clump so that dense cells and many in-cutoff pairs exist
    x[:600] = (8.0 + 0.3 * rng.standard_normal(600)).astype(np.float32)
    y[:600] = (15.8 + 0.3 * rng.standard_normal(600)).astype(np.float32) % np.float32(L)
    z[:600] = (0.1 + 0.3 * rng.standard_normal(600)).astype(np.float32) % np.float32(L)
    m = (0.5 + rng.random(n)).astype(np.float32)
    return x, y, z, m, L


def test_newtons_third_law_p4(small_set):
    x, y, z, m, L = small_set
    o = orc.sr_brute(x, y, z, m, L, RMAX, EPS, POLY)
    md = m.astype(np.float64)
    scale = np.sum(md * np.sqrt(o["ax"] ** 2 + o["ay"] ** 2 + o["az"] ** 2))
    for k in ("ax", "ay", "az"):
        assert abs(np.sum(md * o[k])) < 1e-12 * scale
    assert o["C"] % 2 == 0 and o["C"] == int(o["nbr"].sum())


def test_permutation_invariance_p5(small_set):
    x, y, z, m, L = small_set
    o = orc.sr_brute(x, y, z, m, L, RMAX, EPS, POLY)
    p = np.random.default_rng(3).permutation(len(x))
    q = orc.sr_brute(x[p], y[p], z[p], m[p], L, RMAX, EPS, POLY)
    assert np.array_equal(q["nbr"], o["nbr"][p])
    scale = np.sqrt(np.mean(o["ax"] ** 2 + o["ay"] ** 2 + o["az"] ** 2))
    for k in ("ax", "ay", "az"):
        assert np.max(np.abs(q[k] - o[k][p])) < 1e-12 * scale


def test_translation_invariance_on_dyadic_lattice_p5():
    """Positions on a 2^-9 lattice and a shift by a lattice vector are exact in float32, so the
    wrapped set is the same physical configuration: counts identical, forces to rounding."""
    L = 16.0
    x, y, z = wl.dyadic_particles(2500, L, 9, seed=11)
    o = orc.sr_brute(x, y, z, None, L, RMAX, EPS, POLY)
    sh = np.float32([5.376953125, 11.0, 15.998046875])
    xs, ys, zs = [((a + s) % np.float32(L)).astype(np.float32) for a, s in zip((x, y, z), sh)]
    q = orc.sr_brute(xs, ys, zs, None, L, RMAX, EPS, POLY)
    assert np.array_equal(q["nbr"], o["nbr"])
    scale = np.sqrt(np.mean(o["ax"] ** 2 + o["ay"] ** 2 + o["az"] ** 2))
    for k in ("ax", "ay", "az"):
        assert np.max(np.abs(q[k] - o[k])) < 1e-11 * scale


def test_brute_force_equals_cell_list_p6(small_set):
    """27-cell completeness: the linked-list mesh evaluation finds exactly the
    brute-force pairs; nc = 5 gives w = 3.2 >= r_max."""
    x, y, z, m, L = small_set
    o = orc.sr_brute(x, y, z, m, L, RMAX, EPS, POLY)
    c = orc.sr_celllist(x, y, z, m, L, 5, RMAX, EPS, POLY)
    assert np.array_equal(c["nbr"], o["nbr"]) and c["C"] == o["C"]
    scale = np.sqrt(np.mean(o["ax"] ** 2 + o["ay"] ** 2 + o["az"] ** 2))
    for k in ("ax", "ay", "az"):
        assert np.max(np.abs(c[k] - o[k])) < 1e-12 * scale
    me = orc.mesh(x, y, z, L, 5)
    cnt = me["count"].astype(np.int64).reshape(5, 5, 5)
    nb = sum(np.roll(cnt, (i, j, k), (0, 1, 2)) for i in (-1, 0, 1) for j in (-1, 0, 1)
             for k in (-1, 0, 1))
    assert c["n_eval"] == int((cnt * nb).sum()) - len(x)
    assert o["min_gap"] > 1e-12           # S11: no pair within rounding of the cutoff


def test_brute_targets_subset(small_set):
    x, y, z, m, L = small_set
    o = orc.sr_brute(x, y, z, m, L, RMAX, EPS, POLY)
    t = np.array([5, 0, 2999, 17, 599])
    q = orc.sr_brute(x, y, z, m, L, RMAX, EPS, POLY, targets=t)
    assert np.array_equal(q["nbr"], o["nbr"][t])
    for k in ("ax", "ay", "az"):
        assert np.array_equal(q[k], o[k][t])


def test_celllist_targets_subset_equals_brute_subset(small_set):
    """The cell-list oracle restricted to a target list (used by bench.py's cpu_baseline
    sample) gives the brute-force rows of those targets."""
    x, y, z, m, L = small_set
    t = np.array([7, 0, 2999, 1234, 42])
    b = orc.sr_brute(x, y, z, m, L, RMAX, EPS, POLY, targets=t)
    nc = int(L // RMAX)
    q = orc.sr_celllist(x, y, z, m, L, nc, RMAX, EPS, POLY, targets=t)
    assert np.array_equal(q["nbr"], b["nbr"]) and q["C"] == b["C"]
    for k in ("ax", "ay", "az"):
        assert np.allclose(q[k], b[k], rtol=1e-12, atol=1e-13)
    assert q["seconds"][1] >= 0.0


def test_plummer_reduction_vs_numpy_p8():
    """poly = 0 and all particles within r_max/2 of a point: every pair interacts, no image
    matters, and the sum is the textbook softened N-body direct sum."""
    rng = np.random.default_rng(5)
    n, L = 48, 32.0
    p = (16.0 + (rng.random((3, n)) - 0.5) * 1.6).astype(np.float32)   # diameter < 1.39 < 3
    m = (0.5 + rng.random(n)).astype(np.float32)
    o = orc.sr_brute(p[0], p[1], p[2], m, L, RMAX, EPS, ZERO_POLY)
    P = p.astype(np.float64).T
    D = P[None, :, :] - P[:, None, :]
    S = np.einsum("ijk,ijk->ij", D, D) + np.float64(np.float32(EPS))
    W = S ** -1.5
    np.fill_diagonal(W, 0.0)
    A = np.einsum("ij,j,ijk->ik", W, m.astype(np.float64), D)
    got = np.stack([o["ax"], o["ay"], o["az"]], axis=1)
    np.testing.assert_allclose(got, A, rtol=1e-12, atol=1e-12)
    assert np.all(o["nbr"] == n - 1)


def test_uniform_pair_count_statistics_p7():
    """Config 0: E[C] = N(N-1)(4 pi/3) r_max^3 / L^3 ~ 3.706e6 (sigma ~ 2e3)."""
    cfg = wl.CONFIGS[0]
    p = wl.make_particles(cfg)
    c = orc.sr_celllist(p["x"], p["y"], p["z"], None, cfg.box_l, cfg.nc, cfg.r_max, cfg.eps,
                        POLY, want_force=False)
    n = cfg.n
    expect = n * (n - 1) * (4.0 * np.pi / 3.0) * cfg.r_max ** 3 / cfg.box_l ** 3
    assert abs(c["C"] - expect) < 1.5e4
    assert abs(c["n_eval"] - n * (n - 1) * 27.0 / cfg.nc ** 3) < 2e5


# ----------------------------------------------------------------------------- mesh, P10
def test_mesh_properties_p10():
    cfg = wl.scaled_config(wl.CONFIGS[1], 24)
    p = wl.make_particles(cfg)
    me = orc.mesh(p["x"], p["y"], p["z"], cfg.box_l, cfg.nc)
    nc, w = cfg.nc, cfg.box_l / cfg.nc
    assert int(me["count"].sum()) == cfg.n and me["cell_start"][-1] == cfg.n
    assert np.all(np.diff(me["cell_start"].astype(np.int64)) == me["count"])
    cid = me["cid"].astype(np.int64)
    cx, cy, cz = cid % nc, (cid // nc) % nc, cid // (nc * nc)
    for c, a in ((cx, p["x"]), (cy, p["y"]), (cz, p["z"])):
        a = a.astype(np.float64)
        assert np.all(a >= c * w - 1e-9) and np.all(a < (c + 1) * w + 1e-9)
    assert np.array_equal(np.bincount(cid, minlength=nc ** 3), me["count"])


def test_mesh_boundary_goes_to_upper_cell_p10():
    """x*nc/L integer -> upper cell (floor); nc = 10, L = 32: x = 16 -> cell 5; x = 0 -> 0;
    largest float below L -> nc-1.  x fastest in the linearisation (S13)."""
    L, nc = 32.0, 10
    top = np.nextafter(np.float32(L), np.float32(0))
    x = _arr(16.0, 0.0, top, np.nextafter(np.float32(16.0), np.float32(0)), 3.2)
    y = _arr(0.0, 16.0, 0.0, 0.0, 0.0)
    z = _arr(0.0, 0.0, 16.0, top, 0.0)
    me = orc.mesh(x, y, z, L, nc)
    # float32(3.2) = 3.2000000477 > 3.2 -> cell 1
    assert list(me["cid"]) == [5, 5 * nc, 9 + 5 * nc * nc, 4 + 9 * nc * nc, 1]


# ----------------------------------------------------------------------------- kick, drift
def test_kick_and_drift_closed_forms():
    v = _arr(1.0, -2.0, 0.0)
    a = np.array([4.0, 0.5, -8.0])
    dt = np.float32(0.01)
    np.testing.assert_allclose(orc.kick(v, a, dt), v.astype(np.float64) + float(dt) * a,
                               rtol=1e-15)
    L = 32.0
    x = _arr(31.995, 0.001, 5.0, 10.0, 0.0)
    vv = _arr(1.0, -1.0, 3200.0 * 3 + 100.0, -6400.0, 0.0)      # |dt v| > L too (S16)
    got = orc.drift(x, vv, dt, L)
    raw = x.astype(np.float64) + float(dt) * vv.astype(np.float64)
    assert np.all(got >= 0.0) and np.all(got < L)
    k = np.rint((raw - got) / L)
    np.testing.assert_allclose(got + k * L, raw, atol=1e-9)
    assert list(k) == [1.0, -1.0, 3.0, -2.0, 0.0]


# ------------------------------------------------------------------ SKS sub-cycle composition
def test_sks_single_subcycle_matches_hand_composition_two_particles():
    """n_sub = 1 on two particles against the maps written out by hand with the closed form
    of Eq. 12: x' = x + dt/2 v; v' = v + dt a(x'); x'' = x' + dt/2 v'."""
    L, dt, eps = 32.0, 0.05, 0.1
    c = np.asarray(POLY, dtype=np.float32).astype(np.float64)
    x0 = np.array([[10.0, 11.25], [7.0, 7.5], [20.0, 19.0]])          # [axis, particle]
    v0 = np.array([[0.5, -0.25], [0.125, 0.0], [-1.0, 0.75]])
    m = np.array([2.0, 3.0], np.float32)
    x1 = x0 + 0.5 * dt * v0
    d = x1[:, 1] - x1[:, 0]
    s = float(d @ d)
    f = (s + eps) ** -1.5 - sum(c[k] * s ** k for k in range(6))
    a = np.stack([m[1] * f * d, -m[0] * f * d], axis=1)               # on particle 0, 1
    v1 = v0 + dt * a
    x2 = x1 + 0.5 * dt * v1
    pos, vel, acc = orc.subcycle_sks(x0[0], x0[1], x0[2], v0[0], v0[1], v0[2], m, L, 10, 3.0, eps,
                                   POLY, dt, 1)
    for k in range(3):
        assert np.allclose(pos[k], x2[k], rtol=0, atol=4e-6)
        assert np.allclose(vel[k], v1[k], rtol=0, atol=1e-6)
        assert np.allclose(acc[k], a[k], rtol=2e-5, atol=1e-9)   # streamed state is float32


def test_sks_is_time_reversible():
    """SKS is a symmetric composition: running it with -dt undoes it (up to the float32
    rounding of the state)."""
    rng = np.random.default_rng(12)
    n, L = 3000, 32.0
    x, y, z = ((rng.random(n) * L).astype(np.float32) for _ in range(3))
    v = [(rng.standard_normal(n) * 0.3).astype(np.float32) for _ in range(3)]
    p1, v1, _ = orc.subcycle_sks(x, y, z, *v, None, L, 10, 3.0, 0.1, POLY, 0.01, 3)
    p0, v0, _ = orc.subcycle_sks(*p1, *v1, None, L, 10, 3.0, 0.1, POLY, -0.01, 3)
    for a, b in zip(p0, (x, y, z)):
        dd = np.abs(a - b)
        assert np.minimum(dd, L - dd).max() < 2e-5
    for a, b in zip(v0, v):
        assert np.abs(a - b).max() < 2e-5


# ------------------------------------------------------------------ overloading (NEXT-2)
@pytest.mark.parametrize("n_slabs", [2, 3, 4])
def test_overloaded_slabs_reproduce_the_whole_box(n_slabs):
    """with one >= r_max wide passive layer on each side, the union of the
    per-slab all-pairs sums (active targets, active + passive sources) IS the whole-box sum:
    identical neighbour counts, accelerations equal up to FP64 summation order.  Pinned
    against oracle_sr_brute on the whole box (not against itself); clustered particles, some
    halos straddling the slab faces and the periodic boundary, unequal masses."""
    from oracle import sharding as S
    W = wl

    cfg = W.scaled_config(W.CONFIGS[1], 24)          # 13 824 particles, L = 24, nc = 7
    p = W.make_particles(cfg)
    rng = np.random.default_rng(3)
    x, y, z = p["x"].copy(), p["y"].copy(), p["z"].copy()
    # a clump on a slab face and one across the periodic boundary in z
    z[:400] = np.mod(cfg.box_l / 2 + rng.standard_normal(400) * 0.7, cfg.box_l).astype(np.float32)
    z[400:800] = np.mod(rng.standard_normal(400) * 0.7, cfg.box_l).astype(np.float32)
    z[z >= cfg.box_l] = 0
    m = rng.uniform(0.5, 2.0, cfg.n).astype(np.float32)
    whole = orc.sr_brute(x, y, z, m, cfg.box_l, cfg.r_max, cfg.eps, W.DEFAULT_POLY)
    sh = S.sr_sharded(x, y, z, m, cfg.box_l, cfg.nc, cfg.r_max, cfg.eps, W.DEFAULT_POLY, n_slabs)
    assert np.array_equal(sh["nbr"], whole["nbr"])
    assert sh["C"] == whole["C"]
    scale = max(np.abs(whole[k]).max() for k in ("ax", "ay", "az"))
    for k in ("ax", "ay", "az"):
        assert np.abs(sh[k] - whole[k]).max() <= 1e-13 * scale
    # the passive sets are exactly the populations of the two adjacent layers
    cz = S.layer_of(z, cfg.box_l, cfg.nc)
    pop = np.bincount(cz, minlength=cfg.nc)
    for (lo, nz_own), n_pas in zip(S.slab_layers(cfg.nc, n_slabs), sh["n_passive"]):
        assert n_pas == pop[(lo - 1) % cfg.nc] + pop[(lo + nz_own) % cfg.nc]
    # layers from the mesh agree with the definition floor(z nc / L)
    assert np.array_equal(cz, np.floor(z.astype(np.float64) * cfg.nc / cfg.box_l).astype(np.int64))


def test_slab_layers_partition_the_mesh():
    from oracle import sharding as S

    for nc, k in ((7, 2), (10, 3), (42, 4), (170, 8), (85, 8)):
        sl = S.slab_layers(nc, k)
        assert sl[0][0] == 0 and sum(nz for _, nz in sl) == nc
        assert all(sl[i][0] + sl[i][1] == sl[i + 1][0] for i in range(k - 1))
        assert max(nz for _, nz in sl) - min(nz for _, nz in sl) <= 1
    with pytest.raises(ValueError):
        S.slab_layers(4, 2) if False else S.slab_layers(3, 2)


# ------------------------------------------------------------- multi-level stepping (NEXT-3)
def test_eq11_kick_counts_and_levels():
    """PAPER.md:321, Eq. 11 under reading S21: l = floor((rho/rho0)/d) + 1, clipped to
    [l_min, l_max], level = floor(log2 l).  Values worked by hand: N = 1000 particles on 10^3
    cells (rho0 = 1 per cell), d = 20."""
    l, k = orc.kick_counts([0, 1, 19, 20, 39, 40, 79, 80, 159, 160, 10 ** 6], 1000, 1000, 20, 1, 8)
    assert l.tolist() == [1, 1, 1, 2, 2, 3, 4, 5, 8, 8, 8]
    assert k.tolist() == [0, 0, 0, 1, 1, 1, 2, 2, 3, 3, 3]
    l, k = orc.kick_counts([0, 100, 10 ** 6], 1000, 1000, 20, 2, 4)      # "at least 2 sub-cycles"
    assert l.tolist() == [2, 4, 4] and k.tolist() == [1, 2, 2]
    # rho0 is the MEAN occupancy: the same cell in a box with twice the particles is half as dense
    assert orc.kick_counts([40], 2000, 1000, 20, 1, 8)[0].tolist() == [2]


def test_multilevel_all_on_one_level_is_the_sks_map():
    """Everybody on the finest level: the multi-level map IS (SKS(T/n))^n, bit for bit."""
    rng = np.random.default_rng(1)
    n, L, nc, T = 3000, 32.0, 10, 0.04
    x, y, z = ((rng.random(n) * L).astype(np.float32) for _ in range(3))
    v = [(rng.standard_normal(n) * 0.5).astype(np.float32) for _ in range(3)]
    for lv in (1, 4):
        p1, v1, lev, _ = orc.subcycle_multilevel(x, y, z, *v, None, L, nc, RMAX, EPS, POLY, T, 20,
                                                 lv, lv)
        p2, v2, _ = orc.subcycle_sks(x, y, z, *v, None, L, nc, RMAX, EPS, POLY, T / lv, lv)
        assert set(lev.tolist()) == {int(np.log2(lv))}
        for a, b in zip(p1 + v1, p2 + v2):
            assert np.array_equal(a, b)


def test_multilevel_two_levels_hand_composition():
    """Three particles, two levels, composed by hand from the two-body closed form (no cell
    list, no target lists): A and B share a cell (2 kicks each, level 1), C sits alone in the
    next cell within reach of B (1 kick, level 0).  l_max = 2: four half streams of T/4; A, B
    are kicked by T/2 after half streams 1 and 3, C by T after half stream 2."""
    L, nc, T, d = 32.0, 10, 0.08, 400.0
    x = _arr(4.0, 5.0, 6.9)
    y = _arr(4.0, 4.5, 4.2)
    z = _arr(4.0, 4.2, 3.9)
    v = [_arr(0.3, -0.2, 0.1), _arr(0.0, 0.4, -0.3), _arr(-0.1, 0.2, 0.25)]
    lev = orc.assign_levels(x, y, z, L, nc, d, 1, 2)
    assert lev.tolist() == [1, 1, 0]        # rho/rho0 = 2*1000/3 = 667 -> l = 2; 333 -> l = 1
    pos, vel, lev2, _ = orc.subcycle_multilevel(x, y, z, *v, None, L, nc, RMAX, EPS, POLY, T, d,
                                                1, 2)
    assert lev2.tolist() == [1, 1, 0]
    c = POLY.astype(np.float64)
    P = np.stack([x, y, z], 1).astype(np.float32)
    V = np.stack(v, 1).astype(np.float32)

    def acc(P64):
        a = np.zeros((3, 3))
        for i in range(3):
            for j in range(3):
                if i != j:
                    dvec = P64[j] - P64[i]
                    s = float(dvec @ dvec)
                    if s < RMAX ** 2:
                        a[i] += dvec * ((s + EPS) ** -1.5 - sum(c[k] * s ** k for k in range(6)))
        return a

    half = np.float32(0.5 * T / 2)
    for h in (1, 2, 3, 4):
        P = (P.astype(np.float64) + np.float64(half) * V.astype(np.float64)).astype(np.float32)
        a = acc(P.astype(np.float64))
        if h in (1, 3):
            V[:2] = (V[:2].astype(np.float64) + np.float64(np.float32(T / 2)) * a[:2]).astype(np.float32)
        elif h == 2:
            V[2] = (V[2].astype(np.float64) + np.float64(np.float32(T)) * a[2]).astype(np.float32)
    for k in range(3):
        assert np.allclose(pos[k], P[:, k], rtol=0, atol=1e-6)
        assert np.allclose(vel[k], V[:, k], rtol=0, atol=2e-7)
    assert np.abs(V - np.stack(v, 1)).max() > 1e-3      # the kicks did something


def test_multilevel_time_reversibility():
    """The map is a composition of symmetric SKS maps on a fixed level assignment, so running
    it, flipping the velocities and running it again returns to the start (to float32
    rounding of the state)."""
    rng = np.random.default_rng(8)
    n, L, nc, T = 1500, 16.0, 5, 0.02
    x, y, z = ((rng.random(n) * L).astype(np.float32) for _ in range(3))
    x[:300] = (8.0 + rng.standard_normal(300) * 0.4).astype(np.float32)     # a dense clump
    y[:300] = (8.0 + rng.standard_normal(300) * 0.4).astype(np.float32)
    z[:300] = (8.0 + rng.standard_normal(300) * 0.4).astype(np.float32)
    v = [(rng.standard_normal(n) * 0.2).astype(np.float32) for _ in range(3)]
    p1, v1, lev, ev = orc.subcycle_multilevel(x, y, z, *v, None, L, nc, RMAX, EPS, POLY, T, 2.0,
                                              1, 4)
    assert len(set(lev.tolist())) >= 2                   # really several levels
    full = orc.subcycle_multilevel(x, y, z, *v, None, L, nc, RMAX, EPS, POLY, T, 2.0, 4, 4)[3]
    assert ev < full                                      # and fewer evaluations than uniform
    p2, v2, _, _ = orc.subcycle_multilevel(*p1, *[-c for c in v1], None, L, nc, RMAX, EPS, POLY,
                                           T, 2.0, 1, 4, levels=lev)
    for a, b in zip(p2, (x, y, z)):
        dd = np.abs(a - b)
        assert np.minimum(dd, L - dd).max() <= 2e-5
    for a, b in zip(v2, v):
        assert np.abs(-a - b).max() <= 2e-4
