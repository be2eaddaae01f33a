"""-m gpu parity tests: the CUDA path (through the C ABI) against the FP64 CPU oracle on the
same seeded inputs.  Integers (cell ids, cell_start, neighbour counts, C) bit-exact;
accelerations within 1e-4 x A_rms on every component (north_star), written in gpu_helpers."""
import numpy as np
import pytest
import torch

from oracle import sr_oracle as O
from paper_1410_2805_b200 import haccsr
from paper_1410_2805_b200 import workloads as W

import gpu_helpers as H

pytestmark = pytest.mark.gpu

POLY = W.DEFAULT_POLY


def _ref_cell(p, cfg, mass=None, poly=POLY):
    return O.sr_celllist(p["x"], p["y"], p["z"], mass, cfg.box_l, cfg.nc, cfg.r_max, cfg.eps, poly)


# ------------------------------------------------------------------ config 0, full brute force
def test_config0_uniform_full_bruteforce_parity():
    cfg = W.CONFIGS[0]
    p = W.make_particles(cfg)
    ref = O.sr_brute(p["x"], p["y"], p["z"], None, cfg.box_l, cfg.r_max, cfg.eps, POLY)
    assert ref["min_gap"] > 1e-12  # no pair within rounding of the cutoff (reading S11)
    v0 = [p["vx"], p["vy"], p["vz"]]
    out, ctx = H.gpu_step(p["x"], p["y"], p["z"], cfg.box_l, cfg.nc, v=v0, dt=cfg.dt)
    H.check_mesh(ctx, O.mesh(p["x"], p["y"], p["z"], cfg.box_l, cfg.nc), p["x"], p["y"], p["z"])
    assert np.array_equal(out["nbr"], ref["nbr"])
    assert out["C"] == ref["C"]
    H.assert_accel_parity(out, ref)
    # kick: v + dt*a
    arms = H.accel_errors(out, ref)["arms"]
    for k, c in enumerate(("ax", "ay", "az")):
        vref = O.kick(v0[k], ref[c], cfg.dt)
        assert np.abs(out["v"][k] - vref).max() <= H.TOL_RMS * arms * cfg.dt + 1e-7
    assert out["stats"].n_eval - cfg.n == O.sr_celllist(
        p["x"], p["y"], p["z"], None, cfg.box_l, cfg.nc, cfg.r_max, cfg.eps, POLY,
        want_force=False)["n_eval"]


# ------------------------------------------------------ clustered mixtures at oracle-sized N
@pytest.mark.parametrize("ci,n_side", [(1, 48), (2, 56), (3, 56)])
def test_clustered_scaled_configs_parity(ci, n_side):
    cfg = W.scaled_config(W.CONFIGS[ci], n_side)
    p = W.make_particles(cfg)
    ref = _ref_cell(p, cfg)
    out, ctx = H.gpu_step(p["x"], p["y"], p["z"], cfg.box_l, cfg.nc)
    H.check_mesh(ctx, O.mesh(p["x"], p["y"], p["z"], cfg.box_l, cfg.nc), p["x"], p["y"], p["z"])
    assert np.array_equal(out["nbr"], ref["nbr"])
    assert out["C"] == ref["C"]
    assert out["stats"].n_eval - cfg.n == ref["n_eval"]
    e = H.assert_accel_parity(out, ref)
    # densest cell explicitly (FP32 accumulation over the longest source lists, reading S20)
    m = O.mesh(p["x"], p["y"], p["z"], cfg.box_l, cfg.nc)
    dense = np.nonzero(m["cid"] == np.argmax(m["count"]))[0]
    sub = {k: ref[k][dense] for k in ("ax", "ay", "az")}
    g = {k: out[k][dense] for k in ("ax", "ay", "az")}
    err = max(np.abs(g[k] - sub[k]).max() for k in sub)
    assert err <= H.TOL_RMS * e["arms"]
    assert out["stats"].n_split_items > 0  # the load-balance split path ran


@pytest.mark.parametrize("mode", ["0", "2"])
def test_sparse_item_kernel_on_and_off(mode, monkeypatch):
    """k_force_sparse (the sparse cells' items in a 64-register kernel, with k_force stealing
    from the back of the list) is switched on by particle count; force it on ("2") and off
    ("0") on an oracle-sized clustered problem: both must be the oracle's result.  Graphs are
    off so that the switch is read at every call."""
    monkeypatch.setenv("HACCSR_SPARSE_KERNEL", mode)
    monkeypatch.setenv("HACCSR_GRAPHS", "0")
    cfg = W.scaled_config(W.CONFIGS[2], 48)
    p = W.make_particles(cfg)
    rng = np.random.default_rng(17)
    m = rng.uniform(0.5, 2.0, cfg.n).astype(np.float32)
    ref = _ref_cell(p, cfg, mass=m)
    v = [np.zeros(cfg.n, np.float32) for _ in range(3)]
    out, _ = H.gpu_step(p["x"], p["y"], p["z"], cfg.box_l, cfg.nc, mass=m, v=v, dt=cfg.dt)
    assert np.array_equal(out["nbr"], ref["nbr"])
    assert out["C"] == ref["C"]
    e = H.assert_accel_parity(out, ref)
    for k, c in enumerate(("ax", "ay", "az")):
        assert np.abs(out["v"][k] - cfg.dt * ref[c]).max() <= H.TOL_RMS * e["arms"] * cfg.dt + 1e-7


# ---------------------------------------------------------------- closed forms / fixtures
def test_cubic_lattice_92_neighbours_zero_force():
    x, y, z = W.lattice_particles(16, 1.0, 0.25)
    out, _ = H.gpu_step(x, y, z, 16.0, 5)
    assert np.all(out["nbr"] == 92)
    assert out["C"] == 92 * 16 ** 3
    # symmetric sums of terms up to ~f_SR(1)*1 ~ 0.66: FP32 cancellation residue only
    assert max(np.abs(out[k]).max() for k in ("ax", "ay", "az")) < 2e-5


def test_dyadic_lattice_positions_exact_arithmetic():
    x, y, z = W.dyadic_particles(20000, 32.0, 9, seed=7)
    ref = O.sr_celllist(x, y, z, None, 32.0, 10, 3.0, 0.1, POLY)
    out, _ = H.gpu_step(x, y, z, 32.0, 10)
    assert np.array_equal(out["nbr"], ref["nbr"])
    H.assert_accel_parity(out, ref)


def test_two_particles_across_the_periodic_corner():
    L = 32.0
    x = np.array([0.25, 31.5], np.float32)
    y = np.array([31.75, 0.5], np.float32)
    z = np.array([0.125, 31.0], np.float32)
    m = np.array([2.0, 3.0], np.float32)
    ref = O.sr_brute(x, y, z, m, L, 3.0, 0.1, POLY)
    out, _ = H.gpu_step(x, y, z, L, 10, mass=m)
    assert ref["C"] == 2 and out["C"] == 2
    for k in ("ax", "ay", "az"):
        assert np.allclose(out[k], ref[k], rtol=3e-6, atol=1e-7)


def test_random_masses():
    cfg = W.scaled_config(W.CONFIGS[1], 32)
    p = W.make_particles(cfg)
    rng = np.random.default_rng(5)
    m = rng.uniform(0.5, 2.0, cfg.n).astype(np.float32)
    ref = _ref_cell(p, cfg, mass=m)
    out, _ = H.gpu_step(p["x"], p["y"], p["z"], cfg.box_l, cfg.nc, mass=m)
    assert np.array_equal(out["nbr"], ref["nbr"])
    H.assert_accel_parity(out, ref)


def test_polynomial_coefficients_are_an_input():
    cfg = W.CONFIGS[0]
    p = W.make_particles(W.scaled_config(cfg, 20))
    c2 = W.scaled_config(cfg, 20)
    poly = [0.3, -0.05, 0.02, -0.001, 1e-4, -2e-6]
    ref = _ref_cell(p, c2, poly=poly)
    out, _ = H.gpu_step(p["x"], p["y"], p["z"], c2.box_l, c2.nc, poly=poly)
    H.assert_accel_parity(out, ref)
    ref0 = _ref_cell(p, c2, poly=[0] * 6)   # Plummer-only
    out0, _ = H.gpu_step(p["x"], p["y"], p["z"], c2.box_l, c2.nc, poly=[0] * 6)
    H.assert_accel_parity(out0, ref0)


# ------------------------------------------------------------ the cutoff, adversarially
def test_pairs_at_the_cutoff_are_decided_exactly():
    """Pairs at |d| = 3 exactly and one float32 ulp either side, all orientations of
    (1,2,2), (0,0,3), and across the periodic boundary.  s = 9 is NOT inside (strict)."""
    L, nc = 64.0, 21
    rng = np.random.default_rng(11)
    dirs = []
    for base in [(1, 2, 2), (2, 1, 2), (2, 2, 1), (0, 0, 3), (0, 3, 0), (3, 0, 0)]:
        for sx in (1, -1):
            for sy in (1, -1):
                for sz in (1, -1):
                    dirs.append((base[0] * sx, base[1] * sy, base[2] * sz))
    xs, ys, zs = [], [], []
    k = 0
    # isolated pairs on a coarse grid of anchor points 8 apart (no cross-talk), anchors
    # include cells on the periodic faces
    anchors = [(a, b, c) for a in range(0, 64, 8) for b in range(0, 64, 8)
               for c in range(0, 64, 8)]
    rng.shuffle(anchors)
    for (a, b, c) in anchors:
        d = dirs[k % len(dirs)]
        mode = (k // len(dirs)) % 3  # exactly 3, one ulp closer, one ulp farther
        k += 1
        p0 = np.array([a + 0.5, b + 0.5, c + 0.5], np.float32)
        p1 = (p0 + np.array(d, np.float32)).astype(np.float32)
        ax = int(np.argmax(np.abs(d)))
        toward = p0[ax] if mode == 1 else (p1[ax] + np.float32(10 * np.sign(d[ax])))
        if mode != 0:
            p1[ax] = np.nextafter(p1[ax], np.float32(toward))
        p1 = np.where(p1 >= L, p1 - np.float32(L), p1)
        p1 = np.where(p1 < 0, p1 + np.float32(L), p1).astype(np.float32)
        xs += [p0[0], p1[0]]
        ys += [p0[1], p1[1]]
        zs += [p0[2], p1[2]]
    x, y, z = (np.array(v, np.float32) for v in (xs, ys, zs))
    ref = O.sr_celllist(x, y, z, None, L, nc, 3.0, 0.1, POLY)
    out, _ = H.gpu_step(x, y, z, L, nc)
    assert 0 < ref["C"] < len(x)            # some pairs in, some out
    assert np.array_equal(out["nbr"], ref["nbr"])
    assert out["stats"].n_recheck_tiles > 0  # the FP64 guard-band path decided them
    for k in ("ax", "ay", "az"):
        assert np.allclose(out[k], ref[k], rtol=1e-4, atol=2e-6)


# ------------------------------------------------------------------ degenerate inputs
def test_empty_and_single_particle():
    ctx = haccsr.Context(16, 32.0, 10)
    e = torch.empty(0, dtype=torch.float32, device="cuda:0")
    haccsr.hacc_sr_bin(ctx, e, e, e)
    a = torch.empty(1, dtype=torch.float32, device="cuda:0")
    tot = torch.full((1,), 12345, dtype=torch.int64, device="cuda:0")
    haccsr.hacc_sr_force(ctx, 0.1, 3.0, POLY, a, a.clone(), a.clone(), None, tot)
    haccsr.haccsr_sync(ctx)
    assert haccsr.haccsr_get_stats(ctx).n_items == 0
    assert int(tot.item()) == 0        # an empty mesh has C = 0 (the output is written)
    out, _ = H.gpu_step(np.array([5.0], np.float32), np.array([6.0], np.float32),
                        np.array([7.0], np.float32), 32.0, 10)
    assert out["C"] == 0 and out["nbr"][0] == 0
    assert out["ax"][0] == 0 and out["ay"][0] == 0 and out["az"][0] == 0


def test_all_particles_in_one_cell_and_coincident_points():
    """One dense cell: many target chunks x split source chunks (atomic combine), plus
    exactly coincident particles (count as pairs, add zero force; reading S8)."""
    rng = np.random.default_rng(3)
    n = 5000
    x = (rng.random(n) * 3.0 + 9.7).astype(np.float32)
    y = (rng.random(n) * 3.0 + 12.9).astype(np.float32)
    z = (rng.random(n) * 3.0 + 16.1).astype(np.float32)
    x[100:110] = x[100]
    y[100:110] = y[100]
    z[100:110] = z[100]
    ref = O.sr_brute(x, y, z, None, 32.0, 3.0, 0.1, POLY)
    v = [np.zeros(n, np.float32)] * 3
    out, _ = H.gpu_step(x, y, z, 32.0, 10, v=[c.copy() for c in v], dt=0.01)
    assert np.array_equal(out["nbr"], ref["nbr"])
    assert out["C"] == ref["C"]
    e = H.assert_accel_parity(out, ref)
    assert out["stats"].n_split_items > 0
    for k, c in enumerate(("ax", "ay", "az")):
        assert np.abs(out["v"][k] - 0.01 * ref[c]).max() <= H.TOL_RMS * e["arms"] * 0.01


def test_fused_kick_equals_force_then_kick():
    cfg = W.scaled_config(W.CONFIGS[2], 32)
    p = W.make_particles(cfg)
    rng = np.random.default_rng(9)
    v = [rng.standard_normal(cfg.n).astype(np.float32) for _ in range(3)]
    a, _ = H.gpu_step(p["x"], p["y"], p["z"], cfg.box_l, cfg.nc, v=[c.copy() for c in v],
                      fused=True)
    b, _ = H.gpu_step(p["x"], p["y"], p["z"], cfg.box_l, cfg.nc, v=[c.copy() for c in v],
                      fused=False)
    ref = _ref_cell(p, cfg)
    arms = H.accel_errors(a, ref)["arms"]
    for k, c in enumerate(("ax", "ay", "az")):
        vref = O.kick(v[k], ref[c], 0.01)
        assert np.abs(a["v"][k] - vref).max() <= H.TOL_RMS * arms * 0.01 + 1e-6
        assert np.abs(b["v"][k] - vref).max() <= H.TOL_RMS * arms * 0.01 + 1e-6


def test_box_whose_cell_scale_is_not_a_float():
    """L = 30, nc = 9: nc/L is not representable, the cell index takes the double path."""
    rng = np.random.default_rng(21)
    n = 30000
    L, nc = 30.0, 9
    x, y, z = ((rng.random(n) * L).astype(np.float32) for _ in range(3))
    x[:64] = np.float32(L / nc) * np.arange(64, dtype=np.float32) % np.float32(L)  # near edges
    for a in (x, y, z):
        a[a >= L] = 0
    ref = O.sr_celllist(x, y, z, None, L, nc, 3.0, 0.1, POLY)
    out, ctx = H.gpu_step(x, y, z, L, nc)
    H.check_mesh(ctx, O.mesh(x, y, z, L, nc), x, y, z)
    assert np.array_equal(out["nbr"], ref["nbr"])
    H.assert_accel_parity(out, ref)


def test_positions_on_cell_and_box_boundaries():
    L, nc = 32.0, 10
    g = np.arange(0, 32, dtype=np.float32)
    zz, yy, xx = np.meshgrid(g, g, g, indexing="ij")
    x, y, z = (np.ascontiguousarray(a.ravel()) for a in (xx, yy, zz))  # includes 0, 16 = L/2
    x = np.concatenate([x, np.array([np.nextafter(np.float32(32), np.float32(0))] * 3)])
    y = np.concatenate([y, np.array([0.0, 15.999999, 16.0], np.float32)])
    z = np.concatenate([z, np.array([31.999998, 3.2, 6.4], np.float32)])
    x, y, z = (a.astype(np.float32) for a in (x, y, z))
    out, ctx = H.gpu_step(x, y, z, L, nc)
    H.check_mesh(ctx, O.mesh(x, y, z, L, nc), x, y, z)
    ref = O.sr_celllist(x, y, z, None, L, nc, 3.0, 0.1, POLY)
    assert np.array_equal(out["nbr"], ref["nbr"])


def test_out_of_range_positions_wrap_and_nan_is_reported():
    L, nc = 32.0, 10
    rng = np.random.default_rng(2)
    n = 4000
    x, y, z = ((rng.random(n) * L).astype(np.float32) for _ in range(3))
    xo = x.copy()
    xo[:100] += np.float32(L)      # one box to the right
    xo[100:200] -= np.float32(2 * L)
    xw = O.drift(xo, np.zeros(n, np.float32), 0.0, L).astype(np.float32)  # the wrap rule
    ref = O.sr_celllist(xw, y, z, None, L, nc, 3.0, 0.1, POLY)
    out, _ = H.gpu_step(xo, y, z, L, nc)
    assert np.array_equal(out["nbr"], ref["nbr"])
    H.assert_accel_parity(out, ref)
    xo[7] = np.nan
    ctx = haccsr.Context(n, L, nc)
    haccsr.hacc_sr_bin(ctx, H.to_dev(xo), H.to_dev(y), H.to_dev(z))
    with pytest.raises(haccsr.HaccsrError) as e:
        haccsr.haccsr_sync(ctx)
    assert e.value.status == haccsr.EDATA


def test_call_order_and_argument_errors():
    ctx = haccsr.Context(100, 32.0, 10)
    a = torch.zeros(100, dtype=torch.float32, device="cuda:0")
    with pytest.raises(haccsr.HaccsrError) as e:
        haccsr.hacc_sr_force(ctx, 0.1, 3.0, POLY, a, a.clone(), a.clone())
    assert e.value.status == haccsr.ESTATE
    haccsr.hacc_sr_bin(ctx, a, a.clone(), a.clone())
    for eps, rmax in ((0.0, 3.0), (1e-30, 3.0), (0.1, 3.3), (0.1, -1.0)):
        with pytest.raises(haccsr.HaccsrError) as e:
            haccsr.hacc_sr_force(ctx, eps, rmax, POLY, a, a.clone(), a.clone())
        assert e.value.status == haccsr.EINVAL
    with pytest.raises(haccsr.HaccsrError) as e:
        haccsr.hacc_sr_kick(ctx, 0.01)
    assert e.value.status == haccsr.ESTATE
    big = torch.zeros(101, dtype=torch.float32, device="cuda:0")
    with pytest.raises(haccsr.HaccsrError) as e:
        haccsr.hacc_sr_bin(ctx, big, big.clone(), big.clone())
    assert e.value.status == haccsr.EINVAL


# -------------------------------------------------------------------- drift and sub-cycles
def test_drift_wraps_into_the_box():
    L = 32.0
    rng = np.random.default_rng(4)
    n = 50000
    x = (rng.random(n) * L).astype(np.float32)
    v = (rng.standard_normal(n) * 2000).astype(np.float32)   # many box lengths per step
    ctx = haccsr.Context(n, L, 10)
    d = [H.to_dev(x), H.to_dev(x[::-1].copy()), H.to_dev(x.copy())]
    dv = [H.to_dev(v), H.to_dev(v), H.to_dev(-v)]
    haccsr.hacc_sr_drift(ctx, *d, *dv, 0.01)
    haccsr.haccsr_sync(ctx)
    for pos, x0, v0 in ((d[0], x, v), (d[1], x[::-1], v), (d[2], x, -v)):
        got = pos.cpu().numpy()
        ref = O.drift(x0, v0, 0.01, L)
        assert np.all((got >= 0) & (got < L))
        diff = np.abs(got - ref)
        diff = np.minimum(diff, L - diff)
        # fma + one wrap rounding at magnitude up to |x + dt v| ~ 100
        assert diff.max() <= 2e-5


def test_subcycles_scaled_config4():
    """config 4 at oracle size: 5 x [drift, re-bin, force+kick]; each sub-cycle is compared
    from the GPU's own state (reading S15: chaotic divergence is not a bug)."""
    cfg = W.scaled_config(W.CONFIGS[4], 32)
    p = W.make_particles(cfg)
    n = cfg.n
    ctx = haccsr.Context(n, cfg.box_l, cfg.nc)
    pos = [H.to_dev(p[k]) for k in "xyz"]
    vel = [H.to_dev(p[k]) for k in ("vx", "vy", "vz")]
    acc = [torch.empty(n, dtype=torch.float32, device="cuda:0") for _ in range(3)]
    nbr = torch.empty(n, dtype=torch.int32, device="cuda:0")
    for sub in range(cfg.n_sub):
        x0 = [c.cpu().numpy() for c in pos]
        v0 = [c.cpu().numpy() for c in vel]
        haccsr.hacc_sr_drift(ctx, *pos, *vel, cfg.dt)
        haccsr.hacc_sr_bin(ctx, *pos, None, *vel)
        haccsr.hacc_sr_force_kick(ctx, cfg.eps, cfg.r_max, POLY, cfg.dt, *acc, nbr, None)
        haccsr.haccsr_sync(ctx)
        x1 = [c.cpu().numpy() for c in pos]
        for k in range(3):
            ref = O.drift(x0[k], v0[k], cfg.dt, cfg.box_l)
            d = np.abs(x1[k] - ref)
            assert np.minimum(d, cfg.box_l - d).max() <= 1e-5
        ref = O.sr_celllist(x1[0], x1[1], x1[2], None, cfg.box_l, cfg.nc, cfg.r_max, cfg.eps,
                            POLY)
        out = dict(ax=acc[0].cpu().numpy(), ay=acc[1].cpu().numpy(), az=acc[2].cpu().numpy())
        assert np.array_equal(nbr.cpu().numpy().view(np.uint32), ref["nbr"])
        e = H.assert_accel_parity(out, ref)
        for k, c in enumerate(("ax", "ay", "az")):
            vref = O.kick(v0[k], ref[c], cfg.dt)
            got = vel[k].cpu().numpy()
            assert np.abs(got - vref).max() <= H.TOL_RMS * e["arms"] * cfg.dt + \
                4e-7 * np.abs(vref).max()


def _count_all(x, y, z, cfg, cid):
    """The oracle's count-only cell list over ALL particles.  The particles are handed over in
    cell order (a permutation of the input: the per-particle result does not depend on it,
    pin P5) because the linked-list traversal is several times faster on a cache-friendly
    order; the counts come back in the original order."""
    order = np.argsort(cid, kind="stable")
    r = O.sr_celllist(x[order], y[order], z[order], None, cfg.box_l, cfg.nc, cfg.r_max, cfg.eps,
                      POLY, want_force=False)
    nbr = np.empty_like(r["nbr"])
    nbr[order] = r["nbr"]
    return dict(nbr=nbr, C=r["C"], n_eval=r["n_eval"])


# ------------------------------------------------- full BASELINE sizes, sampled outputs
def _full_size_sampled(ci, n_random, n_dense, n_dense_cells=1, full_count=False):
    """bench.py's launch configuration (bin with velocities, fused force+kick, no counting)
    at a full BASELINE.json config; the oracle evaluates a sample of targets one by one:
    random particles plus particles of the densest cell.  Whole-array properties that hold
    at any size: mesh equal to the oracle's, N_eval from the oracle's histogram, Newton's
    third law."""
    cfg = W.CONFIGS[ci]
    p = W.make_particles(cfg)
    n = cfg.n
    ctx = haccsr.Context(n, cfg.box_l, cfg.nc)
    pos = [H.to_dev(p[k]) for k in "xyz"]
    vel = [H.to_dev(p[k]) for k in ("vx", "vy", "vz")]
    acc = [torch.empty(n, dtype=torch.float32, device="cuda:0") for _ in range(3)]
    haccsr.hacc_sr_bin(ctx, *pos, None, *vel)
    haccsr.hacc_sr_force_kick(ctx, cfg.eps, cfg.r_max, POLY, cfg.dt, *acc, None, None)
    haccsr.haccsr_sync(ctx)
    st = haccsr.haccsr_get_stats(ctx)

    # mesh: bit-exact cell_start and per-particle cell ids against the oracle
    ref_mesh = O.mesh(p["x"], p["y"], p["z"], cfg.box_l, cfg.nc)
    m = haccsr.haccsr_get_mesh(ctx)
    assert np.array_equal(m["cell_start"].cpu().numpy().astype(np.uint32), ref_mesh["cell_start"])
    assert np.array_equal(m["cell_id"].cpu().numpy().astype(np.uint32), ref_mesh["cid"])
    perm = m["perm"].cpu().numpy()
    seen = np.zeros(n, dtype=bool)
    seen[perm] = True
    assert seen.all()                                        # perm is a permutation
    assert np.array_equal(m["sorted_pos"][:, 0].cpu().numpy(), p["x"][perm])
    del m, seen
    # candidate pairs of the plain 27-cell mesh from the oracle's histogram
    cnt = ref_mesh["count"].astype(np.int64).reshape(cfg.nc, cfg.nc, cfg.nc)
    s27 = np.zeros_like(cnt)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                s27 += np.roll(cnt, (dz, dy, dx), axis=(0, 1, 2))
    assert st.n_eval == int((cnt * s27).sum())
    assert st.max_cell_count == int(cnt.max())

    # sampled targets
    rng = np.random.default_rng(100 + ci)
    t_rand = rng.choice(n, size=n_random, replace=False)
    # n_dense particles from each of the n_dense_cells densest cells (BASELINE.md section 3:
    # the dense cores are where FP32 accumulation and the split/atomic path are exercised)
    dense_cells = np.argsort(ref_mesh["count"])[::-1][:n_dense_cells]
    order = np.argsort(ref_mesh["cid"], kind="stable")
    t_dense = []
    for dc in dense_cells:
        in_dense = order[ref_mesh["cell_start"][dc]:ref_mesh["cell_start"][dc + 1]]
        t_dense.append(rng.choice(in_dense, size=min(n_dense, len(in_dense)), replace=False))
    del order
    targets = np.unique(np.concatenate([t_rand] + t_dense))
    ref = O.sr_celllist(p["x"], p["y"], p["z"], None, cfg.box_l, cfg.nc, cfg.r_max, cfg.eps,
                        POLY, targets=targets)
    a = [c.cpu().numpy() for c in acc]
    out = dict(ax=a[0][targets], ay=a[1][targets], az=a[2][targets])
    # A_rms of the whole set is not known to the oracle; the sample's own RMS (random
    # targets only, an unbiased estimate) sets the scale, reading S17
    is_rand = np.isin(targets, t_rand)
    r = np.stack([ref["ax"], ref["ay"], ref["az"]], 1)
    arms = float(np.sqrt(np.mean(np.sum(r[is_rand] ** 2, axis=1))))
    g = np.stack([out["ax"], out["ay"], out["az"]], 1).astype(np.float64)
    err = np.abs(g - r).max()
    assert err <= H.TOL_RMS * arms, (err, arms)
    rel = np.sqrt(((g - r) ** 2).sum(1)) / np.maximum(np.sqrt((r ** 2).sum(1)), 1e-30)
    assert np.median(rel) <= 2e-5
    # fused kick on the sampled targets
    for k, c in enumerate(("ax", "ay", "az")):
        vref = O.kick(p[("vx", "vy", "vz")[k]][targets], ref[c], cfg.dt)
        got = vel[k].cpu().numpy()[targets]
        assert np.abs(got - vref).max() <= H.TOL_RMS * arms * cfg.dt + 4e-7 * np.abs(vref).max()
    # Newton's third law over the whole box (unit masses): |sum a| is rounding noise of
    # N terms of size ~A_rms
    tot = np.array([float(c.double().sum().item()) for c in acc])
    assert np.abs(tot).max() <= 1e-5 * arms * n

    # the counting variant: neighbour counts bit-exact on the sample, total C consistent
    nbr = torch.empty(n, dtype=torch.int32, device="cuda:0")
    ctot = torch.zeros(1, dtype=torch.int64, device="cuda:0")
    haccsr.hacc_sr_force(ctx, cfg.eps, cfg.r_max, POLY, *acc, nbr, ctot)
    haccsr.haccsr_sync(ctx)
    nbr_gpu = nbr.cpu().numpy().view(np.uint32)
    assert np.array_equal(nbr_gpu[targets], ref["nbr"])
    # C restricted to the sampled targets, bit-exact against the oracle's own total
    assert int(nbr_gpu[targets].astype(np.int64).sum()) == ref["C"]
    assert int(ctot.item()) == int(nbr.to(torch.int64).sum().item())
    if full_count:
        # north_star: "bit-exact interacting-pair count" -- the oracle's count-only cell list
        # over ALL particles: every n_i and the total C (the numerator of bench.py's value)
        full = _count_all(p["x"], p["y"], p["z"], cfg, ref_mesh["cid"])
        assert np.array_equal(nbr_gpu, full["nbr"])
        assert int(ctot.item()) == full["C"]
        assert st.n_eval - n == full["n_eval"]
    return st


def test_full_size_config1_sampled_forces_and_full_exact_count():
    _full_size_sampled(1, n_random=20000, n_dense=512, full_count=True)


def test_full_size_config2_sampled_forces_and_full_exact_count():
    _full_size_sampled(2, n_random=8192, n_dense=256, full_count=True)


def test_full_size_config3_sampled_bench_configuration():
    """configs[3] (the bench workload): 65 536 random targets plus 128 particles from each of
    the 64 densest cells (every particle of those cells would be 1e13
    candidate pairs for the linked-list oracle), n_i bit-exact on all of them and the GPU's C
    over those targets equal to the oracle's."""
    st = _full_size_sampled(3, n_random=65536, n_dense=128, n_dense_cells=64)
    assert st.n_split_items > 0


def test_full_size_config4_subcycles_sampled():
    """configs[4] at full size: 5 x [drift, re-bin, force+kick] on the 256^3 halo mixture with
    Gaussian velocities.  Every sub-cycle is checked from the GPU's own state (reading S15) on
    sampled targets: drift against the oracle's stream map, mesh against the oracle's mesh,
    accelerations and kicked velocities against the oracle's cell list."""
    cfg = W.CONFIGS[4]
    p = W.make_particles(cfg)
    n = cfg.n
    ctx = haccsr.Context(n, cfg.box_l, cfg.nc)
    pos = [H.to_dev(p[k]) for k in "xyz"]
    vel = [H.to_dev(p[k]) for k in ("vx", "vy", "vz")]
    acc = [torch.empty(n, dtype=torch.float32, device="cuda:0") for _ in range(3)]
    rng = np.random.default_rng(404)
    occupancy = []
    for sub in range(cfg.n_sub):
        targets = np.sort(rng.choice(n, size=2048, replace=False))
        x0 = [c.cpu().numpy() for c in pos]
        v0 = [c.cpu().numpy()[targets] for c in vel]
        haccsr.hacc_sr_drift(ctx, *pos, *vel, cfg.dt)
        haccsr.hacc_sr_bin(ctx, *pos, None, *vel)
        haccsr.hacc_sr_force_kick(ctx, cfg.eps, cfg.r_max, POLY, cfg.dt, *acc, None, None)
        haccsr.haccsr_sync(ctx)
        x1 = [c.cpu().numpy() for c in pos]
        for k in range(3):   # stream map on the sample
            ref = O.drift(x0[k][targets], v0[k], cfg.dt, cfg.box_l)
            d = np.abs(x1[k][targets] - ref)
            assert np.minimum(d, cfg.box_l - d).max() <= 2e-5 + 1e-6 * np.abs(v0[k]).max() * cfg.dt
            assert x1[k].min() >= 0.0 and x1[k].max() < cfg.box_l
        ref_mesh = O.mesh(x1[0], x1[1], x1[2], cfg.box_l, cfg.nc)
        m = haccsr.haccsr_get_mesh(ctx)
        assert np.array_equal(m["cell_start"].cpu().numpy().astype(np.uint32),
                              ref_mesh["cell_start"])
        del m
        if sub == 0:
            # exact interacting-pair count of the whole sub-cycle: the counting variant of the
            # same kernel on the same mesh against the oracle's count-only pass over all
            # particles (north_star: bit-exact pair count)
            nbr = torch.empty(n, dtype=torch.int32, device="cuda:0")
            ctot = torch.zeros(1, dtype=torch.int64, device="cuda:0")
            scratch = [torch.empty_like(acc[0]) for _ in range(3)]
            haccsr.hacc_sr_force(ctx, cfg.eps, cfg.r_max, POLY, *scratch, nbr, ctot)
            haccsr.haccsr_sync(ctx)
            full = _count_all(x1[0], x1[1], x1[2], cfg, ref_mesh["cid"])
            assert np.array_equal(nbr.cpu().numpy().view(np.uint32), full["nbr"])
            assert int(ctot.item()) == full["C"]
            del nbr, scratch, full
        occupancy.append(int(ref_mesh["count"].max()))
        dense = np.nonzero(ref_mesh["cid"] == int(np.argmax(ref_mesh["count"])))[0]
        t_all = np.unique(np.concatenate([targets, rng.choice(dense, size=min(64, len(dense)),
                                                              replace=False)]))
        ref = O.sr_celllist(x1[0], x1[1], x1[2], None, cfg.box_l, cfg.nc, cfg.r_max, cfg.eps,
                            POLY, targets=t_all)
        r = np.stack([ref["ax"], ref["ay"], ref["az"]], 1)
        g = np.stack([c.cpu().numpy()[t_all] for c in acc], 1).astype(np.float64)
        is_rand = np.isin(t_all, targets)
        arms = float(np.sqrt(np.mean(np.sum(r[is_rand] ** 2, axis=1))))
        assert np.abs(g - r).max() <= H.TOL_RMS * arms, (sub, np.abs(g - r).max(), arms)
        sel = np.searchsorted(t_all, targets)
        for k in range(3):   # kick from the velocities the GPU held before this sub-cycle
            vref = O.kick(v0[k], r[sel, k], cfg.dt)
            got = vel[k].cpu().numpy()[targets]
            assert np.abs(got - vref).max() <= H.TOL_RMS * arms * cfg.dt + \
                4e-7 * np.abs(vref).max()
    assert len(occupancy) == cfg.n_sub


# ------------------------------------------------------------- sort edge cases (sort.cu)
def test_long_rows_with_masses_take_the_multi_tile_sort_path():
    """Two adjacent cells hold 30 000 particles (one (cz,cy) row longer than a sort tile),
    random masses: the count pass + tile passes of k_sort_rows and the index array."""
    rng = np.random.default_rng(31)
    L, nc, n = 32.0, 10, 30000
    x = (rng.random(n) * 6.0 + 12.9).astype(np.float32)
    y = (rng.random(n) * 3.0 + 9.7).astype(np.float32)
    z = (rng.random(n) * 3.0 + 16.1).astype(np.float32)
    bg = 3000
    x[:bg], y[:bg], z[:bg] = ((rng.random(bg) * L).astype(np.float32) for _ in range(3))
    m = rng.uniform(0.5, 2.0, n).astype(np.float32)
    out, ctx = H.gpu_step(x, y, z, L, nc, mass=m, count=True)
    mesh = H.check_mesh(ctx, O.mesh(x, y, z, L, nc), x, y, z)
    perm = mesh["perm"].cpu().numpy()
    assert np.array_equal(mesh["sorted_pos"].cpu().numpy()[:, 3], m[perm])   # masses travel
    t = np.sort(rng.choice(n, 3000, replace=False))
    ref = O.sr_celllist(x, y, z, m, L, nc, 3.0, 0.1, POLY, targets=t)
    assert np.array_equal(out["nbr"][t], ref["nbr"])
    sub = dict(ax=out["ax"][t], ay=out["ay"][t], az=out["az"][t])
    H.assert_accel_parity(sub, ref)


@pytest.mark.parametrize("nc,L", [(4, 12.5), (230, 700.0), (256, 768.0)])
def test_smallest_and_largest_meshes(nc, L):
    """nc = 4 (every cell is its own periodic neighbour's neighbour) and meshes whose nc^2 row
    histogram does not fit shared memory (global-counter path of k_count_rows)."""
    rng = np.random.default_rng(nc)
    n = 4000 if nc == 4 else 60000
    x, y, z = ((rng.random(n) * L).astype(np.float32) for _ in range(3))
    if nc > 4:   # a clump so that some pairs interact in the huge box
        x[:20000] = (rng.random(20000) * 9.0 + (L - 4.0)).astype(np.float32) % np.float32(L)
        y[:20000] = (rng.random(20000) * 9.0).astype(np.float32)
        z[:20000] = (rng.random(20000) * 9.0 + L / 2).astype(np.float32)
    for a in (x, y, z):
        a[a >= L] = 0
    out, ctx = H.gpu_step(x, y, z, L, nc)
    H.check_mesh(ctx, O.mesh(x, y, z, L, nc), x, y, z)
    ref = O.sr_celllist(x, y, z, None, L, nc, 3.0, 0.1, POLY)
    assert np.array_equal(out["nbr"], ref["nbr"])
    assert out["C"] == ref["C"] and ref["C"] > 0
    H.assert_accel_parity(out, ref)


def test_rebinning_the_same_context_with_fewer_particles():
    """A context is reused with a different n (sub-cycles do this every step): no stale
    mesh state may survive."""
    rng = np.random.default_rng(77)
    L, nc = 32.0, 10
    ctx = haccsr.Context(50000, L, nc)
    for n in (50000, 777, 20000):
        x, y, z = ((rng.random(n) * L).astype(np.float32) for _ in range(3))
        d = [H.to_dev(a) for a in (x, y, z)]
        acc = [torch.empty(n, dtype=torch.float32, device="cuda:0") for _ in range(3)]
        nbr = torch.empty(n, dtype=torch.int32, device="cuda:0")
        haccsr.hacc_sr_bin(ctx, *d)
        haccsr.hacc_sr_force(ctx, 0.1, 3.0, POLY, *acc, nbr, None)
        haccsr.haccsr_sync(ctx)
        H.check_mesh(ctx, O.mesh(x, y, z, L, nc), x, y, z)
        ref = O.sr_celllist(x, y, z, None, L, nc, 3.0, 0.1, POLY)
        assert np.array_equal(nbr.cpu().numpy().view(np.uint32), ref["nbr"])


# ------------------------------------------------------------------ SKS sub-cycles (Eq. 9)
@pytest.mark.parametrize("n_sub", [1, 4, 10])
def test_subcycle_sks_matches_the_oracle_composition(n_sub):
    """hacc_sr_subcycle = n_sub x [S(dt/2) K(dt) S(dt/2)] against the
    oracle's step-by-step composition on a smooth problem (uniform points, small velocities:
    no chaotic amplification over a few sub-cycles), masses included."""
    rng = np.random.default_rng(90 + n_sub)
    n, L, nc, dt = 20000, 32.0, 10, 0.01
    x, y, z = ((rng.random(n) * L).astype(np.float32) for _ in range(3))
    v = [(rng.standard_normal(n) * 0.5).astype(np.float32) for _ in range(3)]
    m = rng.uniform(0.5, 2.0, n).astype(np.float32)
    pos_ref, vel_ref, acc_ref = O.subcycle_sks(x, y, z, *v, m, L, nc, 3.0, 0.1, POLY, dt, n_sub)
    ctx = haccsr.Context(n, L, nc)
    dp = [H.to_dev(a) for a in (x, y, z)]
    dv = [H.to_dev(a) for a in v]
    da = [torch.empty(n, dtype=torch.float32, device="cuda:0") for _ in range(3)]
    haccsr.hacc_sr_subcycle(ctx, *dp, H.to_dev(m), *dv, 0.1, 3.0, POLY, dt, n_sub, *da)
    haccsr.haccsr_sync(ctx)
    r = np.stack(acc_ref, 1)
    arms = float(np.sqrt(np.mean(np.sum(r * r, axis=1))))
    # The two sides round their float32 state independently, so after the first sub-cycle
    # their positions differ by an ulp or two; a pair that sits within that of the cutoff
    # then interacts on one side only (a jump of |f_SR(9)| r_max m ~ 3e-3 in a, reading S7).
    # So: nearly all particles within the force tolerance, every particle within a few
    # such jumps.
    jump = 4e-3
    for k in range(3):
        dd = np.abs(dp[k].cpu().numpy() - pos_ref[k])
        # 2 n_sub streams, each rounded once on either side: up to an ulp (1.9e-6 at x in
        # [16, 32)) per stream, plus the velocity differences times the elapsed time
        assert np.minimum(dd, L - dd).max() <= max(1e-5, (2 * n_sub + 2) * 1.91e-6 + 1e-5)
        ev = np.abs(dv[k].cpu().numpy() - vel_ref[k])
        assert np.quantile(ev, 0.99) <= n_sub * (H.TOL_RMS * arms * dt + 2e-7)
        assert ev.max() <= n_sub * (H.TOL_RMS * arms * dt + 2e-7 + 2 * jump * dt)
        ea = np.abs(da[k].cpu().numpy() - acc_ref[k])
        assert np.quantile(ea, 0.99) <= 4 * H.TOL_RMS * arms
        assert ea.max() <= 4 * H.TOL_RMS * arms + 2 * jump


def test_subcycle_argument_errors():
    ctx = haccsr.Context(100, 32.0, 10)
    a = torch.zeros(100, dtype=torch.float32, device="cuda:0")
    b = [a.clone() for _ in range(9)]
    with pytest.raises(haccsr.HaccsrError) as e:
        haccsr.hacc_sr_subcycle(ctx, b[0], b[1], b[2], None, b[3], b[4], b[5], 0.1, 3.0, POLY,
                                0.01, 0, b[6], b[7], b[8])
    assert e.value.status == haccsr.EINVAL
    with pytest.raises(haccsr.HaccsrError) as e:
        haccsr.hacc_sr_subcycle(ctx, b[0], b[1], b[2], None, None, None, None, 0.1, 3.0, POLY,
                                0.01, 2, b[6], b[7], b[8])
    assert e.value.status == haccsr.EINVAL


def test_subcycle_error_return_leaves_the_state_untouched():
    """Argument errors are found before anything is enqueued: after an EINVAL return the
    positions and velocities are bit-identical (no half stream without its kick)."""
    rng = np.random.default_rng(12)
    n, L, nc = 5000, 32.0, 10
    host = [(rng.random(n) * L).astype(np.float32) for _ in range(3)] + \
           [rng.standard_normal(n).astype(np.float32) for _ in range(3)]
    ctx = haccsr.Context(n, L, nc)
    a = [torch.zeros(n, dtype=torch.float32, device="cuda:0") for _ in range(3)]
    bad_poly = list(POLY)
    bad_poly[2] = float("nan")
    cases = [dict(eps=0.0), dict(eps=1e-30), dict(r_max=3.3), dict(poly=bad_poly),
             dict(acc=[a[0], None, a[2]])]
    for case in cases:
        d = [H.to_dev(h) for h in host]
        acc = case.get("acc", a)
        with pytest.raises(haccsr.HaccsrError) as e:
            haccsr.hacc_sr_subcycle(ctx, d[0], d[1], d[2], None, d[3], d[4], d[5],
                                    case.get("eps", 0.1), case.get("r_max", 3.0),
                                    case.get("poly", POLY), 0.01, 3, *acc)
        assert e.value.status == haccsr.EINVAL, case
        haccsr.haccsr_sync(ctx)
        for t, h in zip(d, host):
            assert np.array_equal(t.cpu().numpy(), h), case


# ------------------------------------------------------------------ randomised sweep
@pytest.mark.parametrize("seed", range(10))
def test_random_problem_sweep(seed):
    """Random small problems: box length, mesh, cutoff (r_max <= L/nc, sometimes equal),
    softening, masses on/off, clustering, out-of-box inputs; counts bit-exact, accelerations
    within tolerance, mesh equal to the oracle's."""
    rng = np.random.default_rng(1000 + seed)
    nc = int(rng.integers(4, 24))
    w = float(rng.choice([3.0, 3.2, 3.75, 5.0]))
    L = float(np.float32(nc * w))
    r_max = float(np.float32(w if seed % 3 == 0 else rng.uniform(0.5 * w, w)))
    while L / nc < r_max:                       # float32 rounding of L
        r_max = float(np.nextafter(np.float32(r_max), np.float32(0)))
    eps = float(rng.choice([0.01, 0.1, 0.5]))
    n = int(rng.integers(200, 20000))
    x, y, z = ((rng.random(n) * L).astype(np.float32) for _ in range(3))
    k = n // 3                                   # a clump spanning a few cells
    c = rng.random(3) * L
    for a, c0 in zip((x, y, z), c):
        a[:k] = np.mod(c0 + rng.standard_normal(k) * 1.5, L).astype(np.float32)
        a[a >= L] = 0
    m = rng.uniform(0.25, 4.0, n).astype(np.float32) if seed % 2 else None
    xo = x.copy()
    if seed % 4 == 1:                            # some inputs outside the box: they wrap (S16)
        xo[: n // 10] += np.float32(L)
        x = O.drift(xo, np.zeros(n, np.float32), 0.0, L).astype(np.float32)
        x[x >= L] = 0
    ref = O.sr_celllist(x, y, z, m, L, nc, r_max, eps, POLY)
    out, ctx = H.gpu_step(xo, y, z, L, nc, r_max=r_max, eps=eps, mass=m)
    ref_mesh = O.mesh(x, y, z, L, nc)
    mesh = haccsr.haccsr_get_mesh(ctx)
    assert np.array_equal(mesh["cell_start"].cpu().numpy().astype(np.uint32),
                          ref_mesh["cell_start"])
    assert np.array_equal(mesh["cell_id"].cpu().numpy().astype(np.uint32), ref_mesh["cid"])
    assert np.array_equal(out["nbr"], ref["nbr"]), (nc, L, r_max, eps, n)
    assert out["C"] == ref["C"]
    if ref["C"] > 0:
        H.assert_accel_parity(out, ref)


def test_two_contexts_interleaved_on_different_streams():
    """Two contexts of different meshes, each on its own stream, used alternately (state,
    kernel configuration and the cached CUDA graphs are per context): both must give the
    oracle's result, twice (the second round replays the captured graphs)."""
    rng = np.random.default_rng(55)
    probs = []
    for n, L, nc in ((30000, 32.0, 10), (50000, 48.0, 15)):
        x, y, z = ((rng.random(n) * L).astype(np.float32) for _ in range(3))
        k = n // 4
        for a in (x, y, z):
            a[:k] = np.mod(L / 3 + rng.standard_normal(k) * 1.0, L).astype(np.float32)
            a[a >= L] = 0
        st = torch.cuda.Stream()
        ctx = haccsr.Context(n, L, nc, stream=st)
        ref = O.sr_celllist(x, y, z, None, L, nc, 3.0, 0.1, POLY)
        with torch.cuda.stream(st):
            d = [H.to_dev(a) for a in (x, y, z)]
            acc = [torch.empty(n, dtype=torch.float32, device="cuda:0") for _ in range(3)]
            nbr = torch.empty(n, dtype=torch.int32, device="cuda:0")
        probs.append((ctx, st, d, acc, nbr, ref))
    torch.cuda.synchronize()
    for _ in range(2):
        for ctx, st, d, acc, nbr, ref in probs:          # enqueue both before either is read
            with torch.cuda.stream(st):
                haccsr.hacc_sr_bin(ctx, *d)
                haccsr.hacc_sr_force(ctx, 0.1, 3.0, POLY, *acc, nbr, None)
        for ctx, st, d, acc, nbr, ref in probs:
            haccsr.haccsr_sync(ctx)
            assert np.array_equal(nbr.cpu().numpy().view(np.uint32), ref["nbr"])
            out = dict(ax=acc[0].cpu().numpy(), ay=acc[1].cpu().numpy(), az=acc[2].cpu().numpy())
            H.assert_accel_parity(out, ref)
