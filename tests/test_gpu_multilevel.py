"""-m gpu: multi-level time stepping (NEXT-3, Eq. 11) through the C ABI against the
oracle's step-by-step composition."""
import numpy as np
import pytest
import torch

from oracle import sr_oracle as O
from paper_1410_2805_b200 import haccsr
from paper_1410_2805_b200 import workloads as W

import gpu_helpers as H

pytestmark = pytest.mark.gpu
POLY = W.DEFAULT_POLY


def _run(x, y, z, v, m, L, nc, T, d, l_min, l_max):
    n = len(x)
    ctx = haccsr.Context(n, L, nc)
    dp = [H.to_dev(a) for a in (x, y, z)]
    dv = [H.to_dev(a) for a in v]
    da = [torch.zeros(n, dtype=torch.float32, device="cuda:0") for _ in range(3)]
    lev = torch.zeros(n, dtype=torch.uint8, device="cuda:0")
    ev = torch.zeros(1, dtype=torch.int64, device="cuda:0")
    haccsr.hacc_sr_subcycle_multilevel(ctx, *dp, None if m is None else H.to_dev(m), *dv, 0.1, 3.0,
                                       POLY, T, d, l_min, l_max, *da, lev, ev)
    haccsr.haccsr_sync(ctx)
    return ([c.cpu().numpy() for c in dp], [c.cpu().numpy() for c in dv], lev.cpu().numpy(),
            int(ev.item()), [c.cpu().numpy() for c in da])


def _clumpy(seed, n=20000, L=32.0):
    rng = np.random.default_rng(seed)
    x, y, z = ((rng.random(n) * L).astype(np.float32) for _ in range(3))
    k = n // 4
    for a, c0 in zip((x, y, z), (9.0, 20.0, 16.5)):     # one clump over a few cells
        a[:k] = np.mod(c0 + rng.standard_normal(k) * 1.2, L).astype(np.float32)
        a[a >= L] = 0
    v = [(rng.standard_normal(n) * 0.3).astype(np.float32) for _ in range(3)]
    return x, y, z, v


@pytest.mark.parametrize("l_min,l_max,with_mass", [(1, 4, False), (2, 8, True), (4, 4, False)])
def test_multilevel_matches_the_oracle_composition(l_min, l_max, with_mass):
    L, nc, T, d = 32.0, 10, 0.04, 2.0
    x, y, z, v = _clumpy(l_max)
    n = len(x)
    m = np.random.default_rng(3).uniform(0.5, 2.0, n).astype(np.float32) if with_mass else None
    pos_ref, vel_ref, lev_ref, ev_ref = O.subcycle_multilevel(x, y, z, *v, m, L, nc, 3.0, 0.1, POLY,
                                                              T, d, l_min, l_max)
    pos, vel, lev, ev, acc = _run(x, y, z, v, m, L, nc, T, d, l_min, l_max)
    assert np.array_equal(lev, lev_ref)                  # Eq. 11 decides integers: bit-exact
    if l_min < l_max:
        assert len(set(lev.tolist())) >= 2
    # exactly the oracle's target lists were evaluated: the same candidate pairs, plus the
    # targets' self pairs, which the GPU's statistic includes
    self_pairs = sum(2 ** int(k) * int((lev == k).sum()) for k in set(lev.tolist()))
    assert ev == ev_ref + self_pairs
    full = O.subcycle_multilevel(x, y, z, *v, m, L, nc, 3.0, 0.1, POLY, T, d, l_max, l_max)[3]
    if l_min < l_max:
        assert ev_ref < full                                 # fewer evaluations than all-finest
    # state: as for the SKS map, the two sides round their float32 state independently, so a
    # pair within an ulp of the cutoff may interact on one side only (|f_SR(9)| r_max ~ 3e-3)
    a = O.sr_celllist(x, y, z, m, L, nc, 3.0, 0.1, POLY)
    r = np.stack([a["ax"], a["ay"], a["az"]], 1)
    arms = float(np.sqrt(np.mean(np.sum(r * r, axis=1))))
    jump, kicks = 4e-3 * (2.0 if with_mass else 1.0), l_max
    for k in range(3):
        dd = np.abs(pos[k] - pos_ref[k])
        assert np.minimum(dd, L - dd).max() <= 2e-5
        e = np.abs(vel[k] - vel_ref[k])
        dt = T / 1.0
        assert np.quantile(e, 0.99) <= kicks * (H.TOL_RMS * arms * dt / kicks + 2e-7) * 2
        assert e.max() <= H.TOL_RMS * arms * dt * 2 + kicks * 2e-7 + 2 * jump * dt


def test_multilevel_argument_errors_leave_the_state_untouched():
    x, y, z, v = _clumpy(1, n=2000)
    n = len(x)
    ctx = haccsr.Context(n, 32.0, 10)
    a = [torch.zeros(n, dtype=torch.float32, device="cuda:0") for _ in range(3)]
    lev = torch.zeros(n, dtype=torch.uint8, device="cuda:0")
    for kw in (dict(l_min=3), dict(l_max=128), dict(l_min=4, l_max=2), dict(d=0.0), dict(eps=0.0)):
        dp = [H.to_dev(c) for c in (x, y, z)]
        dv = [H.to_dev(c) for c in v]
        with pytest.raises(haccsr.HaccsrError) as e:
            haccsr.hacc_sr_subcycle_multilevel(ctx, *dp, None, *dv, kw.get("eps", 0.1), 3.0, POLY,
                                               0.04, kw.get("d", 20.0), kw.get("l_min", 1),
                                               kw.get("l_max", 4), *a, lev)
        assert e.value.status == haccsr.EINVAL, kw
        haccsr.haccsr_sync(ctx)
        for t, h in zip(dp + dv, [x, y, z] + v):
            assert np.array_equal(t.cpu().numpy(), h)


def test_multilevel_on_a_clustered_config_of_many_tiles():
    """configs[4]'s mixture at 64^3 particles (21^3 cells, rows of thousands of particles in the
    halos): every sort pass runs many tiles, the level-ordered pass 3 several batches per row.
    Levels and the evaluated target lists bit-exact, the state within the map's tolerance."""
    cfg = W.scaled_config(W.CONFIGS[4], 64)
    p = W.make_particles(cfg)
    x, y, z = (p[k] for k in "xyz")
    v = [p[k] for k in ("vx", "vy", "vz")]
    L, nc, T, d, l_min, l_max = cfg.box_l, cfg.nc, 0.04, 20.0, 1, 4
    pos_ref, vel_ref, lev_ref, ev_ref = O.subcycle_multilevel(x, y, z, *v, None, L, nc, cfg.r_max,
                                                              cfg.eps, POLY, T, d, l_min, l_max)
    pos, vel, lev, ev, acc = _run(x, y, z, [c.copy() for c in v], None, L, nc, T, d, l_min, l_max)
    assert np.array_equal(lev, lev_ref) and len(set(lev.tolist())) >= 2
    self_pairs = sum(2 ** int(k) * int((lev == k).sum()) for k in set(lev.tolist()))
    assert ev == ev_ref + self_pairs
    a = O.sr_celllist(x, y, z, None, L, nc, cfg.r_max, cfg.eps, POLY)
    r = np.stack([a["ax"], a["ay"], a["az"]], 1)
    arms = float(np.sqrt(np.mean(np.sum(r * r, axis=1))))
    # velocities: the force tolerance times the kicks' total T; positions: rounding of the
    # 2 l_max streams at |x| < 64 (ulp 7.6e-6) plus the streamed velocity error, T * max|dv|
    # (halo cores: |a| ~ 1e4, a kick of T a ~ 1e2 in float32 on both sides)
    # the largest errors sit in the halo cores, where the force is several times A_rms and a
    # rounding difference of a position changes it at once: the bound on the maximum scales
    # with the largest acceleration, the 99 % quantile with A_rms
    amax = float(np.abs(r).max())
    v_tol = H.TOL_RMS * amax * T * 2 + l_max * 2e-7 + 2 * 4e-3 * T
    for k in range(3):
        dd = np.abs(pos[k] - pos_ref[k])
        dd = np.minimum(dd, L - dd)
        assert np.quantile(dd, 0.999) <= 2e-5 and dd.max() <= 2e-5 + T * v_tol
        e = np.abs(vel[k] - vel_ref[k])
        assert np.quantile(e, 0.99) <= l_max * (H.TOL_RMS * arms * T / l_max + 2e-7) * 2
        assert e.max() <= v_tol
