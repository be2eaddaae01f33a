"""-m gpu: overloaded slabs (NEXT-2) on ONE GPU.  2, 3 and 4 logical slabs of
the same box run one after another through the C ABI (slab contexts, hacc_sr_pack_layer,
hacc_sr_unpack); the exchange itself is emulated by handing each slab its neighbours' packed
layers (the torch.distributed version of that hand-over is tested on gloo in
tests/test_sharding_host.py).  The union of the slabs must be the whole-box oracle:
neighbour counts and C bit-exact, accelerations within the force tolerance, passive copies
untouched."""
import numpy as np
import pytest
import torch

from oracle import sharding as OS
from oracle import sr_oracle as O
from paper_1410_2805_b200 import haccsr
from paper_1410_2805_b200 import sharding as S
from paper_1410_2805_b200 import workloads as W

import gpu_helpers as H

pytestmark = pytest.mark.gpu
POLY = W.DEFAULT_POLY


def _keys(x, y, z):
    """One sortable key per particle from the raw bits of its float32 position."""
    a = np.stack([x, y, z], 1).astype(np.float32).view(np.uint32).astype(np.uint64)
    return (a[:, 0] << np.uint64(42)) ^ (a[:, 1] << np.uint64(21)) ^ a[:, 2]


def _problem(seed=0, with_mass=False):
    cfg = W.scaled_config(W.CONFIGS[2], 48)      # 110 592 particles, L = 48, nc = 15, 50 % halos
    p = W.make_particles(cfg)
    rng = np.random.default_rng(77 + seed)
    z = p["z"].copy()
    # clumps on a slab face and across the periodic z boundary
    z[:3000] = np.mod(cfg.box_l / 2 + rng.standard_normal(3000) * 0.8, cfg.box_l).astype(np.float32)
    z[3000:6000] = np.mod(rng.standard_normal(3000) * 0.8, cfg.box_l).astype(np.float32)
    z[z >= cfg.box_l] = 0
    m = rng.uniform(0.5, 2.0, cfg.n).astype(np.float32) if with_mass else None
    keys = _keys(p["x"], p["y"], z)
    assert len(np.unique(keys)) == cfg.n          # positions identify particles
    return cfg, p["x"], p["y"], z, m, keys


# the last case: slabs of unequal thickness as `slab_layers_balanced` cuts them, one of them a
# single layer (its window is that layer and the two passive ones)
@pytest.mark.parametrize("n_slabs,with_mass,layers", [
    (2, False, None), (3, True, None), (4, False, None),
    (4, False, [(0, 1), (1, 6), (7, 2), (9, 6)])])
def test_logical_slabs_reproduce_the_whole_box(n_slabs, with_mass, layers):
    cfg, x, y, z, m, keys = _problem(n_slabs, with_mass)
    n, L, nc, dt = cfg.n, cfg.box_l, cfg.nc, 0.01
    whole = O.sr_celllist(x, y, z, m, L, nc, cfg.r_max, cfg.eps, POLY)
    order = np.argsort(keys)
    dx, dy, dz = H.to_dev(x), H.to_dev(y), H.to_dev(z)
    dm = H.to_dev(m) if with_mass else None
    ranks = [S.SlabRank(r, n_slabs, L, nc, n, n // 2, "cuda:0", with_mass=with_mass,
                        layers=layers)
             for r in range(n_slabs)]
    if layers is None:     # and the cuts by work are a valid decomposition of this box too
        bal = S.slab_layers_balanced(S.layer_work(dx, dy, dz, L, nc), n_slabs)
        assert bal[0][0] == 0 and sum(k for _, k in bal) == nc
    for rk in ranks:
        S.scatter_to_slab(rk, dx, dy, dz, dm)
        rk.v[0][:rk.n_own] = 0.25            # a velocity to kick
    assert sum(rk.n_own for rk in ranks) == n
    counts = [rk.pack().tolist() for rk in ranks]
    cz = OS.layer_of(z, L, nc)
    pop = np.bincount(cz, minlength=nc)
    c_total = 0
    seen = np.zeros(n, dtype=int)
    for rk in ranks:
        below, above = S.neighbours(rk.rank, n_slabs)
        rk.n_total = rk.n_own
        rk.append(ranks[below].send[1], counts[below][1])    # its highest layer
        rk.append(ranks[above].send[0], counts[above][0])    # its lowest layer
        assert rk.n_total - rk.n_own == pop[(rk.cz_lo - 1) % nc] + pop[(rk.cz_lo + rk.nz_own) % nc]
        pos, mass, vel, acc = rk.views()
        nbr = torch.empty(rk.n_total, dtype=torch.int32, device="cuda:0")
        tot = torch.zeros(1, dtype=torch.int64, device="cuda:0")
        haccsr.hacc_sr_bin(rk.ctx, *pos, mass, *vel)
        haccsr.hacc_sr_force_kick(rk.ctx, cfg.eps, cfg.r_max, POLY, dt, *acc, nbr, tot)
        haccsr.haccsr_sync(rk.ctx)
        st = haccsr.haccsr_get_stats(rk.ctx)
        assert st.n_cells == nc * nc * (rk.nz_own + 2)
        # which whole-box particle is each local particle
        lx, ly, lz = (c.cpu().numpy() for c in pos)
        g = order[np.searchsorted(keys[order], _keys(lx, ly, lz))]
        assert np.array_equal(x[g], lx) and np.array_equal(z[g], lz)
        own, pas = slice(0, rk.n_own), slice(rk.n_own, rk.n_total)
        seen[g[own]] += 1
        # mesh of the window against the oracle's mesh of the same particles
        mesh = haccsr.haccsr_get_mesh(rk.ctx)
        ref = O.mesh(lx, ly, lz, L, nc)
        cid = ref["cid"].astype(np.int64)
        lzw = (cid // (nc * nc) - (rk.cz_lo - 1)) % nc
        wid = cid % (nc * nc) + nc * nc * lzw
        assert lzw.max() < rk.nz_own + 2
        assert np.array_equal(mesh["cell_id"].cpu().numpy(), wid)
        start = np.concatenate([[0], np.cumsum(np.bincount(wid, minlength=st.n_cells))])
        assert np.array_equal(mesh["cell_start"].cpu().numpy(), start)
        # active particles: the whole-box result
        nb = nbr.cpu().numpy().view(np.uint32)
        assert np.array_equal(nb[own], whole["nbr"][g[own]])
        assert int(tot.item()) == int(whole["nbr"][g[own]].astype(np.int64).sum())
        c_total += int(tot.item())
        out = {k: a.cpu().numpy()[own] for k, a in zip(("ax", "ay", "az"), acc)}
        sub = {k: whole[k][g[own]] for k in ("ax", "ay", "az")}
        r = np.stack([whole[k] for k in ("ax", "ay", "az")], 1)
        arms = float(np.sqrt(np.mean(np.sum(r * r, axis=1))))
        for k in ("ax", "ay", "az"):
            assert np.abs(out[k] - sub[k]).max() <= H.TOL_RMS * arms
        vx = vel[0].cpu().numpy()
        assert np.abs(vx[own] - (0.25 + dt * sub["ax"])).max() <= H.TOL_RMS * arms * dt + 1e-7
        # passive copies: sources only
        assert np.all(nb[pas] == 0)
        for a in acc:
            assert np.all(a.cpu().numpy()[pas] == 0)
        assert np.all(vx[pas] == 0)
    assert np.all(seen == 1)
    assert c_total == whole["C"]


def test_a_particle_outside_the_window_is_reported():
    L, nc = 32.0, 10
    ctx = haccsr.Context(100, L, nc, slab=(2, 3))          # window = layers 1..5
    rng = np.random.default_rng(0)
    x, y = ((rng.random(50) * L).astype(np.float32) for _ in range(2))
    z = (3.2 + rng.random(50) * 5 * 3.2).astype(np.float32) * np.float32(0.999)
    haccsr.hacc_sr_bin(ctx, H.to_dev(x), H.to_dev(y), H.to_dev(z))
    haccsr.haccsr_sync(ctx)                                 # all inside: fine
    z[7] = 0.5                                              # layer 0 is outside
    haccsr.hacc_sr_bin(ctx, H.to_dev(x), H.to_dev(y), H.to_dev(z))
    with pytest.raises(haccsr.HaccsrError) as e:
        haccsr.haccsr_sync(ctx)
    assert e.value.status == haccsr.EDATA


def test_slab_argument_errors_and_pack_overflow():
    with pytest.raises(haccsr.HaccsrError):
        haccsr.Context(100, 32.0, 10, slab=(0, 9))          # 9 + 2 layers do not fit 10
    with pytest.raises(haccsr.HaccsrError):
        haccsr.Context(100, 32.0, 10, slab=(10, 2))
    ctx = haccsr.Context(1000, 32.0, 10, slab=(9, 2))       # wraps: owns layers 9 and 0
    rng = np.random.default_rng(1)
    x, y = ((rng.random(1000) * 32).astype(np.float32) for _ in range(2))
    z = (rng.random(1000) * 3.2).astype(np.float32) * np.float32(0.999)   # all in layer 0
    buf = torch.empty(4 * 100, dtype=torch.float32, device="cuda:0")
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda:0")
    haccsr.hacc_sr_pack_layer(ctx, H.to_dev(x), H.to_dev(y), H.to_dev(z), None, 0, buf, cnt)
    assert int(cnt.item()) == 1000                          # count beyond capacity is reported
    haccsr.hacc_sr_pack_layer(ctx, H.to_dev(x), H.to_dev(y), H.to_dev(z), None, 5, buf, cnt)
    assert int(cnt.item()) == 0
