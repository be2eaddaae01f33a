"""Host logic of the overloaded sharding (no GPU): slab bounds, and the neighbour exchange on a
world-size-2 and world-size-3 gloo group.  The records are packed on the CPU by the oracle's
layer selection (the product packs with a CUDA kernel; tests/test_gpu_sharding.py covers
that), sent through paper_1410_2805_b200.sharding.exchange_records, and every rank then runs
the oracle on own + received particles: the union must be the whole-box result."""
import itertools
import os
import random
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from oracle import sharding as OS          # noqa: E402
from oracle import sr_oracle as O          # noqa: E402
from paper_1410_2805_b200 import sharding as S   # noqa: E402
from paper_1410_2805_b200 import workloads as W  # noqa: E402


def test_slab_layers_match_the_oracle_restatement_and_validate():
    for nc, k in ((7, 2), (10, 3), (42, 4), (170, 8), (85, 8), (170, 1)):
        assert S.slab_layers(nc, k) == OS.slab_layers(nc, k)
    with pytest.raises(ValueError):
        S.slab_layers(3, 2)     # 2 + 2 passive layers do not fit 3
    with pytest.raises(ValueError):
        S.slab_layers(4, 5)
    assert S.neighbours(0, 4) == (3, 1) and S.neighbours(3, 4) == (2, 0)
    assert S.neighbours(0, 2) == (1, 1)


def _problem():
    cfg = W.scaled_config(W.CONFIGS[1], 24)
    p = W.make_particles(cfg)
    return cfg, p["x"], p["y"], p["z"]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg, x, y, z = _problem()
    cz = OS.layer_of(z, cfg.box_l, cfg.nc)
    lo, nz_own = S.slab_layers(cfg.nc, world)[rank]
    own = np.nonzero((cz - lo) % cfg.nc < nz_own)[0]

    def records(layer):
        i = own[cz[own] == layer]
        r = np.stack([x[i], y[i], z[i], np.ones(len(i), np.float32)], 1).astype(np.float32)
        return torch.from_numpy(r.ravel().copy()), len(i)

    down, n_down = records(lo)
    up, n_up = records((lo + nz_own - 1) % cfg.nc)
    cap = 4 * len(x)
    rb, ra = torch.empty(cap), torch.empty(cap)
    nb, na = S.exchange_records(rank, world, down, n_down, up, n_up, rb, ra)
    got = torch.cat([rb[:4 * nb], ra[:4 * na]]).numpy().reshape(-1, 4)
    # the oracle on own + received: active = own
    sx = np.concatenate([x[own], got[:, 0]])
    sy = np.concatenate([y[own], got[:, 1]])
    sz = np.concatenate([z[own], got[:, 2]])
    r = O.sr_brute(sx, sy, sz, None, cfg.box_l, cfg.r_max, cfg.eps, W.DEFAULT_POLY,
                   targets=np.arange(len(own)))
    q.put((rank, own, r["nbr"], r["ax"], nb, na, np.sort(cz[own][:0]).tolist()))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,port", [(2, 29641), (3, 29643)])
def test_exchange_records_gloo_union_is_the_whole_box(world, port):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    out = [q.get(timeout=300) for _ in range(world)]
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    cfg, x, y, z = _problem()
    whole = O.sr_brute(x, y, z, None, cfg.box_l, cfg.r_max, cfg.eps, W.DEFAULT_POLY)
    cz = OS.layer_of(z, cfg.box_l, cfg.nc)
    pop = np.bincount(cz, minlength=cfg.nc)
    seen = np.zeros(cfg.n, dtype=int)
    for rank, own, nbr, ax, nb, na, _ in out:
        seen[own] += 1
        assert np.array_equal(nbr, whole["nbr"][own])          # bit-exact counts
        assert np.abs(ax - whole["ax"][own]).max() <= 1e-12 * np.abs(whole["ax"]).max()
        lo, nz_own = S.slab_layers(cfg.nc, world)[rank]
        assert nb == pop[(lo - 1) % cfg.nc] and na == pop[(lo + nz_own) % cfg.nc]
    assert np.all(seen == 1)


def _brute_min_max(w, k):
    nc, best = len(w), None
    for cuts in itertools.combinations(range(1, nc), k - 1):
        e = (0,) + cuts + (nc,)
        if max(e[i + 1] - e[i] for i in range(k)) > nc - 2:
            continue
        m = max(sum(w[e[i]:e[i + 1]]) for i in range(k))
        best = m if best is None else min(best, m)
    return best


def test_balanced_slabs_partition_the_mesh_and_minimise_the_largest_slab():
    rng = random.Random(1410)
    checked = 0
    for _ in range(400):
        nc = rng.randint(4, 12)
        k = rng.randint(2, min(nc, 5))
        if -(-nc // k) > nc - 2:
            continue
        w = [rng.choice([0, 1, 2, 5, 50, 1000]) * rng.randint(0, 3) for _ in range(nc)]
        sl = S.slab_layers_balanced(w, k)
        assert sl[0][0] == 0 and sum(n for _, n in sl) == nc
        assert all(1 <= n <= nc - 2 for _, n in sl)
        assert all(sl[i][0] + sl[i][1] == sl[i + 1][0] for i in range(k - 1))
        assert max(sum(w[lo:lo + n]) for lo, n in sl) == _brute_min_max(w, k), (w, k, sl)
        checked += 1
    assert checked > 200
    # uniform work: as even as the plain decomposition; one slab: the whole box
    assert sorted(n for _, n in S.slab_layers_balanced([7] * 170, 8)) == \
        sorted(n for _, n in S.slab_layers(170, 8))
    assert S.slab_layers_balanced([3, 1, 4, 1, 5], 1) == [(0, 5)]
    # a heavy layer gets a slab of its own, thin slabs around it
    sl = S.slab_layers_balanced([1, 1, 1, 100, 1, 1, 1, 1], 3)
    assert (3, 1) in sl
    with pytest.raises(ValueError):
        S.slab_layers_balanced([1, 1, 1], 2)      # 2 + 2 passive layers do not fit 3
    with pytest.raises(ValueError):
        S.slab_layers_balanced([1, -1, 1, 1, 1], 2)


def test_layer_work_counts_candidate_pairs_per_layer():
    cfg = W.scaled_config(W.CONFIGS[2], 24)
    p = W.make_particles(cfg)
    nc, L = cfg.nc, cfg.box_l
    got = S.layer_work(*(torch.from_numpy(p[k]) for k in "xyz"), L, nc)
    cid = [np.clip(np.floor(p[k] * np.float32(nc / L)).astype(np.int64), 0, nc - 1) for k in "xyz"]
    cnt = np.zeros((nc, nc, nc), dtype=np.int64)
    np.add.at(cnt, (cid[2], cid[1], cid[0]), 1)
    ref = []
    for cz in range(nc):
        tot = 0
        for cy in range(nc):
            for cx in range(nc):
                s = sum(cnt[(cz + a) % nc, (cy + b) % nc, (cx + c) % nc]
                        for a in (-1, 0, 1) for b in (-1, 0, 1) for c in (-1, 0, 1))
                tot += int(cnt[cz, cy, cx]) * int(s)
        ref.append(tot)
    assert got == ref and sum(got) > 0
