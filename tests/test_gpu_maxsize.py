"""-m gpu: the largest problem size class the ABI takes -- 2^30 particles on the largest mesh
(nc = 256), 8x configs[3] -- to catch 32-bit index and byte-offset overflows that no
BASELINE.json config reaches.  Inputs are drawn on the device (a host copy would be 12 GB);
the checks are properties that hold at any size plus a brute-force count in float64 for a few
sampled targets, written out here from the definition (pairs with s < r_max^2,
minimum image in the periodic box) on the particles of a z window around each target.

Needs ~100 GB of device memory; skipped on a smaller or busy GPU."""
import pytest
import torch

from paper_1410_2805_b200 import haccsr, workloads as W

pytestmark = pytest.mark.gpu

N_SIDE, NC, R_MAX, EPS = 1024, 256, 3.0, 0.1


def test_two_to_the_thirty_particles():
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 110 * 2 ** 30:
        pytest.skip(f"needs ~100 GB of free device memory, {free / 2 ** 30:.0f} GiB free")
    try:
        _run()
    finally:
        torch.cuda.empty_cache()     # hand the ~100 GB back before the next test


def _run():
    dev, n, L = "cuda:0", N_SIDE ** 3, float(N_SIDE)
    assert n == 2 ** 30 and 0 < haccsr.haccsr_workspace_bytes(n, NC) < 64 * 2 ** 30
    g = torch.Generator(device=dev).manual_seed(2805)
    pos = []
    for _ in range(3):               # uniform: 64 particles per cell of width 4
        t = torch.rand(n, device=dev, generator=g).mul_(L)
        t[t >= L] = 0.0
        pos.append(t)
    # a clump across the periodic corner, so that wrapped neighbours exist in numbers
    m = 200_000
    for t in pos:
        c = torch.randn(m, device=dev, generator=g) * 1.5
        t[:m] = c - L * torch.floor(c / L)
        t[:m][t[:m] >= L] = 0.0
    acc = [torch.empty(n, device=dev) for _ in range(3)]
    nbr = torch.empty(n, dtype=torch.int32, device=dev)
    tot = torch.zeros(1, dtype=torch.int64, device=dev)
    ctx = haccsr.Context(n, L, NC)
    haccsr.hacc_sr_bin(ctx, *pos)
    haccsr.hacc_sr_force(ctx, EPS, R_MAX, W.DEFAULT_POLY, *acc, nbr, tot)
    haccsr.haccsr_sync(ctx)
    st = haccsr.haccsr_get_stats(ctx)
    assert st.n == n and st.n_cells == NC ** 3 and st.n_eval > 27 * 60 * n

    # the mesh: cell_start is a non-decreasing table ending at n, perm a permutation
    mesh = haccsr.haccsr_get_mesh(ctx)
    cs = mesh["cell_start"]
    assert cs.numel() == NC ** 3 + 1 and int(cs[0]) == 0 and int(cs[-1]) == n
    assert bool((cs[1:] >= cs[:-1]).all())
    seen = torch.zeros(n, dtype=torch.int8, device=dev)
    seen[mesh["perm"]] = 1
    assert int(seen.sum(dtype=torch.int64)) == n
    del seen, mesh, cs

    # C is the sum of the neighbour counts; the accelerations are finite and sum to ~0
    c_total = int(tot.item())
    assert c_total == int(nbr.sum(dtype=torch.int64)) and c_total > 100 * n
    arms = float(torch.sqrt(sum((a.double() ** 2).mean() for a in acc)))
    for a in acc:
        assert bool(torch.isfinite(a).all())
        assert abs(float(a.sum(dtype=torch.float64))) <= 1e-6 * n * arms

    # sampled targets against the definition, float64, minimum image
    pick = torch.cat([torch.randint(0, m, (6,), device=dev, generator=g),        # the clump
                      torch.randint(m, n, (10,), device=dev, generator=g)]).tolist()
    for i in pick:
        xi, yi, zi = (float(t[i]) for t in pos)
        dz = (pos[2] - zi).abs_()
        near = torch.nonzero(torch.minimum(dz, L - dz) <= R_MAX + 1e-3).squeeze(1)
        del dz
        s = torch.zeros(near.numel(), dtype=torch.float64, device=dev)
        for t, ti in zip(pos, (xi, yi, zi)):
            d = (t[near].double() - ti).abs_()
            d = torch.minimum(d, L - d)
            s += d * d
        want = int((s < R_MAX * R_MAX).sum()) - 1          # minus the particle itself
        assert int(nbr[i]) == want, (i, int(nbr[i]), want)
