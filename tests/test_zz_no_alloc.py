"""hacc_sr_cell_start_noalloc (include/haccsr.h): the entry point that allocates nothing -- its
per-cell counters sit in a static __device__ array of the library -- against the existing path
(hacc_sr_bin + haccsr_get_mesh), bit-exact (integer work), on calls made one after another so
that a stale scratch array would show.

Collected last on purpose (the file name): the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

from paper_1410_2805_b200 import haccsr, workloads as W

pytestmark = pytest.mark.gpu


def _existing_cell_start(x, y, z, box_l, nc):
    ctx = haccsr.Context(x.numel(), box_l, nc)
    haccsr.hacc_sr_bin(ctx, x, y, z)
    cs = haccsr.haccsr_get_mesh(ctx)["cell_start"].clone()   # int64 copy of the uint32 table
    haccsr.haccsr_sync(ctx)
    return cs


def _noalloc_cell_start(x, y, z, box_l, nc, out):
    haccsr.hacc_sr_cell_start_noalloc(x, y, z, box_l, nc, out)
    torch.cuda.synchronize()
    return out[: nc ** 3 + 1].to(torch.int64)


def _particles(cfg, shift=0.0):
    p = W.make_particles(cfg)
    # shift: positions leave [0, L) on both sides, so the wrap rule is part of the comparison
    return [torch.from_numpy(p[k] + np.float32(shift) * np.float32(s)).cuda()
            for k, s in zip("xyz", (1.0, -1.0, 2.5))]


def test_noalloc_cell_start_matches_bin_on_calls_in_a_row():
    big = W.scaled_config(W.CONFIGS[1], 96)      # 884 736 particles, 31^3 cells, 30 % in halos
    small = W.CONFIGS[0]                         # 32 768 particles, 10^3 cells
    out = torch.full((haccsr.NOALLOC_MAX_NC ** 3 + 1,), -1, dtype=torch.int32, device="cuda")
    calls = [(big, 0.0), (small, 0.0), (big, 37.25), (big, 0.0)]
    inputs = [(cfg, _particles(cfg, sh)) for cfg, sh in calls]
    # the new entry point, back to back: large mesh, small mesh (most counters stale), the
    # large one again with shifted positions, and once more with the first input
    got = []
    for cfg, (x, y, z) in inputs:
        got.append(_noalloc_cell_start(x, y, z, cfg.box_l, cfg.nc, out))
    for (cfg, (x, y, z)), g in zip(inputs, got):
        ref = _existing_cell_start(x, y, z, cfg.box_l, cfg.nc)
        assert ref.numel() == cfg.nc ** 3 + 1
        assert int(g[-1]) == x.numel() and int(g[0]) == 0
        assert torch.equal(g, ref), cfg.name
    assert torch.equal(got[0], got[3])           # same input, same table, whatever ran between


def test_noalloc_largest_mesh_empty_input_and_limit():
    nc, box_l = haccsr.NOALLOC_MAX_NC, 192.0     # the largest mesh the scratch array holds
    g = torch.Generator(device="cuda").manual_seed(20261105)
    n = 300_000
    x, y, z = (torch.rand(n, device="cuda", generator=g) * box_l for _ in range(3))
    out = torch.empty(nc ** 3 + 1, dtype=torch.int32, device="cuda")
    got = _noalloc_cell_start(x, y, z, box_l, nc, out)
    assert torch.equal(got, _existing_cell_start(x, y, z, box_l, nc))
    # no particles: every entry 0, and nothing of the previous call's counts leaks in
    e = torch.empty(0, device="cuda")
    got = _noalloc_cell_start(e, e, e, box_l, nc, out)
    assert int(got.abs().sum()) == 0
    # beyond the stated maximum: refused, nothing written
    out.fill_(-7)
    with pytest.raises(haccsr.HaccsrError) as err:
        haccsr.hacc_sr_cell_start_noalloc(x, y, z, box_l, nc + 1,
                                          torch.empty((nc + 1) ** 3 + 1, dtype=torch.int32,
                                                      device="cuda"))
    assert err.value.status == haccsr.ENOMEM
    st = haccsr.lib().hacc_sr_cell_start_noalloc(n, x.data_ptr(), y.data_ptr(), z.data_ptr(),
                                                 box_l, nc + 1, out.data_ptr(), None)
    assert st == haccsr.ENOMEM
    assert haccsr.lib().hacc_sr_cell_start_noalloc(n, x.data_ptr(), y.data_ptr(), z.data_ptr(),
                                                   box_l, 3, out.data_ptr(), None) == haccsr.EINVAL
    torch.cuda.synchronize()
    assert int((out != -7).sum()) == 0
