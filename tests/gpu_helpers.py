"""Helpers shared by the -m gpu parity tests: run the CUDA path through the binding and
compare with oracle outputs.  The CUDA path and the oracle only meet here, in tests/."""
from __future__ import annotations

import numpy as np
import torch

from paper_1410_2805_b200 import haccsr
from paper_1410_2805_b200.workloads import DEFAULT_POLY

# north_star tolerance: per-particle acceleration error <= 1e-4 x RMS acceleration on every
# component (FP32 vs FP64).  DESIGN.md reading S17: A_rms = sqrt(mean |a_ref|^2).
TOL_RMS = 1e-4


def to_dev(a, dtype=torch.float32):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0", dtype=dtype)


def gpu_step(x, y, z, box_l, nc, r_max=3.0, eps=0.1, poly=DEFAULT_POLY, mass=None, v=None,
             dt=0.01, count=True, fused=True, n_max=None):
    """bin -> force(+kick) on the GPU.  Returns dict of numpy results and the Context."""
    n = len(x)
    ctx = haccsr.Context(n_max or max(n, 1), box_l, nc)
    dx, dy, dz = to_dev(x), to_dev(y), to_dev(z)
    dm = to_dev(mass) if mass is not None else None
    if v is not None:
        dv = [to_dev(c) for c in v]
    else:
        dv = [None, None, None]
    haccsr.hacc_sr_bin(ctx, dx, dy, dz, dm, *dv)
    ax, ay, az = (torch.empty(max(n, 1), dtype=torch.float32, device="cuda:0") for _ in range(3))
    nbr = torch.empty(max(n, 1), dtype=torch.int32, device="cuda:0") if count else None
    tot = torch.zeros(1, dtype=torch.int64, device="cuda:0") if count else None
    if v is not None and fused:
        haccsr.hacc_sr_force_kick(ctx, eps, r_max, poly, dt, ax, ay, az, nbr, tot)
    else:
        haccsr.hacc_sr_force(ctx, eps, r_max, poly, ax, ay, az, nbr, tot)
        if v is not None:
            haccsr.hacc_sr_kick(ctx, dt)
    haccsr.haccsr_sync(ctx)
    out = dict(ax=ax[:n].cpu().numpy(), ay=ay[:n].cpu().numpy(), az=az[:n].cpu().numpy())
    if count:
        out["nbr"] = nbr[:n].cpu().numpy().view(np.uint32)
        out["C"] = int(tot.item())
    if v is not None:
        out["v"] = [c.cpu().numpy() for c in dv]
    out["stats"] = haccsr.haccsr_get_stats(ctx)
    return out, ctx


def check_mesh(ctx, ref, x, y, z):
    """Bit-exact mesh parity: per-particle cell id, cell_start, per-cell index sets, and the
    sorted float4 rows are the input rows."""
    m = haccsr.haccsr_get_mesh(ctx)
    cid = m["cell_id"].cpu().numpy().astype(np.uint32)
    start = m["cell_start"].cpu().numpy().astype(np.uint32)
    perm = m["perm"].cpu().numpy()
    sp = m["sorted_pos"].cpu().numpy()
    assert np.array_equal(cid, ref["cid"])
    assert np.array_equal(start, ref["cell_start"])
    n = len(x)
    assert np.array_equal(np.sort(perm), np.arange(n))          # a permutation
    # slot s lies in cell of its original particle: cell ids along the sorted order
    # must be non-decreasing and equal to cid[perm]
    sc = ref["cid"][perm]
    assert np.all(np.diff(sc.astype(np.int64)) >= 0)
    slot_cell = np.searchsorted(ref["cell_start"], np.arange(n), side="right") - 1
    assert np.array_equal(slot_cell.astype(np.uint32), sc)
    assert np.array_equal(sp[:, 0], x[perm])
    assert np.array_equal(sp[:, 1], y[perm])
    assert np.array_equal(sp[:, 2], z[perm])
    return m


def accel_errors(out, ref, idx=None):
    """max |a_gpu - a_ref| over particles and components, in units of A_rms of the reference."""
    g = np.stack([out["ax"], out["ay"], out["az"]], 1).astype(np.float64)
    if idx is not None:
        g = g[idx]
    r = np.stack([ref["ax"], ref["ay"], ref["az"]], 1)
    arms = float(np.sqrt(np.mean(np.sum(r * r, axis=1))))
    err = np.abs(g - r)
    mag = np.sqrt(np.sum(r * r, axis=1))
    rel = np.sqrt(np.sum((g - r) ** 2, axis=1)) / np.maximum(mag, 1e-30)
    return dict(arms=arms, max_abs=float(err.max()) if err.size else 0.0,
                max_over_rms=float(err.max() / arms) if err.size and arms > 0 else 0.0,
                median_rel=float(np.median(rel)) if rel.size else 0.0,
                p99_rel=float(np.quantile(rel, 0.99)) if rel.size else 0.0)


def assert_accel_parity(out, ref, idx=None, tol=TOL_RMS):
    e = accel_errors(out, ref, idx)
    assert e["max_over_rms"] <= tol, e
    # the RMS criterion is loose for low-acceleration particles; the typical particle
    # must also agree to FP32 accumulation accuracy
    assert e["median_rel"] <= 2e-5, e
    return e
