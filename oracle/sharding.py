"""Oracle restatement of HACC's particle overloading for the short-range force.
TEST INFRASTRUCTURE ONLY (see sr_oracle.c header): only tests/ may import this.

PAPER.md:112-122 (section 2.2): the box is split into spatial domains; "particles close to the
boundaries of their domain are replicated" in the neighbouring domains.  The copies are
PASSIVE: they act as sources for the domain's own (ACTIVE) particles, and "passive particles
near the outer edge get no short-range force"; after the replication the short-range step
needs no communication.  PAPER.md:388-394 (Fig. 13): the same idea one level down, device
blocks with r_s-wide boundary slabs.

Restated plainly: cut the chaining mesh into slabs of whole cell layers along z.  Slab s owns
the particles whose layer cz = floor(z nc / L) lies in [lo_s, lo_s + nz_s); its passive
particles are those of the two adjacent layers (periodic).  Every slab evaluates the plain
all-pairs definition (oracle_sr_brute, minimum image in the FULL box, positions unshifted)
with its active particles as targets and active + passive particles as sources.  Because a
layer is at least r_max wide, every neighbour of an active particle is inside the slab's
window, so the union over slabs must equal the whole-box result: identical n_i, and
accelerations equal up to FP64 summation order.  That equality is the pin
(tests/test_oracle_pins.py), checked against oracle_sr_brute on the whole box.
"""
from __future__ import annotations

import numpy as np

from . import sr_oracle as O


def slab_layers(nc: int, n_slabs: int):
    """[(cz_lo, nz_own)] for n_slabs slabs of whole layers, as even as possible."""
    if n_slabs < 1 or (n_slabs > 1 and nc // n_slabs < 1):
        raise ValueError("too many slabs")
    edges = [(s * nc) // n_slabs for s in range(n_slabs + 1)]
    out = [(edges[s], edges[s + 1] - edges[s]) for s in range(n_slabs)]
    if n_slabs > 1 and max(nz for _, nz in out) > nc - 2:
        raise ValueError("a slab and its two passive layers must fit the box")
    return out


def layer_of(z, box_l: float, nc: int):
    """Global cell layer of every particle, from the oracle's own mesh (reading S12)."""
    zz = np.ascontiguousarray(z, dtype=np.float32)
    zero = np.zeros_like(zz)
    cid = O.mesh(zero, zero, zz, box_l, nc)["cid"]
    return (cid // np.uint32(nc * nc)).astype(np.int64)


def slab_members(cz, nc: int, cz_lo: int, nz_own: int):
    """(indices of the slab's active particles, indices of its passive particles)."""
    rel = (cz - cz_lo) % nc
    active = np.nonzero(rel < nz_own)[0]
    passive = np.nonzero((rel == nc - 1) | (rel == nz_own))[0]
    return active, passive


def sr_sharded(x, y, z, m, box_l, nc, r_max, eps, poly, n_slabs):
    """Union of the per-slab evaluations.  Returns dict(ax, ay, az, nbr, C, n_passive)."""
    n = len(x)
    cz = layer_of(z, box_l, nc)
    ax, ay, az = np.zeros(n), np.zeros(n), np.zeros(n)
    nbr = np.zeros(n, dtype=np.uint32)
    owner = np.full(n, -1, dtype=np.int64)
    total, n_passive = 0, []
    for s, (lo, nz_own) in enumerate(slab_layers(nc, n_slabs)):
        if n_slabs == 1:
            act, pas = np.arange(n), np.zeros(0, dtype=np.int64)
        else:
            act, pas = slab_members(cz, nc, lo, nz_own)
        sub = np.concatenate([act, pas])
        r = O.sr_brute(x[sub], y[sub], z[sub], None if m is None else m[sub], box_l, r_max, eps,
                       poly, targets=np.arange(len(act)))
        assert np.all(owner[act] == -1)
        owner[act] = s
        ax[act], ay[act], az[act], nbr[act] = r["ax"], r["ay"], r["az"], r["nbr"]
        total += r["C"]
        n_passive.append(len(pas))
    assert np.all(owner >= 0)  # every particle is active in exactly one slab
    return dict(ax=ax, ay=ay, az=az, nbr=nbr, C=total, n_passive=n_passive, owner=owner)
