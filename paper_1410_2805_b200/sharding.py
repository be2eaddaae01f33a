"""Overloaded multi-GPU sharding of the short-range step.

One process per GPU.  The global chaining mesh is cut into slabs of whole cell layers along
z; rank r owns the particles of its layers and, every step, receives passive copies of the
two adjacent layers (one from each neighbour, periodic): ONE neighbour exchange, no
reduction, after which every rank runs the unchanged single-GPU path on a slab context
(haccsr_create_slab) and kicks only its own particles.

This module is host logic only: integer slab bounds, buffer bookkeeping and the
torch.distributed plumbing of the exchange.  Selecting a layer's particles
(hacc_sr_pack_layer), appending received records (hacc_sr_unpack) and everything else that
touches particle data runs in the library's kernels.  Positions are never shifted: the slab
context works in global box coordinates, so the rank that owns the layer across the periodic
boundary just sends it as it is.
"""
from __future__ import annotations

import torch

from . import haccsr


def slab_layers(nc: int, world: int):
    """[(cz_lo, nz_own)] per rank: whole layers, as even as possible."""
    if world < 1 or nc // world < 1:
        raise ValueError("more ranks than cell layers")
    edges = [(r * nc) // world for r in range(world + 1)]
    out = [(edges[r], edges[r + 1] - edges[r]) for r in range(world)]
    if world > 1 and max(nz for _, nz in out) > nc - 2:
        raise ValueError("a slab and its two passive layers must fit the box (nc too small)")
    return out


def slab_layers_balanced(work, world: int):
    """[(cz_lo, nz_own)] per rank for slabs of EQUAL WORK instead of equal thickness.

    `work[cz]` >= 0 is the cost of layer cz (for the short-range force: its candidate pairs,
    sum over the layer's cells of n_c * S_c, see `layer_work`).  Contiguous slabs starting at
    layer 0, every slab at least one layer and (for world > 1) at most nc - 2 (a slab and its
    two passive layers must fit the box), chosen so that the LARGEST slab work is minimal:
    bisection on that bound with a greedy fill, then the greedy cut for the smallest feasible
    bound.  With clustered particles the slowest slab bounds the step (PAPER.md:386-394 moves
    boundary slabs between devices for the same reason); integer work gives identical cuts
    on every rank."""
    w = [int(v) for v in work]
    nc = len(w)
    if world < 1 or nc // world < 1:
        raise ValueError("more ranks than cell layers")
    if min(w) < 0:
        raise ValueError("negative work")
    if world == 1:
        return [(0, nc)]
    max_len = nc - 2
    if -(-nc // world) > max_len:
        raise ValueError("a slab and its two passive layers must fit the box (nc too small)")

    def greedy(bound, lo=0, r0=0):
        """Edges after `lo` when each slab from r0 on takes layers while its work stays <= bound,
        its length <= max_len and enough layers remain for the slabs after it; None if a
        slab overflows the bound or the layers do not run out exactly."""
        edges = []
        for r in range(r0, world):
            left = world - r - 1                      # slabs still to come
            # at least enough that the rest can cover what remains with max_len each
            need = max(1, (nc - lo) - left * max_len)
            hi, acc = lo, 0
            while hi < nc - left and hi - lo < max_len:
                if hi - lo >= need and acc + w[hi] > bound:
                    break
                acc += w[hi]
                hi += 1
            if hi == lo or acc > bound:
                return None
            edges.append(hi)
            lo = hi
        return edges if lo == nc else None

    lo_b, hi_b = max(w), sum(w)
    if greedy(hi_b) is None:                          # cannot happen for valid input
        raise ValueError("no valid slab decomposition")
    while lo_b < hi_b:
        mid = (lo_b + hi_b) // 2
        if greedy(mid) is None:
            lo_b = mid + 1
        else:
            hi_b = mid
    bound = hi_b
    # among the decompositions that meet the bound, an even one: every slab stops as soon as it
    # holds its share of the work that is left, provided the slabs after it can still meet
    # the bound (the plain greedy fill would leave the last slab nearly empty)
    edges, lo = [0], 0
    for r in range(world - 1):
        left = world - r - 1
        need = max(1, (nc - lo) - left * max_len)
        share = -(-sum(w[lo:]) // (left + 1))
        hi, acc, pick = lo, 0, None
        while hi < nc - left and hi - lo < max_len:
            if hi - lo >= need and acc + w[hi] > bound:
                break
            acc += w[hi]
            hi += 1
            if hi - lo >= need and greedy(bound, hi, r + 1) is not None:
                pick = hi
                if acc >= share:
                    break
        edges.append(pick)
        lo = pick
    edges.append(nc)
    return [(edges[r], edges[r + 1] - edges[r]) for r in range(world)]


def layer_work(x, y, z, box_l: float, nc: int):
    """Candidate pairs of the short-range force per cell layer cz, as a list of nc ints:
    sum over the layer's cells of n_c * S_c, S_c the particles of the 27 neighbouring cells
    (periodic).  An ESTIMATE for `slab_layers_balanced`: the cell index here is plain float32
    arithmetic, not the library's exact floor (a particle on a cell face may land next door).
    x, y, z: torch tensors (any device)."""
    scale = float(nc) / float(box_l)

    def coord(t):
        return (t * scale).floor().clamp_(0, nc - 1).to(torch.int64)

    cid = (coord(z) * nc + coord(y)) * nc + coord(x)
    cnt = torch.bincount(cid, minlength=nc ** 3).reshape(nc, nc, nc)
    del cid
    s = torch.zeros_like(cnt)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                s += torch.roll(cnt, (dz, dy, dx), (0, 1, 2))
    return [int(v) for v in (cnt * s).sum(dim=(1, 2)).tolist()]


def neighbours(rank: int, world: int):
    """(rank owning the layer below my slab, rank owning the layer above), periodic."""
    return (rank - 1) % world, (rank + 1) % world


def exchange_records(rank, world, send_down, n_down, send_up, n_up, recv_below, recv_above,
                     group=None):
    """The neighbour exchange of one step: `send_down[:4 n_down]` (my lowest layer) goes to the
    rank below, `send_up[:4 n_up]` (my highest layer) to the rank above; the highest layer of
    the rank below arrives in recv_below, the lowest layer of the rank above in recv_above.
    Flat float32 tensors on the process group's device (NCCL: CUDA, gloo: CPU).
    Returns (n_from_below, n_from_above)."""
    import torch.distributed as dist

    below, above = neighbours(rank, world)
    mine = torch.tensor([n_down, n_up], dtype=torch.int32, device=send_down.device)
    allc = torch.empty(2 * world, dtype=torch.int32, device=send_down.device)
    dist.all_gather_into_tensor(allc, mine, group=group)
    allc = allc.view(world, 2).cpu()
    n_from_below, n_from_above = int(allc[below, 1]), int(allc[above, 0])
    if 4 * n_from_below > recv_below.numel() or 4 * n_from_above > recv_above.numel():
        raise RuntimeError("receive buffer too small")
    # order matters when below == above (two ranks): on both sides first everything that
    # travels up, then everything that travels down
    ops = [dist.P2POp(dist.isend, send_up[:4 * n_up], above, group=group, tag=1),
           dist.P2POp(dist.isend, send_down[:4 * n_down], below, group=group, tag=0),
           dist.P2POp(dist.irecv, recv_below[:4 * n_from_below], below, group=group, tag=1),
           dist.P2POp(dist.irecv, recv_above[:4 * n_from_above], above, group=group, tag=0)]
    ops = [op for op in ops if op.tensor.numel() > 0]
    for req in (dist.batch_isend_irecv(ops) if ops else []):
        req.wait()
    return n_from_below, n_from_above


class SlabRank:
    """One rank's slab: context, particle arrays with room for the passive copies, message
    buffers.  `n_cap` = capacity of the particle arrays (own + passive), `msg_cap` = capacity
    of one message in particles."""

    def __init__(self, rank, world, box_l, nc, n_cap, msg_cap, device, with_mass=False,
                 layers=None):
        """layers: the decomposition [(cz_lo, nz_own)] per rank (default: `slab_layers`)."""
        self.rank, self.world = int(rank), int(world)
        self.box_l, self.nc = float(box_l), int(nc)
        self.cz_lo, self.nz_own = (layers or slab_layers(nc, world))[rank]
        self.device = torch.device(device)
        self.n_cap, self.msg_cap = int(n_cap), int(msg_cap)
        slab = None if world == 1 else (self.cz_lo, self.nz_own)
        self.ctx = haccsr.Context(self.n_cap, box_l, nc, device=self.device, slab=slab)
        f = dict(dtype=torch.float32, device=self.device)
        self.x, self.y, self.z = (torch.zeros(self.n_cap, **f) for _ in range(3))
        self.mass = torch.ones(self.n_cap, **f) if with_mass else None
        self.v = [torch.zeros(self.n_cap, **f) for _ in range(3)]
        self.a = [torch.zeros(self.n_cap, **f) for _ in range(3)]
        self.n_own = 0
        self.n_total = 0
        # messages: [0] my lowest layer -> rank below, [1] my highest layer -> rank above
        self.send = [torch.empty(4 * self.msg_cap, **f) for _ in range(2)]
        self.recv = [torch.empty(4 * self.msg_cap, **f) for _ in range(2)]
        self.counts = torch.zeros(2, dtype=torch.int32, device=self.device)

    # -- layers -------------------------------------------------------------------------
    def boundary_layers(self):
        """(global layer sent down, global layer sent up)."""
        return self.cz_lo, (self.cz_lo + self.nz_own - 1) % self.nc

    def pack(self):
        """Enqueue the two selections; returns the device counts tensor (not synchronised)."""
        lo, hi = self.boundary_layers()
        n = self.n_own
        for k, layer in enumerate((lo, hi)):
            haccsr.hacc_sr_pack_layer(self.ctx, self.x, self.y, self.z, self.mass, layer,
                                      self.send[k], self.counts[k:k + 1], n=n)
        return self.counts

    def append(self, records, n):
        """Append n received float4 records as passive particles."""
        if self.n_total + n > self.n_cap:
            raise RuntimeError("particle arrays too small for the passive copies")
        o = self.n_total
        haccsr.hacc_sr_unpack(self.ctx, records, n, self.x[o:], self.y[o:], self.z[o:],
                              None if self.mass is None else self.mass[o:])
        self.n_total += int(n)

    # -- the exchange -------------------------------------------------------------------
    def exchange(self, group=None):
        """Refresh the passive copies: pack, swap records with the two neighbours, unpack.
        Returns (n_from_below, n_from_above)."""
        self.n_total = self.n_own
        if self.world == 1:
            return 0, 0
        n_dn, n_up = (int(v) for v in self.pack().tolist())   # synchronises the stream
        if max(n_dn, n_up) > self.msg_cap:
            raise RuntimeError(f"message buffer too small: {n_dn}, {n_up} > {self.msg_cap}")
        import torch.distributed as dist

        if dist.get_backend(group) == "gloo":
            # a CPU process group (tests on a box with fewer GPUs than ranks): the records
            # travel through host memory; NCCL moves them GPU to GPU over NVLink
            host = [t.cpu() for t in self.send]
            rb, ra = (torch.empty(4 * self.msg_cap) for _ in range(2))
            got = exchange_records(self.rank, self.world, host[0], n_dn, host[1], n_up, rb, ra,
                                   group)
            self.recv[0][:4 * got[0]].copy_(rb[:4 * got[0]])
            self.recv[1][:4 * got[1]].copy_(ra[:4 * got[1]])
        else:
            got = exchange_records(self.rank, self.world, self.send[0], n_dn, self.send[1],
                                   n_up, self.recv[0], self.recv[1], group)
        self.append(self.recv[0], got[0])
        self.append(self.recv[1], got[1])
        return got

    # -- the step -----------------------------------------------------------------------
    def views(self):
        n = self.n_total
        pos = (self.x[:n], self.y[:n], self.z[:n])
        vel = tuple(c[:n] for c in self.v)
        acc = tuple(c[:n] for c in self.a)
        mass = None if self.mass is None else self.mass[:n]
        return pos, mass, vel, acc

    def step(self, eps, r_max, poly, dt, nbr=None, pair_total=None, group=None):
        """exchange -> bin -> force+kick on this rank's slab."""
        self.exchange(group)
        pos, mass, vel, acc = self.views()
        haccsr.hacc_sr_bin(self.ctx, *pos, mass, *vel)
        haccsr.hacc_sr_force_kick(self.ctx, eps, r_max, poly, dt, *acc, nbr, pair_total)


def scatter_to_slab(slab: SlabRank, x, y, z, mass=None):
    """Fill a rank's own particles from arrays holding the WHOLE box (device tensors): one
    hacc_sr_pack_layer per owned layer, then hacc_sr_unpack.  Set-up only (not a step)."""
    n = x.numel()
    buf = torch.empty(4 * slab.msg_cap, dtype=torch.float32, device=slab.device)
    cnt = torch.zeros(1, dtype=torch.int32, device=slab.device)
    slab.n_own = slab.n_total = 0
    for k in range(slab.nz_own):
        layer = (slab.cz_lo + k) % slab.nc
        haccsr.hacc_sr_pack_layer(slab.ctx, x, y, z, mass, layer, buf, cnt, n=n)
        c = int(cnt.item())
        if c > slab.msg_cap:
            raise RuntimeError("layer larger than the message buffer")
        slab.append(buf, c)
    slab.n_own = slab.n_total
    return slab.n_own
