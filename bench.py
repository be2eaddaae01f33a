"""bench.py -- one JSON line for the short-range force path on N B200s of one node.

A "step" is one pass of the whole hot path over one synthetic particle set already resident in
HBM: hacc_sr_bin (cell index + histogram, scan, scatter, work list) followed by
hacc_sr_force_kick (force kernel with the kick fused into its epilogue) -- SURVEY.md section
8(a) rows a1-a6.  Default workload: BASELINE.json configs[3] (512^3 particles, L = 512,
170^3 cells, 40 % in Plummer halos), the configuration north_star's target is quoted on; it
fits one GPU (about 10 GB).  `--config i` selects another BASELINE.json config.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config i] [--impl reference]

With --gpus N > 1 (launched by torchrun, one rank per GPU) ONE box is sharded over the ranks
as overloaded z slabs: every step exchanges one
passive cell layer with each neighbour rank, then runs the unchanged single-GPU path on the
slab; "scaling": "strong".  The slabs hold equal work (candidate pairs), not equal numbers of
layers (--even-slabs: equal thickness).  --replicas runs N independent boxes instead.

Two side modes, each one JSON line of its own (not the headline metric): --slab-sim N runs
the N slabs of the sharded box one after another on ONE GPU and prints the strong scaling
their times predict; --long-range times hacc_lr_force (the PM force, libhaccpm.so).

--impl reference times the CPU oracle (oracle/, FP64 cell list, as it stands) on a bounded
sample of the same workload on this box's host cores; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

# dram__bytes_read.sum + dram__bytes_write.sum of one force evaluation (k_force<0,0> +
# k_force_sparse<0,0>) of this build per config, from the ncu captures summarised in
# profiles/r02_force_dram.md (bytes per launch; configs[4]: one of its five sub-cycles)
FORCE_TRAFFIC_BYTES = {
    0: (1.62e6, "profiles/r02_force_dram.md (k_force alone: 1.6 MB read, nothing written back: "
                "the problem lives in L2)"),
    1: (185.4e6, "profiles/r02_force_dram.md (k_force 75.7 MB read + 9.5 MB written, "
                 "k_force_sparse 85.2 + 15.0 MB)"),
    2: (10.93e9, "profiles/r02_force_dram.md (k_force 2.93 GB read + 1.41 GB written, "
                 "k_force_sparse 4.62 + 1.98 GB)"),
    3: (105.39e9, "profiles/r02_force_dram.md (k_force 25.95 GB read + 9.99 GB written, "
                  "k_force_sparse 52.01 + 17.43 GB)"),
    4: (10.93e9, "profiles/r02_force_dram.md (one sub-cycle: k_force 2.93 GB read + 1.43 GB "
                 "written, k_force_sparse 4.60 + 1.96 GB)"),
}
FLOPS_PER_PAIR = 30.0        # canonical op count per evaluated pair
FP32_LANES_PER_SM = 128      # B200 SM: 4 sub-partitions x 32 FP32 lanes, FMA = 2 flops
BIN_BYTES_PER_PARTICLE = 44  # 12 r (hist) + 12 r + 16 w + 4 w (scatter)
METRIC = "short-range pair interactions/s"
UNIT = "pairs/s"


def measured_hbm_gbs():
    """HBM copy bandwidth: MEASURED_PEAKS.json (driver-written) or the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index (0-4)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=15.0,
                    help="target CPU time of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--replicas", action="store_true",
                    help="with N > 1 ranks: N independent boxes instead of one sharded box")
    ap.add_argument("--even-slabs", action="store_true",
                    help="with N > 1 ranks: slabs of equal thickness instead of equal work")
    ap.add_argument("--slab-sim", type=int, default=0, metavar="N",
                    help="ONE GPU: run the N slabs of the sharded box one after another and "
                         "print the strong scaling their times predict (no exchange)")
    ap.add_argument("--long-range", action="store_true",
                    help="time hacc_lr_force (the PM force, SURVEY.md section 8(f) NEXT-4b) on the "
                         "config's particles instead of the short-range step; one GPU")
    return ap.parse_args()


def workload_name(cfg):
    return (f"configs[{cfg.index}]: {cfg.n_side}^3={cfg.n} particles, L={cfg.box_l:g}, "
            f"{cfg.nc}^3 cells, {int(round(cfg.f_halo * 100))}% in Plummer halos, "
            f"r_max={cfg.r_max:g}, eps={cfg.eps:g}, " +
            (f"one bin + force+kick step dt={cfg.dt:g}" if cfg.n_sub == 1 else
             f"{cfg.n_sub} sub-cycles of drift + bin + force+kick, dt={cfg.dt:g}, "
             f"Gaussian velocities sigma={cfg.sigma_v:g}"))


# --------------------------------------------------------------------------------------------
# clocks during the timed region (nvml, 100 ms period)
# --------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown",
               0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.power = [], set(), []
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                try:
                    bits = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    bits = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for b, name in self.REASONS.items():
                    if bits & b:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.1)

    def start(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples),
                "power_w_max": max(self.power) if self.power else None}


# --------------------------------------------------------------------------------------------
# the CPU oracle, timed (cpu_baseline leg and --impl reference): test infrastructure run on
# the host cores, never on the product path
# --------------------------------------------------------------------------------------------
def oracle_sample(cfg, p, n_targets, seed=2805):
    """FP64 cell-list oracle on `n_targets` random targets of the workload.
    Returns (interacting pairs found, evaluation seconds, list-build seconds, evaluated)."""
    from oracle import sr_oracle as O
    from paper_1410_2805_b200.workloads import DEFAULT_POLY

    rng = np.random.default_rng(seed)
    t = rng.choice(cfg.n, size=min(n_targets, cfg.n), replace=False)
    r = O.sr_celllist(p["x"], p["y"], p["z"], None, cfg.box_l, cfg.nc, cfg.r_max, cfg.eps,
                      DEFAULT_POLY, want_force=True, targets=np.sort(t))
    return r["C"], r["seconds"][1], r["seconds"][0], r["n_eval"]


def cpu_baseline(cfg, p, target_seconds):
    from oracle import sr_oracle as O

    cores = O.num_threads()
    # pilot to size the sample, then the timed sample
    n0 = min(cfg.n, 2048)
    c0, t0, tb0, _ = oracle_sample(cfg, p, n0, seed=1)
    n1 = int(min(cfg.n, max(n0, n0 * target_seconds / max(t0, 1e-3))))
    c1, t1, tb1, ev1 = oracle_sample(cfg, p, n1)
    return {"value": c1 / t1, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": (f"oracle.sr_celllist (FP64 linked-list cell list, OpenMP) on {n1} random "
                       f"targets of the same particle set: {c1} interacting pairs, {ev1} "
                       f"evaluated pairs in {t1:.2f} s (+{tb1:.2f} s linked-list build over all "
                       f"{cfg.n} particles, not counted)"),
            "evaluated_pairs_per_s": ev1 / t1,
            "ns_per_particle_step_extrapolated": t1 / n1 * 1e9}


def run_reference(args):
    """--impl reference: the oracle as it stands, K steps of a bounded sample each."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import sr_oracle as O
    from paper_1410_2805_b200 import workloads as W

    cfg = W.CONFIGS[args.config]
    p = W.make_particles(cfg)
    n_t = min(cfg.n, 8192)
    for _ in range(args.warmup):
        oracle_sample(cfg, p, min(n_t, 1024))
    pairs = secs = 0.0
    evals = 0
    wall0 = time.time()
    for _ in range(args.steps):
        c, t, _, ev = oracle_sample(cfg, p, n_t)
        pairs += c
        secs += t
        evals += ev
    wall = time.time() - wall0
    v = pairs / secs
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * wall / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": workload_name(cfg)},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
                         "sample": (f"each step: oracle.sr_celllist on {n_t} random targets of the "
                                    f"workload ({evals // args.steps} evaluated pairs/step); rate "
                                    f"uses the evaluation time, the per-call linked-list build "
                                    f"over all particles is in ms_per_step only")},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------
# the CUDA path
# --------------------------------------------------------------------------------------------
def max_over_ranks(ms: float, world: int, device) -> float:
    """Slowest rank's time (the contract: multi-GPU numbers are the max over ranks)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist

    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def kernels_per_step(n: int, nc: int) -> int:
    """Kernels of this repo launched by one hacc_sr_bin + hacc_sr_force_kick (whole box)."""
    rows = 1 if nc * nc < 1024 else 4            # (scan x 3 +) k_sort_setup
    items = 1 if nc ** 3 <= 2047 else 5          # k_items_small | k_item_count, scan x 3, k_emit_items
    binning = 5 + rows + items                   # k_count_rows, k_part_z, k_part_y, k_sort_rows, k_cell_sources
    force = 2 + (1 if n >= (1 << 20) else 0)     # k_zero_outputs, k_force (, k_force_sparse)
    return binning + force


def whole_job_rate(units_per_rank: float, world: int, seconds_per_step: float) -> float:
    """Replicas only: every rank processes the same number of units per step."""
    return world * units_per_rank / seconds_per_step


def run_sharded(args):
    """--gpus N > 1: STRONG scaling of one box over N overloaded slabs (
    DESIGN.md section 8).  Every step: exchange of the passive layers with the two neighbour
    ranks (pack kernels, send/recv, unpack kernel), bin, force+kick on the slab context."""
    import torch
    import torch.distributed as dist

    from paper_1410_2805_b200 import haccsr, sharding
    from paper_1410_2805_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    backend = os.environ.get("HACCSR_BENCH_BACKEND", "nccl")   # gloo: ranks sharing one GPU (tests)
    ndev = torch.cuda.device_count()
    dev = torch.device("cuda", local % ndev)
    torch.cuda.set_device(dev)
    if backend == "nccl":
        dist.init_process_group("nccl", device_id=dev)
    else:
        dist.init_process_group(backend)

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    cfg = W.CONFIGS[args.config]
    if cfg.n_sub != 1:
        raise SystemExit("bench.py: the sharded run supports the single-step configs (0-3)")
    p = W.make_particles(cfg)          # every rank draws the same box and keeps its slab
    n, poly = cfg.n, W.DEFAULT_POLY
    # set-up (untimed): the whole box on the device once, this rank's layers selected by the
    # library's own cell index (hacc_sr_pack_layer), the rest dropped
    full = [torch.from_numpy(p[k]).to(dev) for k in "xyz"]
    probe = haccsr.Context(1, cfg.box_l, cfg.nc, device=dev)
    cnt = torch.zeros(1, dtype=torch.int32, device=dev)
    dummy = torch.empty(4, dtype=torch.float32, device=dev)
    # slabs of equal WORK (candidate pairs per layer) unless --even-slabs: with halos the
    # slowest slab bounds the step; every rank derives the same cuts from the same box
    layers = sharding.slab_layers(cfg.nc, world) if args.even_slabs else \
        sharding.slab_layers_balanced(sharding.layer_work(*full, cfg.box_l, cfg.nc), world)
    lo, nz_own = layers[rank]
    pop = []
    for k in range(-1, nz_own + 1):    # my layers and the two passive ones: counts only
        haccsr.hacc_sr_pack_layer(probe, *full, None, (lo + k) % cfg.nc, dummy, cnt)
        pop.append(int(cnt.item()))
    n_own, msg_cap = sum(pop[1:-1]), int(max(pop) * 1.05) + 1024
    n_cap = n_own + pop[0] + pop[-1] + 4096
    slab = sharding.SlabRank(rank, world, cfg.box_l, cfg.nc, n_cap, msg_cap, dev, layers=layers)
    assert sharding.scatter_to_slab(slab, *full) == n_own
    del full, probe
    torch.cuda.empty_cache()

    ev = lambda: torch.cuda.Event(enable_timing=True)
    # C and N_eval of this rank's active particles once, outside the timed region
    tot = torch.zeros(1, dtype=torch.int64, device=dev)
    slab.step(cfg.eps, cfg.r_max, poly, cfg.dt, None, tot)
    haccsr.haccsr_sync(slab.ctx)
    st = haccsr.haccsr_get_stats(slab.ctx)
    mine = torch.tensor([float(tot.item()), float(st.n_eval - slab.n_own), float(slab.n_total)],
                        dtype=torch.float64, device=dev)
    sums = mine.clone()
    dist.all_reduce(sums)
    pairs_c, n_eval, n_with_copies = (int(v) for v in sums.tolist())
    for c in slab.v:
        c.zero_()
    for _ in range(args.warmup):
        slab.step(cfg.eps, cfg.r_max, poly, cfg.dt)
    haccsr.haccsr_sync(slab.ctx)

    marks = [[ev() for _ in range(4)] for _ in range(args.steps)]
    clocks = ClockSampler(dev.index)
    barrier()
    clocks.start()
    t0, t1 = ev(), ev()
    t0.record()
    for k in range(args.steps):
        marks[k][0].record()
        slab.exchange()
        marks[k][1].record()
        pos, mass, vel, acc = slab.views()
        haccsr.hacc_sr_bin(slab.ctx, *pos, mass, *vel)
        marks[k][2].record()
        haccsr.hacc_sr_force_kick(slab.ctx, cfg.eps, cfg.r_max, poly, cfg.dt, *acc, None, None)
        marks[k][3].record()
    t1.record()
    barrier()
    clk = clocks.stop()
    elapsed_ms = max_over_ranks(t0.elapsed_time(t1), world, dev)
    part = [float(np.mean([marks[k][j].elapsed_time(marks[k][j + 1]) for k in range(args.steps)]))
            for j in range(3)]
    exch_ms, bin_ms, force_ms = (max_over_ranks(v, world, dev) for v in part)

    # end to end with HOST buffers: this rank's own particles up, kicked velocities down
    no = slab.n_own
    host = [t[:no].cpu().pin_memory() for t in (slab.x, slab.y, slab.z, *slab.v)]
    out_host = [torch.empty(no, dtype=torch.float32).pin_memory() for _ in range(3)]
    e2e_steps = max(1, min(args.steps, 5))

    def e2e_run(k):
        for _ in range(k):
            for dst, src in zip((slab.x, slab.y, slab.z, *slab.v), host):
                dst[:no].copy_(src, non_blocking=True)
            slab.step(cfg.eps, cfg.r_max, poly, cfg.dt)
            for o, v in zip(out_host, slab.v):
                o.copy_(v[:no], non_blocking=True)

    e2e_run(1)
    barrier()
    s0, s1 = ev(), ev()
    s0.record()
    e2e_run(e2e_steps)
    s1.record()
    barrier()
    e2e_ms = max_over_ranks(s0.elapsed_time(s1), world, dev)
    own_max = max_over_ranks(float(no), world, dev)
    if rank != 0:
        dist.destroy_process_group()
        return
    n_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    hbm_peak, hbm_src = measured_hbm_gbs()
    max_mhz = clk["sm_max_mhz"] or 1965.0
    peak_tflops = n_sms * FP32_LANES_PER_SM * 2 * max_mhz * 1e6 / 1e12
    step_s = elapsed_ms * 1e-3 / args.steps
    # the force launch of the slowest rank evaluates about n_eval / world pairs; the chip-level
    # figure of one GPU: (n_eval / world) / force time of the slowest rank
    achieved = FLOPS_PER_PAIR * (n_eval / world) / (force_ms * 1e-3) / 1e12
    line = {
        "metric": METRIC, "value": pairs_c / step_s, "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * step_s,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": workload_name(cfg),
                   "parallelism": f"{world} overloaded z slabs of whole cell layers "
                                  f"({'equal thickness' if args.even_slabs else 'equal work'}: "
                                  f"{[nz for _, nz in layers]} layers), one passive "
                                  f"layer exchanged with each neighbour per step ({backend})",
                   "l2": "inputs larger than L2" if n * 24 / world > 126e6 else
                         "inputs smaller than L2",
                   "particles_with_passive_copies": n_with_copies,
                   "largest_slab_particles": int(own_max)},
        "interacting_pairs": pairs_c, "evaluated_pairs": n_eval,
        "evaluated_pairs_per_s": n_eval / step_s,
        "ns_per_particle_step": step_s / n * 1e9,
        "exchange_ms": exch_ms, "bin_ms": bin_ms, "force_kick_ms": force_ms,
        "roofline": {"bound": "alu", "kernel": "k_force (slowest rank, mean share of the pairs)",
                     "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                     "frac": achieved / peak_tflops, "traffic": None,
                     "peak_source": (f"derived: {n_sms} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 "
                                     f"x {max_mhz:g} MHz (clocks.max.sm)"),
                     "flops_per_pair": FLOPS_PER_PAIR, "pairs_per_launch": n_eval / world},
        "clocks": clk,
        "e2e": {"value": pairs_c / (e2e_ms * 1e-3 / e2e_steps), "unit": UNIT,
                "h2d_bytes_per_step": 24 * n, "d2h_bytes_per_step": 12 * n,
                "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps},
        # per rank and step: 2 packs + 2 unpacks, then the kernels of bin + force
        "gpu_launches": (4 + kernels_per_step(n // world, cfg.nc)) * args.steps * world,
    }
    print(json.dumps(line), flush=True)
    dist.destroy_process_group()


def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_1410_2805_b200 import haccsr
    from paper_1410_2805_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = W.CONFIGS[args.config]
    p = W.make_particles(cfg)          # every rank: an independent replica of the same box
    n = cfg.n
    poly = W.DEFAULT_POLY
    ctx = haccsr.Context(n, cfg.box_l, cfg.nc, device=dev)
    host = {k: torch.from_numpy(p[k]).pin_memory() for k in ("x", "y", "z", "vx", "vy", "vz")}
    d = {k: host[k].to(dev, non_blocking=True) for k in host}
    acc = [torch.empty(n, dtype=torch.float32, device=dev) for _ in range(3)]
    pos = (d["x"], d["y"], d["z"])
    vel = (d["vx"], d["vy"], d["vz"])

    # configs[4] runs n_sub sub-cycles of [drift, re-bin, force+kick] per step, restarted from
    # the initial state every step (a device-to-device copy of the six arrays, inside the step)
    nsub = cfg.n_sub
    d0 = {k: d[k].clone() for k in d} if nsub > 1 else None

    def step(events=None, counts=None):
        if nsub > 1:
            for k in d:
                d[k].copy_(d0[k])
        for s in range(nsub):
            if nsub > 1:
                haccsr.hacc_sr_drift(ctx, *pos, *vel, cfg.dt)
            if events is not None:
                events[s][0].record()
            haccsr.hacc_sr_bin(ctx, *pos, None, *vel)
            if events is not None:
                events[s][1].record()
            haccsr.hacc_sr_force_kick(ctx, cfg.eps, cfg.r_max, poly, cfg.dt, *acc, None,
                                      counts[s] if counts is not None else None)
            if events is not None:
                events[s][2].record()
            if counts is not None:
                haccsr.haccsr_sync(ctx)
                stats.append(haccsr.haccsr_get_stats(ctx))

    # C (interacting ordered pairs) and N_eval of every sub-cycle once, outside the timed
    # region, with the counting variant of the same kernel (same arithmetic, same state)
    stats = []
    tots = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(nsub)]
    step(counts=tots)
    haccsr.haccsr_sync(ctx)
    st = stats[0]
    pairs_sub = [int(t.item()) for t in tots]
    eval_sub = [s_.n_eval - n for s_ in stats]  # candidate ordered pairs, self pairs excluded
    pairs_c, n_eval = sum(pairs_sub), sum(eval_sub)
    if nsub == 1:   # velocities were kicked by the counting pass; start the timed runs clean
        for k in ("vx", "vy", "vz"):
            d[k].copy_(host[k], non_blocking=True)

    for _ in range(args.warmup):
        step()
    haccsr.haccsr_sync(ctx)

    ev = lambda: torch.cuda.Event(enable_timing=True)
    e_sub = [[(ev(), ev(), ev()) for _ in range(nsub)] for _ in range(args.steps)]
    clocks = ClockSampler(local)
    barrier()
    clocks.start()
    t_start, t_stop = ev(), ev()
    t_start.record()
    for k in range(args.steps):
        step(events=e_sub[k])
    t_stop.record()
    barrier()
    clk = clocks.stop()
    elapsed_ms = max_over_ranks(t_start.elapsed_time(t_stop), world, dev)
    bin_sub = [float(np.mean([e_sub[k][s][0].elapsed_time(e_sub[k][s][1])
                              for k in range(args.steps)])) for s in range(nsub)]
    for_sub = [float(np.mean([e_sub[k][s][1].elapsed_time(e_sub[k][s][2])
                              for k in range(args.steps)])) for s in range(nsub)]
    bin_ms, force_ms = float(np.sum(bin_sub)), float(np.sum(for_sub))  # per step
    haccsr.haccsr_sync(ctx)

    # configs[4] only: the same five sub-cycles as ONE call of hacc_sr_subcycle (the SKS map of
    # PAPER.md Eq. 9: half streams at both ends), timed on its own
    sks_ms = None
    if nsub > 1:
        e0, e1 = ev(), ev()
        ts = []
        for _ in range(max(2, min(args.steps, 3)) + 1):
            for k in d:
                d[k].copy_(d0[k])
            e0.record()
            haccsr.hacc_sr_subcycle(ctx, *pos, None, *vel, cfg.eps, cfg.r_max, poly, cfg.dt,
                                    nsub, *acc)
            e1.record()
            haccsr.haccsr_sync(ctx)
            ts.append(e0.elapsed_time(e1))
        sks_ms = float(np.min(ts[1:]))

    # configs[4] only: the same long step T = n_sub dt with multi-level time stepping
    # (Eq. 11; the paper's example: at least 2 sub-cycles, two more levels, d = 20)
    multilevel = None
    if nsub > 1:
        lev = torch.zeros(n, dtype=torch.uint8, device=dev)
        evs = torch.zeros(1, dtype=torch.int64, device=dev)
        e0, e1 = ev(), ev()
        ts = []
        for _ in range(3):
            for k in d:
                d[k].copy_(d0[k])
            e0.record()
            haccsr.hacc_sr_subcycle_multilevel(ctx, *pos, None, *vel, cfg.eps, cfg.r_max, poly,
                                               nsub * cfg.dt, 20.0, 2, 8, *acc, lev, evs)
            e1.record()
            haccsr.haccsr_sync(ctx)
            ts.append(e0.elapsed_time(e1))
        hist = torch.bincount(lev.to(torch.int64), minlength=4).tolist()
        ml_evals = int(evs.item())
        multilevel = {"call_ms": float(np.min(ts[1:])), "T": nsub * cfg.dt, "d": 20.0,
                      "l_min": 2, "l_max": 8,
                      "particles_per_level": {str(1 << k): hist[k] for k in range(len(hist))},
                      "evaluated_pairs": ml_evals,
                      "evaluated_pairs_uniform_%d_subcycles" % nsub: n_eval + n * nsub,
                      "evaluations_saved_factor_vs_uniform_%d" % nsub:
                          (n_eval + n * nsub) / max(ml_evals, 1),
                      "evaluations_saved_factor_vs_uniform_8":
                          8.0 * (n_eval + n * nsub) / nsub / max(ml_evals, 1)}

    # end to end through the public API with HOST buffers: H2D of the six particle arrays,
    # bin, force, kick, D2H of the kicked velocities, every step
    e2e_steps = max(1, min(args.steps, 5))
    out_host = [torch.empty(n, dtype=torch.float32).pin_memory() for _ in range(3)]

    copy_stream = torch.cuda.Stream(device=dev)
    out_stream = torch.cuda.Stream(device=dev)

    def e2e_run(n_steps):
        """n_steps steps, each with its own uploads and download, software-pipelined over
        three streams: the velocity upload rides under bin + force (the force needs positions
        only; the kick is then its own call), the NEXT step's position upload rides under the
        force (hacc_sr_bin has copied the positions into the workspace by then), and the
        download of the kicked velocities rides under the next step (PCIe is full duplex)."""
        main = torch.cuda.current_stream(dev)
        if nsub > 1:   # configs[4]: plain serial sequence
            for _ in range(n_steps):
                for k in host:
                    d0[k].copy_(host[k], non_blocking=True)
                step()
                for o, v in zip(out_host, vel):
                    o.copy_(v, non_blocking=True)
            return
        pos_ready = torch.cuda.Event()
        copy_stream.wait_stream(main)
        with torch.cuda.stream(copy_stream):
            for k in ("x", "y", "z"):
                d[k].copy_(host[k], non_blocking=True)
            pos_ready.record(copy_stream)
        for s_ in range(n_steps):
            vel_ready, bin_done, kick_done = (torch.cuda.Event() for _ in range(3))
            copy_stream.wait_stream(out_stream)      # previous download has left the buffers
            with torch.cuda.stream(copy_stream):
                for k in ("vx", "vy", "vz"):
                    d[k].copy_(host[k], non_blocking=True)
                vel_ready.record(copy_stream)
            main.wait_event(pos_ready)
            haccsr.hacc_sr_bin(ctx, *pos, None, *vel)
            bin_done.record(main)
            if s_ + 1 < n_steps:
                pos_ready = torch.cuda.Event()
                with torch.cuda.stream(copy_stream):
                    copy_stream.wait_event(bin_done)
                    for k in ("x", "y", "z"):
                        d[k].copy_(host[k], non_blocking=True)
                    pos_ready.record(copy_stream)
            haccsr.hacc_sr_force(ctx, cfg.eps, cfg.r_max, poly, *acc, None, None)
            main.wait_event(vel_ready)
            haccsr.hacc_sr_kick(ctx, cfg.dt)
            kick_done.record(main)
            with torch.cuda.stream(out_stream):
                out_stream.wait_event(kick_done)
                for o, v in zip(out_host, vel):
                    o.copy_(v, non_blocking=True)
        main.wait_stream(out_stream)   # the last download is inside the timed region
        main.wait_stream(copy_stream)

    e2e_run(1)
    barrier()
    s0, s1 = ev(), ev()
    s0.record()
    e2e_run(e2e_steps)
    s1.record()
    barrier()
    e2e_ms = max_over_ranks(s0.elapsed_time(s1), world, dev)

    # the same end to end step with nothing overlapped: upload, step, download, wait
    def serial_step():
        src = d0 if nsub > 1 else d
        for k in host:
            src[k].copy_(host[k], non_blocking=True)
        step()
        for o, v in zip(out_host, vel):
            o.copy_(v, non_blocking=True)
        torch.cuda.synchronize()

    serial_step()
    s0.record()
    for _ in range(e2e_steps):
        serial_step()
    s1.record()
    barrier()
    e2e_serial_ms = max_over_ranks(s0.elapsed_time(s1), world, dev) / e2e_steps

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    n_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    hbm_peak, hbm_src = measured_hbm_gbs()
    max_mhz = clk["sm_max_mhz"] or 1965.0
    peak_tflops = n_sms * FP32_LANES_PER_SM * 2 * max_mhz * 1e6 / 1e12
    probe_ms, probe_ops = haccsr.haccsr_probe_peak(1, 3)
    probe_tflops = 2 * probe_ops / (probe_ms * 1e-3) / 1e12
    achieved = FLOPS_PER_PAIR * n_eval / (force_ms * 1e-3) / 1e12
    useful = FLOPS_PER_PAIR * pairs_c / (force_ms * 1e-3) / 1e12   # interacting pairs only
    step_s = elapsed_ms * 1e-3 / args.steps
    value = whole_job_rate(pairs_c, world, step_s)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * step_s, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "parallelism": "one GPU" if world == 1 else "replicas only (--replicas)",
                   "l2": "inputs larger than L2 (bin re-reads the particle arrays from HBM "
                         "every step)" if n * 24 > 126e6 else "inputs smaller than L2",
                   "halos": int(p["n_halos"]), "max_cell_count": st.max_cell_count,
                   "work_items": st.n_items, "sources_per_split": st.sources_per_split},
        "interacting_pairs": pairs_c, "evaluated_pairs": n_eval,
        "evaluated_pairs_per_s": world * n_eval / step_s,
        "ns_per_particle_step": step_s / n / nsub * 1e9,
        "bin_ms": bin_ms, "force_kick_ms": force_ms,
        "bin_gbs": BIN_BYTES_PER_PARTICLE * n * nsub / (bin_ms * 1e-3) / 1e9,
        "fp32_frac_of_peak": achieved / peak_tflops,
        "fp32_frac_of_peak_useful": useful / peak_tflops,
        "roofline": {"bound": "alu",
                     "kernel": "k_force + k_force_sparse (one force evaluation)" if n >= (1 << 20)
                     else "k_force", "achieved": achieved,
                     "peak": peak_tflops, "unit": "TFLOP/s", "frac": achieved / peak_tflops,
                     "traffic": FORCE_TRAFFIC_BYTES.get(cfg.index, (None, None))[0],
                     "traffic_source": FORCE_TRAFFIC_BYTES.get(cfg.index, (None, None))[1],
                     "peak_source": (f"derived: {n_sms} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 "
                                     f"x {max_mhz:g} MHz (clocks.max.sm)"),
                     "peak_probe_ffma2": probe_tflops,
                     # per force evaluation (configs[4]: the mean of its sub-cycles)
                     "flops_per_pair": FLOPS_PER_PAIR, "pairs_per_launch": n_eval / nsub,
                     # the same with only the pairs inside the cutoff counted (north_star's
                     # "useful pair-interaction flops"): the select zeroes the others
                     "achieved_useful": useful, "frac_useful": useful / peak_tflops},
        "bin_roofline": {"bound": "hbm", "kernel": "hacc_sr_bin (all its kernels)",
                         "achieved": BIN_BYTES_PER_PARTICLE * n * nsub / (bin_ms * 1e-3) / 1e9,
                         "peak": hbm_peak, "unit": "GB/s",
                         "frac": BIN_BYTES_PER_PARTICLE * n * nsub / (bin_ms * 1e-3) / 1e9 / hbm_peak,
                         "peak_source": hbm_src,
                         "bytes_per_particle_algorithmic": BIN_BYTES_PER_PARTICLE,
                         "bytes_per_particle_moved": 104},
        "clocks": clk,
        "sks_subcycle_call_ms": sks_ms,
        "multilevel": multilevel,
        "subcycles": [{"bin_ms": bin_sub[s_], "force_kick_ms": for_sub[s_],
                       "interacting_pairs": pairs_sub[s_], "evaluated_pairs": eval_sub[s_],
                       "max_cell_count": stats[s_].max_cell_count} for s_ in range(nsub)],
        "e2e": {"value": world * pairs_c / (e2e_ms * 1e-3 / e2e_steps), "unit": UNIT,
                "h2d_bytes_per_step": 24 * n, "d2h_bytes_per_step": 12 * n,
                "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps,
                "pipelined": nsub == 1,
                "serial_ms_per_step": e2e_serial_ms,
                "serial_value": world * pairs_c / (e2e_serial_ms * 1e-3)},
        "gpu_launches": (kernels_per_step(n, cfg.nc) + (1 if nsub > 1 else 0)) * nsub * args.steps,
    }
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(cfg, p, args.cpu_seconds)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_slab_sim(args):
    """--slab-sim N on ONE GPU: the N slab contexts of the sharded box run
    ONE AFTER ANOTHER, each with its passive layers taken from the whole box (what the
    exchange would deliver), bin + force+kick timed per slab with CUDA events.  The slowest
    slab bounds a step of the N-rank run, so whole-box time / slowest slab time is the strong
    scaling these kernels allow (the 2 x 25 MB exchange per step is not in it).  Printed for
    slabs of equal thickness and of equal work."""
    import torch

    from paper_1410_2805_b200 import haccsr, sharding
    from paper_1410_2805_b200 import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    cfg = W.CONFIGS[args.config]
    world, poly = args.slab_sim, W.DEFAULT_POLY
    p = W.make_particles(cfg)
    full = [torch.from_numpy(p[k]).to(dev) for k in "xyz"]
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def timed(ctx, pos, vel, acc):
        for _ in range(max(1, args.warmup)):
            haccsr.hacc_sr_bin(ctx, *pos, None, *vel)
            haccsr.hacc_sr_force_kick(ctx, cfg.eps, cfg.r_max, poly, cfg.dt, *acc, None, None)
        e0, e1 = ev(), ev()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(args.steps):
            haccsr.hacc_sr_bin(ctx, *pos, None, *vel)
            haccsr.hacc_sr_force_kick(ctx, cfg.eps, cfg.r_max, poly, cfg.dt, *acc, None, None)
        e1.record()
        torch.cuda.synchronize()
        haccsr.haccsr_sync(ctx)
        return e0.elapsed_time(e1) / args.steps

    # the whole box on one GPU
    ctx = haccsr.Context(cfg.n, cfg.box_l, cfg.nc, device=dev)
    vel = [torch.zeros(cfg.n, device=dev) for _ in range(3)]
    acc = [torch.empty(cfg.n, device=dev) for _ in range(3)]
    whole_ms = timed(ctx, full, vel, acc)
    del ctx, vel, acc
    torch.cuda.empty_cache()

    # particles per layer by the library's own cell index
    probe = haccsr.Context(1, cfg.box_l, cfg.nc, device=dev)
    cnt = torch.zeros(1, dtype=torch.int32, device=dev)
    dummy = torch.empty(4, dtype=torch.float32, device=dev)
    pop = []
    for cz in range(cfg.nc):
        haccsr.hacc_sr_pack_layer(probe, *full, None, cz, dummy, cnt)
        pop.append(int(cnt.item()))
    work = sharding.layer_work(*full, cfg.box_l, cfg.nc)
    out = {}
    for name, layers in (("equal_thickness", sharding.slab_layers(cfg.nc, world)),
                         ("equal_work", sharding.slab_layers_balanced(work, world))):
        times = []
        for r, (lo, nz_own) in enumerate(layers):
            below, above = (lo - 1) % cfg.nc, (lo + nz_own) % cfg.nc
            n_own = sum(pop[(lo + k) % cfg.nc] for k in range(nz_own))
            msg_cap = max(pop) + 1024
            slab = sharding.SlabRank(r, world, cfg.box_l, cfg.nc, n_own + pop[below] + pop[above]
                                     + 4096, msg_cap, dev, layers=layers)
            assert sharding.scatter_to_slab(slab, *full) == n_own
            buf = torch.empty(4 * msg_cap, dtype=torch.float32, device=dev)
            for layer in (below, above):      # the passive copies the exchange would deliver
                haccsr.hacc_sr_pack_layer(probe, *full, None, layer, buf, cnt)
                slab.append(buf, int(cnt.item()))
            pos, _, v, a = slab.views()
            times.append(timed(slab.ctx, pos, v, a))
            del slab, buf, pos, v, a
            torch.cuda.empty_cache()
        out[name] = {"layers": [nz for _, nz in layers],
                     "work_share": [sum(work[(lo + k) % cfg.nc] for k in range(nz)) / sum(work)
                                    for lo, nz in layers],
                     "slab_ms": times, "slowest_ms": max(times),
                     "speedup": whole_ms / max(times),
                     "efficiency": whole_ms / max(times) / world}
    print(json.dumps({"metric": "strong scaling predicted from slabs run one after another on one GPU",
                      "n_slabs": world, "whole_box_ms": whole_ms, "steps": args.steps,
                      "warmup": args.warmup, "data": "synthetic",
                      "config": {"workload": workload_name(cfg)}, **out}))


def run_long_range(args):
    """One JSON line for the long-range PM force (libhaccpm.so) on one GPU: a grid of n_side^3
    nodes (one per particle on average), inputs resident, CUDA events."""
    import torch

    from paper_1410_2805_b200 import haccpm
    from paper_1410_2805_b200 import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    cfg = W.CONFIGS[args.config]
    p = W.make_particles(cfg)
    pos = [torch.from_numpy(p[k]).cuda() for k in "xyz"]
    vel = [torch.from_numpy(np.ascontiguousarray(p[k])).cuda() for k in ("vx", "vy", "vz")]
    acc = [torch.empty(cfg.n, device="cuda") for _ in range(3)]
    ctx = haccpm.Context(cfg.n_side, cfg.box_l)

    def step():
        haccpm.hacc_lr_force(ctx, *pos, None, *acc, cfg.dt, *vel)

    for _ in range(max(args.warmup, 1)):
        step()
    clocks = ClockSampler(0)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    torch.cuda.synchronize()
    clocks.start()
    ev[0].record()
    for _ in range(args.steps):
        step()
    ev[1].record()
    torch.cuda.synchronize()
    clk = clocks.stop()
    haccpm.haccpm_sync(ctx)
    ms = ev[0].elapsed_time(ev[1]) / args.steps
    print(json.dumps({
        "metric": "long-range PM force, particles/s", "value": cfg.n / (ms * 1e-3),
        "unit": "particles/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": True, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"configs[{cfg.index}] particles ({cfg.n_side}^3={cfg.n}, L={cfg.box_l:g}, "
                   f"{int(round(cfg.f_halo * 100))}% in Plummer halos), PM grid {cfg.n_side}^3, "
                   "sigma=0.8, n_s=3: CIC deposit + cuFFT R2C + 3 x (spectral multiply + cuFFT "
                   "C2R) + pack + CIC interpolation with kick",
                   "l2": "grid and particle arrays larger than L2" if cfg.n_side >= 512
                   else "grid smaller than L2"},
        "gpu_launches": 6 * args.steps,   # deposit, 3 x green, pack, interp (cuFFT's are a library's)
        "clocks": clk}))


def main():
    args = parse_args()
    if args.slab_sim > 1:
        run_slab_sim(args)
    elif args.long_range:
        run_long_range(args)
    elif args.impl == "reference":
        run_reference(args)
    elif int(os.environ.get("WORLD_SIZE", "1")) > 1 and not args.replicas:
        run_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
