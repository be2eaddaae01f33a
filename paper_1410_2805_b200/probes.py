"""Run the library's probe kernels (haccsr_probe_peak, include/haccsr.h) and print a table.

    python -m paper_1410_2805_b200.probes

These are the measurements DESIGN.md quotes for its design decisions: the FP32 / SFU peaks, what
the force kernel's instruction mix can reach with and without the cutoff select and the
guard-band test, and why the counting sort stages its writes through shared memory (scattered
16-byte stores vs runs; shared vs global atomics).  Needs a CUDA device.
"""
from __future__ import annotations

import torch

from . import haccsr

SM_LANES = 128


def main():
    props = torch.cuda.get_device_properties(0)
    sms = props.multi_processor_count
    try:
        import pynvml
        pynvml.nvmlInit()
        mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(pynvml.nvmlDeviceGetHandleByIndex(0),
                                                     pynvml.NVML_CLOCK_SM))
    except Exception:
        mhz = 1965.0
    fma_peak = sms * SM_LANES * mhz * 1e6          # FMA lane-operations per second
    pair_cap = fma_peak / 16.0                     # 16 FMA-pipe lane-operations per pair
    print(f"{props.name}, {sms} SMs, max SM clock {mhz:g} MHz; FP32 peak "
          f"{2 * fma_peak / 1e12:.2f} TFLOP/s; pair-loop cap {pair_cap / 1e12:.3f} T pairs/s\n")
    rows = [
        (0, "scalar FFMA", "TFLOP/s", 2e-12, 2 * fma_peak),
        (1, "packed fma.rn.f32x2", "TFLOP/s", 2e-12, 2 * fma_peak),
        (2, "MUFU rsqrt", "T/s", 1e-12, None),
        (3, "pair loop: select + band (the kernel's mix)", "T pairs/s", 1e-12, pair_cap),
        (4, "pair loop: select only", "T pairs/s", 1e-12, pair_cap),
        (5, "pair loop: neither", "T pairs/s", 1e-12, pair_cap),
        (6, "16 B stores, random slot in 1 MB window", "G stores/s", 1e-9, None),
        (7, "16 B stores, runs of 32 slots", "G stores/s", 1e-9, None),
        (8, "shared-memory atomics, 9596 counters", "G/s", 1e-9, None),
        (9, "global atomics with return, 9596 counters", "G/s", 1e-9, None),
    ]
    print("| kind | probe | rate | unit | % of cap |")
    print("|---|---|---:|---|---:|")
    for kind, name, unit, scale, cap in rows:
        ms, ops = haccsr.haccsr_probe_peak(kind, 3)
        rate = ops / (ms * 1e-3)
        pct = f"{100 * rate * (2 if kind < 2 else 1) / cap:.1f}" if cap else ""
        print(f"| {kind} | {name} | {rate * scale:.2f} | {unit} | {pct} |")


if __name__ == "__main__":
    main()
