"""Diagnostic: clock counts per phase of the single-histogram normalisation kernel (norm_power_v2.cuh).

Needs a library built with the instrumentation compiled in:
    PULSCAN_NVCC_EXTRA=-DPULSCAN_V2_TIMING python -m paper_2406_15186_b200.build
    python -m paper_2406_15186_b200.phase_timing [config 1-5] [batch]
Thread 0 of every CTA adds clock64() differences between the kernel's CTA barriers to a device array; the numbers are
per normalisation block, summed over both components.  The instrumented build is slower than the product build (two more
live registers at the 64-register cap): read the shares, not the absolutes.  Not used by the tests or by bench.py.
"""
from __future__ import annotations

import ctypes
import sys

import torch

from . import binding, synth

PHASES = ["sample estimate + zeroing", "histogram pass", "chunk totals", "locate (2 of 4 warps)", "gather",
          "resolve (2 of 4 warps)", "output"]
RESOLVE = ["resolve: checks", "resolve: rank median net", "resolve: deviations + rank shells", "resolve: verify + 1/(√2·κ·MAD)"]


def main(argv) -> None:
    cfg = int(argv[1]) if len(argv) > 1 else 3
    batch = int(argv[2]) if len(argv) > 2 else 64
    wl = synth.CONFIGS[cfg]
    lib = binding.load_library()
    if not hasattr(lib, "pulscan_debug_v2_timing"):
        raise SystemExit("libpulscan.so was built without -DPULSCAN_V2_TIMING (see the module docstring)")
    fn = lib.pulscan_debug_v2_timing
    fn.argtypes = [ctypes.c_void_p, ctypes.c_int]
    g = torch.Generator(device="cuda").manual_seed(1)
    X = torch.view_as_complex(torch.randn(batch, wl.n_bins, 2, device="cuda", generator=g) * wl.n_bins ** 0.5).contiguous()
    plan = binding.Plan(wl.n_bins, batch, wl.zmax, wl.block_width, wl.sigma_threshold, norm_block=wl.norm_block)
    plan.attach("cuda:0")
    for _ in range(2):
        plan.search(X)
    torch.cuda.synchronize()
    fn(None, 1)
    plan.search(X)
    torch.cuda.synchronize()
    out = (ctypes.c_ulonglong * 16)()
    fn(out, 0)
    plan.destroy()
    nb = batch * (wl.n_bins // wl.norm_block)
    tot = sum(out[:7])
    print(f"config {cfg}, batch {batch}: {nb} normalisation blocks of {wl.norm_block} bins")
    for k, name in enumerate(PHASES):
        print(f"  {name:34s} {out[k] / nb:9.0f} cycles/block  {100 * out[k] / tot:5.1f} %")
    print(f"  {'total':34s} {tot / nb:9.0f} cycles/block")
    for k, name in zip(range(8, 12), RESOLVE):
        print(f"  {name:34s} {out[k] / nb:9.0f} cycles/block")


if __name__ == "__main__":
    main(sys.argv)
