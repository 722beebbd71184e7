"""pulscan_normalise_power_static — the entry point for callers that cannot allocate device memory.

Some users of this library have nothing to give it but an input and an output buffer: every byte of their GPU was handed out
when their pipeline started, or a host application owns the allocator.  They cannot provide the workspace that the fast
normalisation kernels keep their scratch in (a list of blocks passed on to the general kernel, a few counters), so the library
carries a fixed array for it.  That array is shared by all calls and keeps whatever the last call wrote, which is what these
tests are about: two calls in a row, the second with fewer listed blocks than the first, must each give what the existing
workspace path gives on the same input (tolerance: the parity tests' 1e-5·P + 1e-6).

Collected last on purpose (pytest -x stops at the first failure; a failure here must not hide the parity tests).  It passes on
its own in a fresh process and after the rest of the suite: nothing else touches the array.
"""
import numpy as np
import pytest
import torch

from _parity import POWER_RTOL

N_BINS, BATCH, NORM_BLOCK = 6 * 1024 + 300, 3, 1024      # six full blocks per row + a ragged last one (tail launch)


def _spectra(seed, degenerate):
    """Noise with some blocks the fast kernel declines (constant or heavily quantised values): they go through the list."""
    g = torch.Generator(device="cpu").manual_seed(seed)
    x = torch.view_as_complex(torch.randn(BATCH, N_BINS, 2, generator=g, dtype=torch.float32) * 30.0).clone()
    for row, blk, kind in degenerate:
        lo = blk * NORM_BLOCK
        if kind == "constant":
            x[row, lo:lo + NORM_BLOCK] = 2.0 - 1.0j                  # MAD = 0 in both components: power 0 (R7)
        else:
            x.real[row, lo:lo + 700] = -4.0                          # more than half a block identical: MAD = 0 for re only
    return x.to("cuda")


@pytest.mark.gpu
def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row():
    from paper_2406_15186_b200 import binding

    first = _spectra(11, [(0, 0, "constant"), (0, 3, "half"), (1, 2, "constant"), (2, 1, "half"), (2, 4, "constant")])
    second = _spectra(12, [(1, 4, "half")])                          # fewer listed blocks: stale entries stay behind the count

    # the existing path: workspace attached, fast kernels + list in the workspace
    ws_plan = binding.Plan(N_BINS, BATCH, 8, 16, 6.0, norm_block=NORM_BLOCK)
    ws_plan.attach("cuda")
    want, listed = [], []
    for spec in (first, second):
        want.append(ws_plan.normalise_power(spec).cpu().numpy().astype(np.float64))
        listed.append(int(ws_plan.stats()[1]))
    ws_plan.destroy()
    assert listed[0] >= 4 and 1 <= listed[1] < listed[0], listed     # the list really is used, and shrinks

    # the new entry point: no workspace, output buffers from the caller, calls back to back on one stream
    plan = binding.Plan(N_BINS, BATCH, 8, 16, 6.0, norm_block=NORM_BLOCK)
    assert plan.workspace is None
    outs = [torch.full((BATCH, plan.power_pitch), float("nan"), dtype=torch.float32, device="cuda") for _ in range(2)]
    got = [plan.normalise_power_static(spec, out) for spec, out in zip((first, second), outs)]
    torch.cuda.synchronize()
    got = [g.cpu().numpy().astype(np.float64) for g in got]
    plan.destroy()

    for k in range(2):
        assert np.all(np.isfinite(got[k])), f"call {k}: bins left unwritten"
        err = np.abs(got[k] - want[k])
        assert np.all(err <= POWER_RTOL * want[k] + 1e-6), f"call {k}: max err {err.max()} at {np.unravel_index(err.argmax(), err.shape)}"
    assert np.all(got[0][0, :NORM_BLOCK] == 0)                        # the constant block


def test_static_scratch_rejects_sizes_beyond_its_array():
    """Host-side check, before anything touches a device: 257 x 1024 blocks > PULSCAN_STATIC_MAX_NORM_BLOCKS = 262144."""
    from paper_2406_15186_b200 import build as pbuild
    pbuild.build()
    from paper_2406_15186_b200 import binding

    plan = binding.Plan(1024 * 4096, 257, 8, 16, 6.0, norm_block=4096)
    rc = plan.lib.pulscan_normalise_power_static(plan.handle, 256, 256, None)   # never dereferenced: rejected first
    assert rc == binding.PULSCAN_EINVAL
    assert "PULSCAN_STATIC_MAX_NORM_BLOCKS" in binding.last_error()
    plan.destroy()
