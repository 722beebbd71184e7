"""Shared helpers of the GPU parity tests: run the CUDA path through the C ABI and compare with the oracle."""
import numpy as np
import torch

POWER_RTOL = 1e-5   # BASELINE.json north_star: powers within relative 1e-5
SIGMA_ATOL = 1e-3   # sigma within absolute 1e-3; bins and widths bit-exact


def gpu_search(spectra: torch.Tensor, zmax, norm_block, block_width, thr, n_bins=None, n_trials=None, mode=0, **tuning):
    from paper_2406_15186_b200 import binding

    if spectra.dim() == 1:
        spectra = spectra[None, :]
    batch, pitch = spectra.shape
    n = pitch if n_bins is None else n_bins
    plan = binding.Plan(n, batch, zmax, block_width, thr, norm_block=norm_block, n_trials=n_trials,
                        pitch=pitch if pitch != n else None, mode=mode, **tuning)
    plan.attach(spectra.device)
    plan.search(spectra.contiguous())
    rec = plan.candidates()
    stats = plan.stats()
    plan.destroy()
    return rec, stats


def oracle_search(orc, spectra: torch.Tensor, zmax, norm_block, block_width, thr, n_bins=None, n_trials=1.0, z_step=1,
                  log_sampling=False, r_block=False):
    return orc.search(spectra.cpu().numpy(), zmax, norm_block, block_width, thr, n_trials=n_trials, n_bins=n_bins,
                      z_step=z_step, log_sampling=log_sampling, r_block=r_block)


def assert_same_candidates(gpu, ora, context=""):
    gk = list(zip(gpu["spectrum"].tolist(), gpu["bin"].tolist(), gpu["width"].tolist()))
    ok = list(zip(ora["spectrum"].tolist(), ora["bin"].tolist(), ora["width"].tolist()))
    if gk != ok:
        only_g = sorted(set(gk) - set(ok))[:10]
        only_o = sorted(set(ok) - set(gk))[:10]
        raise AssertionError(f"{context}: candidate (spectrum, bin, width) lists differ: gpu {len(gk)} vs oracle {len(ok)}; "
                             f"only gpu {only_g}; only oracle {only_o}")
    if len(gk):
        rel = np.abs(gpu["power"].astype(np.float64) - ora["power"]) / ora["power"]
        assert rel.max() <= POWER_RTOL, f"{context}: power rel err {rel.max():.3g}"
        dsig = np.abs(gpu["sigma"].astype(np.float64) - ora["sigma"])
        assert dsig.max() <= SIGMA_ATOL, f"{context}: sigma abs err {dsig.max():.3g}"
