"""GPU parity (through the C ABI) against the oracle at sizes the oracle finishes in seconds: several tiles, ragged
tails, both sweep modes, edge and degenerate cases.  Bins/widths bit-exact, power rel 1e-5, sigma abs 1e-3."""
import numpy as np
import pytest
import torch

from _parity import assert_same_candidates, gpu_search, oracle_search
from paper_2406_15186_b200 import synth

pytestmark = pytest.mark.gpu


def noise_spectra(batch, n, seed, scale=50.0, device="cuda"):
    g = torch.Generator(device="cpu").manual_seed(seed)
    x = torch.randn(batch, n, 2, generator=g, dtype=torch.float32) * scale
    return torch.view_as_complex(x).to(device)


def bump(spec, row, start, width, factor):
    spec[row, start:start + width] *= factor


@pytest.mark.parametrize("n,B", [(1000, 256), (4097, 1024), (12289, 4096), (8192, 4096), (16385, 8192), (300, 512),
                                 (40000, 16384), (5000, 100), (2049, 2)])
def test_normalise_power_matches_oracle(orc, n, B):
    from paper_2406_15186_b200 import binding
    spec = noise_spectra(3, n, seed=n + B)
    spec[1] = spec[1] * 1e-3 + (5.0 - 2.0j)     # offset and scale differ per row
    plan = binding.Plan(n, 3, min(8, n - 1), 16, 6.0, norm_block=B)
    P_general = plan.normalise_power(spec).cpu().numpy().astype(np.float64)   # no workspace: general kernels
    plan.attach("cuda")
    P_fast = plan.normalise_power(spec).cpu().numpy().astype(np.float64)      # as in pulscan_search: fast + redo kernels
    stats = plan.stats()
    plan.destroy()
    assert np.array_equal(P_general, P_fast)           # both paths select exactly, then share the arithmetic
    assert stats[1] <= 1                               # fast-path blocks sent to the redo list (h_stats[4..8] say why)
    for b in range(3):
        ref = orc.normalise_power(spec[b].cpu().numpy(), B)
        err = np.abs(P_fast[b] - ref)
        # bins whose component sits next to the block median cancel in v − m: absolute floor
        assert np.all(err <= 1e-5 * ref + 1e-6), f"row {b}: max err {err.max()} at {err.argmax()}"


def test_normalise_power_degenerate_blocks(orc):
    from paper_2406_15186_b200 import binding
    n, B = 3 * 512 + 7, 512
    spec = noise_spectra(1, n, seed=5)
    spec[0, :512] = 3.0 + 4.0j                       # MAD = 0 in both components → power 0 (R7)
    spec[0, 512:1024].imag.round_()                  # heavy duplicates (quantised) in one component
    spec.real[0, 1024:1024 + 300] = 7.0              # > half the block identical → MAD = 0 for re only
    plan = binding.Plan(n, 1, 8, 16, 6.0, norm_block=B)
    plan.attach("cuda")
    P = plan.normalise_power(spec).cpu().numpy().astype(np.float64)
    assert plan.stats()[1] >= 1                        # degenerate blocks leave the fast path for the general one
    plan.destroy()
    ref = orc.normalise_power(spec[0].cpu().numpy(), B)
    assert np.all(P[0, :512] == 0)
    assert np.all(np.abs(P[0] - ref) <= 1e-5 * ref + 1e-6)


def test_normalise_power_extreme_ranges(orc):
    from paper_2406_15186_b200 import binding
    n, B = 4096, 1024
    spec = noise_spectra(1, n, seed=6, scale=1.0)
    spec[0, :1024] *= 1e-30                           # tiny values: linear bucketing scale overflows → key path
    spec[0, 1024:2048] *= 1e30
    spec.real[0, 2048] = 3e38                         # one huge outlier stretches the range
    spec.real[0, 2049] = -3e38
    plan = binding.Plan(n, 1, 8, 16, 6.0, norm_block=B)
    plan.attach("cuda")
    P = plan.normalise_power(spec).cpu().numpy().astype(np.float64)
    plan.destroy()
    ref = orc.normalise_power(spec[0].cpu().numpy(), B)
    ok = ref < 1e30                                   # the two outliers' own powers (~1e76) overflow float32
    assert ok.sum() == n - 2
    bad = np.flatnonzero(np.abs(P[0][ok] - ref[ok]) > 1e-5 * ref[ok] + 1e-6)    # §8(c) step 3's tolerance, as everywhere
    assert bad.size == 0, f"{bad[:10]} gpu {P[0][ok][bad[:5]]} ref {ref[ok][bad[:5]]}"


CASES = [
    # n, batch, zmax, B, C, thr
    (4097, 2, 16, 1024, 64, 4.0),
    (20001, 3, 40, 2048, 100, 4.5),
    (32769, 1, 32, 1024, 64, 4.0),
    (9000, 2, 200, 4096, 200, 4.0),
    (30011, 1, 300, 8192, 1200, 4.0),
    (5000, 4, 7, 512, 1, 3.5),
    (777, 2, 100, 256, 5000, 3.0),
    (2100, 1, 2000, 1024, 50, 3.5),
    (30011, 1, 4096, 8192, 2000, 4.0),     # zmax·C = 8.2 M window sums per block: kernel (c) deals a block's widths to 2 CTAs
    (40001, 2, 3000, 4096, 3100, 4.5),     # … to 3 CTAs
]


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("n,batch,zmax,B,C,thr", CASES)
def test_search_matches_oracle(orc, n, batch, zmax, B, C, thr, mode):
    spec = noise_spectra(batch, n, seed=n * 7 + zmax)
    bump(spec, 0, n // 3, 6, 3.0)
    bump(spec, batch - 1, n // 2, min(zmax, 60), 1.8)
    bump(spec, batch - 1, n - 5, 5, 4.0)             # at the very end of the row: truncated windows (R11)
    gpu, stats = gpu_search(spec, zmax, B, C, thr, mode=mode)
    ora = oracle_search(orc, spec, zmax, B, C, thr)
    assert len(ora) > 0
    assert_same_candidates(gpu, ora, f"n={n} zmax={zmax} mode={mode}")
    assert stats[0] >= len(ora)                      # every emitting block was flagged by the sweep


def test_pruned_equals_exhaustive_on_noise_with_low_threshold(orc):
    spec = noise_spectra(2, 50001, seed=99)
    a, _ = gpu_search(spec, 64, 2048, 128, 3.0, mode=0)
    b, _ = gpu_search(spec, 64, 2048, 128, 3.0, mode=1)
    assert np.array_equal(a, b) and len(a) > 50
    assert_same_candidates(a, oracle_search(orc, spec, 64, 2048, 128, 3.0), "thr=3 noise")


@pytest.mark.parametrize("zmax,thr,z_step,n", [(128, 2.0, 1, 30011), (200, 3.0, 1, 30011), (512, 2.5, 1, 30011), (128, 3.0, 127, 30011),
                                               (256, 2.0, 127, 30011), (1024, 2.0, 1, 20001), (1024, 3.0, 1, 20001),
                                               (4096, 4.0, 1, 30011)])
def test_low_threshold_wide_levels_pruned_equals_exhaustive_equals_oracle(orc, zmax, thr, z_step, n):
    """Levels spanning up to 128 cover lengths (32 steps of 4, the last step included) and plans that need the relaxed flag
    probability: low thresholds with large zmax, and a z_step that leaves one searched width alone in a level's last step."""
    spec = noise_spectra(1, n, seed=zmax * 31 + z_step)
    bump(spec, 0, n // 2, min(zmax, 128), 1.6)
    C = 256
    a, _ = gpu_search(spec, zmax, 4096, C, thr, mode=0, z_step=z_step)
    b, _ = gpu_search(spec, zmax, 4096, C, thr, mode=1, z_step=z_step)
    assert np.array_equal(a, b) and len(a) > 0
    assert_same_candidates(a, oracle_search(orc, spec, zmax, 4096, C, thr, z_step=z_step), f"zmax={zmax} thr={thr} z_step={z_step}")


@pytest.mark.parametrize("tile,lpf", [(1024, -2.0), (2048, -3.0), (8192, -7.0), (16384, -9.0)])
def test_tuning_never_changes_results(orc, tile, lpf):
    spec = noise_spectra(1, 40000, seed=123)
    bump(spec, 0, 17000, 90, 1.7)
    ref, _ = gpu_search(spec, 150, 4096, 200, 4.0)
    got, _ = gpu_search(spec, 150, 4096, 200, 4.0, tile=tile, log10_p_flag=lpf)
    assert np.array_equal(ref, got)


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("z_step,log_sampling", [(4, False), (13, False), (1, True)])
@pytest.mark.parametrize("n,batch,zmax,B,C,thr", [(20001, 2, 40, 2048, 100, 4.0), (9000, 2, 200, 4096, 200, 4.0),
                                                  (30011, 1, 300, 8192, 1200, 4.0)])
def test_width_sampling_matches_oracle(orc, n, batch, zmax, B, C, thr, z_step, log_sampling, mode):
    spec = noise_spectra(batch, n, seed=n + zmax)
    bump(spec, 0, n // 3, 6, 3.0)
    bump(spec, batch - 1, n // 2, min(zmax, 60), 1.8)
    gpu, _ = gpu_search(spec, zmax, B, C, thr, mode=mode, z_step=z_step, log_sampling=log_sampling)
    ora = oracle_search(orc, spec, zmax, B, C, thr, z_step=z_step, log_sampling=log_sampling)
    assert len(ora) > 0
    assert all(orc.width_searched(int(w), z_step, log_sampling) for w in gpu["width"])
    assert_same_candidates(gpu, ora, f"n={n} zmax={zmax} z_step={z_step} log={log_sampling} mode={mode}")


def test_r_block_matches_oracle(orc):
    spec = noise_spectra(2, 20001, seed=4242)
    bump(spec, 1, 7777, 20, 2.5)
    gpu, _ = gpu_search(spec, 48, 2048, 100, 4.0, r_block=True, log_sampling=True)
    ora = oracle_search(orc, spec, 48, 2048, 100, 4.0, r_block=True, log_sampling=True)
    assert len(ora) > 0 and np.all(ora["bin"] % 100 == 0)
    assert_same_candidates(gpu, ora, "R-Block + log sampling")
    exact, _ = gpu_search(spec, 48, 2048, 100, 4.0, log_sampling=True)
    assert np.array_equal(gpu["bin"], exact["bin"] // 100 * 100) and np.array_equal(gpu["sigma"], exact["sigma"])


def _assert_same_hcandidates(gpu, ora, context):
    gk = list(zip(gpu["numharm"].tolist(), gpu["spectrum"].tolist(), gpu["bin"].tolist(), gpu["width"].tolist()))
    ok = list(zip(ora["numharm"].tolist(), ora["spectrum"].tolist(), ora["bin"].tolist(), ora["width"].tolist()))
    assert gk == ok, (f"{context}: gpu {len(gk)} vs oracle {len(ok)}; only gpu {sorted(set(gk) - set(ok))[:8]}; "
                      f"only oracle {sorted(set(ok) - set(gk))[:8]}")
    rel = np.abs(gpu["power"].astype(np.float64) - ora["power"]) / ora["power"]
    assert rel.max() <= 1e-5, f"{context}: power rel err {rel.max():.3g}"
    assert np.abs(gpu["sigma"].astype(np.float64) - ora["sigma"]).max() <= 1e-3, context


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("n,batch,zmax,B,C,thr,numharm,log_sampling", [
    (20001, 2, 40, 2048, 100, 4.0, 4, False), (9001, 2, 200, 4096, 200, 4.0, 3, False), (30011, 1, 64, 8192, 300, 4.5, 4, True),
    (4099, 3, 16, 1024, 64, 3.5, 2, False), (40001, 1, 600, 8192, 700, 4.5, 2, False)])   # the last: 8192-bin tiles, two scan passes
def test_harmonic_search_matches_oracle(orc, n, batch, zmax, B, C, thr, numharm, log_sampling, mode):
    from paper_2406_15186_b200 import binding
    spec = noise_spectra(batch, n, seed=n + numharm)
    for h in range(1, 5):                                  # power at bin 501 and its harmonics, two bins wide
        if h * 501 + 2 < n:
            spec[0, h * 501: h * 501 + 2] *= 3.0
    bump(spec, batch - 1, n // 2, min(zmax, 30), 1.8)
    plan = binding.Plan(n, batch, zmax, C, thr, norm_block=B, mode=mode, numharm=numharm, log_sampling=log_sampling)
    plan.attach("cuda")
    plan.search_harmonics(spec)
    gpu = plan.hcandidates()
    plan.search(spec)                                      # the plain search of the same plan is unaffected
    plain = plan.candidates()
    plan.destroy()
    ora = orc.search_harmonics(spec.cpu().numpy(), zmax, B, C, thr, numharm, log_sampling=log_sampling)
    assert len(ora) > 0 and set(ora["numharm"].tolist()) == set(range(1, numharm + 1))
    _assert_same_hcandidates(gpu, ora, f"n={n} numharm={numharm} mode={mode}")
    h1 = gpu[gpu["numharm"] == 1]
    assert np.array_equal(h1["bin"], plain["bin"]) and np.array_equal(h1["sigma"], plain["sigma"])


@pytest.mark.parametrize("n,B", [(4 * 256 + 3, 256), (3 * 512, 512), (5 * 1024 + 1000, 1024), (2 * 2048 + 1, 2048), (12289, 4096),
                                 (16385, 8192), (40000, 16384)])
def test_median_of_medians_power_matches_oracle(orc, n, B):
    """Fast mode (Alg. 1): the kernel against the oracle's step-by-step Alg. 1."""
    from paper_2406_15186_b200 import binding
    spec = noise_spectra(3, n, seed=n + B)
    spec[1] = spec[1] * 1e-3 + (5.0 - 2.0j)     # offset and scale differ per row
    plan = binding.Plan(n, 3, min(8, n - 1), 16, 6.0, norm_block=B, median_of_medians=True)
    plan.attach("cuda")
    P = plan.normalise_power(spec).cpu().numpy().astype(np.float64)
    assert plan.launches_per_search == 4        # one normalisation kernel + sweep + refine + exact
    plan.destroy()
    for b in range(3):
        ref = orc.normalise_power_mom(spec[b].cpu().numpy(), B)
        err = np.abs(P[b] - ref)
        assert np.all(err <= 1e-5 * ref + 1e-6), f"row {b}: max err {err.max()} at {err.argmax()} (ref {ref[err.argmax()]})"


@pytest.mark.parametrize("n,batch,zmax,B,C,thr,numharm", [(20001, 2, 40, 2048, 100, 4.0, 1), (9001, 2, 100, 4096, 200, 4.0, 3),
                                                          (32769, 1, 32, 1024, 64, 4.0, 1)])
def test_search_with_median_of_medians_matches_oracle(orc, n, batch, zmax, B, C, thr, numharm):
    from paper_2406_15186_b200 import binding
    spec = noise_spectra(batch, n, seed=n * 3 + zmax)
    bump(spec, 0, n // 3, 6, 3.0)
    bump(spec, batch - 1, n // 2, min(zmax, 60), 1.8)
    plan = binding.Plan(n, batch, zmax, C, thr, norm_block=B, numharm=numharm, median_of_medians=True)
    plan.attach("cuda")
    plan.search_harmonics(spec)
    gpu = plan.hcandidates()
    plan.destroy()
    ora = orc.search_harmonics(spec.cpu().numpy(), zmax, B, C, thr, numharm, median_of_medians=True)
    assert len(ora) > 0
    _assert_same_hcandidates(gpu, ora, f"median of medians n={n} numharm={numharm}")


@pytest.mark.parametrize("numharm,log_sampling", [(1, False), (1, True), (3, False)])
def test_per_width_emission_matches_oracle(orc, numharm, log_sampling):
    """The paper's GPU output (Alg. 4): one record per (block, searched width) above the threshold."""
    from paper_2406_15186_b200 import binding
    n, batch, zmax, B, C, thr = 20001, 2, 40, 2048, 100, 4.0
    spec = noise_spectra(batch, n, seed=777)
    bump(spec, 0, n // 3, 6, 3.0)
    bump(spec, 1, n // 2, 30, 1.8)
    ora = orc.search_harmonics(spec.cpu().numpy(), zmax, B, C, thr, numharm, log_sampling=log_sampling, per_width=True)
    ora = ora[np.lexsort((ora["width"], ora["bin"], ora["spectrum"], ora["numharm"]))]
    plan = binding.Plan(n, batch, zmax, C, thr, norm_block=B, numharm=numharm, log_sampling=log_sampling,
                        per_width_capacity=len(ora) + 10)
    plan.attach("cuda")
    assert plan.max_hcandidates == plan.max_candidates == len(ora) + 10
    plan.search_harmonics(spec)
    gpu = plan.hcandidates()
    assert plan.last_count == len(ora) > 20
    _assert_same_hcandidates(gpu, ora, f"per-width numharm={numharm} log={log_sampling}")
    plan.destroy()
    # too small an array: the count still reports everything found, only `capacity` records are written (all genuine)
    small = binding.Plan(n, batch, zmax, C, thr, norm_block=B, numharm=numharm, log_sampling=log_sampling, per_width_capacity=7)
    small.attach("cuda")
    small.search_harmonics(spec)
    part = small.hcandidates()
    assert small.last_count == len(ora) and len(part) == 7
    keys = set(zip(ora["numharm"].tolist(), ora["spectrum"].tolist(), ora["bin"].tolist(), ora["width"].tolist()))
    assert all(k in keys for k in zip(part["numharm"].tolist(), part["spectrum"].tolist(), part["bin"].tolist(), part["width"].tolist()))
    small.destroy()


def test_time_series_pipeline_on_one_stream(orc):
    """cuFFT (torch.fft.rfft) feeding pulscan_search on a side stream: the oracle gets the spectrum the search saw."""
    from paper_2406_15186_b200 import binding, pipeline
    wl = synth.CONFIGS[1]
    g = torch.Generator(device="cpu").manual_seed(11)
    t = torch.arange(wl.n_samples, dtype=torch.float64) * wl.tsamp
    x = torch.randn(2, wl.n_samples, generator=g, dtype=torch.float32)
    x[1] += (0.08 * torch.cos(2 * torch.pi * (173.2 * t + 0.5 * (12 / wl.t_obs ** 2) * t ** 2))).float()
    plan = binding.Plan(wl.n_bins, 2, wl.zmax, wl.block_width, 5.0, norm_block=wl.norm_block)
    plan.attach("cuda")
    side = torch.cuda.Stream()
    xd = x.cuda()
    side.wait_stream(torch.cuda.current_stream())
    spectrum = pipeline.search_time_series(plan, xd, side)
    side.synchronize()
    gpu = plan.candidates()
    plan.destroy()
    ora = oracle_search(orc, spectrum, wl.zmax, wl.norm_block, wl.block_width, 5.0)
    assert len(ora) > 0 and ora[np.argmax(ora["sigma"])]["spectrum"] == 1
    assert_same_candidates(gpu, ora, "time series -> rfft -> search on one stream")


@pytest.mark.parametrize("n,batch,zmax,B,C,thr", [(200001, 2, 4096, 8192, 4096, 5.0), (150000, 1, 3000, 4096, 100, 4.5),
                                                  (65537, 3, 1, 1024, 64, 4.0), (70000, 2, 513, 2048, 7, 4.5),
                                                  (33000, 1, 31, 512, 20000, 3.5)])
def test_pruned_equals_exhaustive_at_the_limits(n, batch, zmax, B, C, thr):
    """Beyond what the oracle finishes in seconds (zmax up to PULSCAN_MAX_ZMAX): the pruned sweep against the exhaustive one."""
    spec = noise_spectra(batch, n, seed=n + zmax)
    bump(spec, 0, n // 3, min(zmax, 200), 1.6)
    bump(spec, batch - 1, n // 2, 3, 4.0)
    a, stats = gpu_search(spec, zmax, B, C, thr, mode=0)
    b, _ = gpu_search(spec, zmax, B, C, thr, mode=1)
    assert len(a) > 0 and np.array_equal(a, b) and stats[3] == 0


def test_full_cell_list_falls_back_to_marking_tiles(orc):
    spec = noise_spectra(2, 50001, seed=99)
    ref, st_ref = gpu_search(spec, 64, 2048, 128, 3.0)
    got, st = gpu_search(spec, 64, 2048, 128, 3.0, cell_capacity=16)
    assert st_ref[3] == 0 and st_ref[2] > 16           # the default list holds every flagged cell of this input
    assert st[3] > 0 and st[0] >= st_ref[0]            # cells were dropped, so whole tiles were marked instead
    assert np.array_equal(ref, got)


def test_pitch_and_trials(orc):
    spec = noise_spectra(3, 6000, seed=321)
    bump(spec, 1, 1000, 12, 3.5)
    gpu, _ = gpu_search(spec, 24, 1024, 50, 3.5, n_bins=5555, n_trials=40.0)
    ora = oracle_search(orc, spec, 24, 1024, 50, 3.5, n_bins=5555, n_trials=40.0)
    assert_same_candidates(gpu, ora, "pitch>n, trials=40")


def test_empty_result_and_all_zero_input():
    spec = noise_spectra(2, 30000, seed=8)
    gpu, stats = gpu_search(spec, 32, 2048, 64, 9.5)
    assert len(gpu) == 0
    zeros = torch.zeros(1, 5000, dtype=torch.complex64, device="cuda")
    gpu, _ = gpu_search(zeros, 32, 1024, 64, 3.0)
    assert len(gpu) == 0                               # MAD = 0 everywhere → power 0 → nothing (R7)


def test_strong_signal_many_flagged_blocks(orc):
    wl = synth.CONFIGS[2].scaled(n_samples=1 << 18, zmax=200, norm_block=4096, block_width=200, n_fixed_random=0,
                                 fixed=(synth.Injection(0, 201.3, 0.3, 150.0), synth.Injection(0, 411.0, 0.2, 0.0)), seed=5)
    X, _ = synth.make_spectra(wl, device="cuda")
    gpu, stats = gpu_search(X, wl.zmax, wl.norm_block, wl.block_width, 6.0)
    ora = oracle_search(orc, X, wl.zmax, wl.norm_block, wl.block_width, 6.0)
    assert len(ora) >= 2
    assert_same_candidates(gpu, ora, "strong signals")
    assert stats[10] > 0       # warp-tasks with many flagged lanes marked their blocks directly (the sweep's strong-signal shortcut)
    # the same search with the shortcut off (a flag probability above 10^-3 disables it): identical candidates
    slow, sstats = gpu_search(X, wl.zmax, wl.norm_block, wl.block_width, 6.0, log10_p_flag=-2.9)
    assert sstats[10] == 0 and np.array_equal(gpu, slow)


def test_batch_rows_independent_on_gpu():
    spec = noise_spectra(4, 20000, seed=77)
    bump(spec, 2, 5000, 20, 2.5)
    full, _ = gpu_search(spec, 48, 2048, 100, 3.5)
    for b in range(4):
        alone, _ = gpu_search(spec[b:b + 1].contiguous(), 48, 2048, 100, 3.5)
        sub = full[full["spectrum"] == b]
        assert np.array_equal(alone["bin"], sub["bin"]) and np.array_equal(alone["width"], sub["width"])
        assert np.array_equal(alone["power"], sub["power"]) and np.array_equal(alone["sigma"], sub["sigma"])


def test_config1_full(orc):
    wl = synth.CONFIGS[1]
    X, inj = synth.make_spectra(wl)                     # host float64 FFT, as BASELINE config 1 specifies
    Xd = X.cuda()
    gpu, _ = gpu_search(Xd, wl.zmax, wl.norm_block, wl.block_width, wl.sigma_threshold)
    ora = oracle_search(orc, Xd, wl.zmax, wl.norm_block, wl.block_width, wl.sigma_threshold)
    assert_same_candidates(gpu, ora, "config 1")
    top = gpu[np.argmax(gpu["sigma"])]
    assert (int(top["bin"]), int(top["width"])) == (727, 14)


def test_first_search_of_a_fresh_plan_is_graph_capturable(orc):
    """pulscan_search allocates nothing and never synchronises, its FIRST call included (everything that needs the runtime
    happens in pulscan_plan_set_workspace): the first search of a fresh plan is captured into a CUDA graph on a side
    stream, replayed on two new inputs, and each replay gives the oracle's list."""
    from paper_2406_15186_b200 import binding
    n, batch, zmax, B, C, thr = 20001, 2, 40, 2048, 100, 4.0
    inputs = []
    for k in range(3):
        spec = noise_spectra(batch, n, seed=900 + k)
        bump(spec, k % batch, 3000 + 2500 * k, 10 + 5 * k, 2.5)
        inputs.append(spec)
    buf = torch.empty_like(inputs[0])
    plan = binding.Plan(n, batch, zmax, C, thr, norm_block=B)
    plan.attach("cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    buf.copy_(inputs[0])
    torch.cuda.synchronize()
    with torch.cuda.graph(graph, stream=side):
        plan.search(buf, torch.cuda.current_stream())       # the first pulscan_search this plan ever sees
    for k in (1, 2):
        buf.copy_(inputs[k])
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
        gpu = plan.candidates()
        ora = oracle_search(orc, inputs[k], zmax, B, C, thr)
        assert len(ora) > 0
        assert_same_candidates(gpu, ora, f"graph replay {k}")
    plan.destroy()


def test_setter_after_attach_needs_a_new_attach():
    from paper_2406_15186_b200 import binding
    spec = noise_spectra(1, 20001, seed=31)
    plan = binding.Plan(20001, 1, 40, 100, 4.0, norm_block=2048)
    plan.attach("cuda")
    plan.search(spec)
    assert plan.lib.pulscan_plan_set_trials(plan.handle, 10.0) == 0
    with pytest.raises(binding.PulscanError) as e:
        plan.search(spec)
    assert e.value.code == binding.PULSCAN_ENOWORKSPACE
    plan.attach("cuda")
    plan.search(spec)
    assert plan.lib.pulscan_plan_set_mode(plan.handle, 1) == 0   # the exhaustive sweep keeps the per-bin powers: new layout
    with pytest.raises(binding.PulscanError):
        plan.search(spec)
    plan.set_mode(1)                                         # the binding attaches again
    plan.search(spec)
    torch.cuda.synchronize()
    plan.destroy()


def test_host_staging_with_per_width_emission(orc):
    """pulscan_search_host under per-(block, width) emission: the staging area follows the caller's capacity and only
    min(found, capacity) records are copied back."""
    from paper_2406_15186_b200 import binding
    n, batch, zmax, B, C, thr = 20001, 1, 40, 2048, 5000, 3.0       # 5 blocks, capacity far above one record per block
    spec = noise_spectra(batch, n, seed=778)
    bump(spec, 0, n // 3, 6, 3.0)
    ora = orc.search_harmonics(spec.cpu().numpy(), zmax, B, C, thr, 1, per_width=True)
    assert len(ora) > 5 * 8
    for cap in (len(ora) + 5, 9):
        plan = binding.Plan(n, batch, zmax, C, thr, norm_block=B, host_staging=True, per_width_capacity=cap)
        plan.attach("cuda")
        hc = np.zeros(cap + 64, dtype=binding.CANDIDATE_DTYPE)       # 64 guard records behind the capacity
        got = plan.search_host(spec.cpu().pin_memory(), hc[:cap])
        assert plan.last_count == len(ora) and len(got) == min(cap, len(ora))
        assert not hc[cap:].view(np.uint8).any()                       # nothing written beyond the caller's capacity
        keys = set(zip(ora["bin"].tolist(), ora["width"].tolist()))
        assert all(k in keys for k in zip(got["bin"].tolist(), got["width"].tolist())) and np.all(got["width"] >= 1)
        plan.destroy()


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("n,batch,zmax,B,C,thr,numharm,log_sampling,mom", [
    (20001, 2, 40, 2048, 100, 4.0, 1, False, False), (9001, 2, 64, 4096, 200, 5.0, 3, False, False),
    (30011, 1, 129, 8192, 300, 6.0, 4, True, True),      # the paper's GPU-native configuration: Alg. 1 + Alg. 3 + log z + 4 harmonics
    (12001, 1, 300, 4096, 400, 6.0, 1, False, False)])   # wide widths: x = 1500·dof/pow > 1100, where Alg. 3 diverges and floods
def test_polynomial_logp_matches_oracle(orc, n, batch, zmax, B, C, thr, numharm, log_sampling, mom, mode):
    """Fast mode (Alg. 3): every ln p from the printed polynomial, on the device and in the oracle; the
    candidate lists (bins, widths exact; sigma = Φ_sf⁻¹(e^{ln p}) within 1e-3, i.e. ln p element by element) must agree."""
    from paper_2406_15186_b200 import binding
    spec = noise_spectra(batch, n, seed=n + 17 * numharm)
    bump(spec, 0, n // 3, 6, 3.0)
    bump(spec, batch - 1, n // 2, min(zmax, 30), 1.8)
    plan = binding.Plan(n, batch, zmax, C, thr, norm_block=B, mode=mode, numharm=numharm, log_sampling=log_sampling,
                        median_of_medians=mom, poly_logp=True)
    plan.attach("cuda")
    plan.search_harmonics(spec)
    gpu = plan.hcandidates()
    plan.destroy()
    ora = orc.search_harmonics(spec.cpu().numpy(), zmax, B, C, thr, numharm, log_sampling=log_sampling, median_of_medians=mom,
                               poly_logp=True)
    assert len(ora) > 0
    _assert_same_hcandidates(gpu, ora, f"Alg. 3 n={n} zmax={zmax} numharm={numharm} mode={mode}")
    exact = orc.search_harmonics(spec.cpu().numpy(), zmax, B, C, thr, numharm, log_sampling=log_sampling, median_of_medians=mom)
    if zmax <= 64 and numharm == 1:
        assert len(ora) <= len(exact)        # usable region: Alg. 3 under-states significance, marginal candidates drop out
    if zmax == 300:
        assert len(ora) > 2 * len(exact)     # divergent region: wide widths pass on pure noise


@pytest.mark.parametrize("n,B", [(4097, 1024), (12289, 4096), (8192, 4096), (16385, 8192), (2051, 512), (40000, 16384), (5003, 100),
                                 (1 << 16, 2048)])
def test_group_sums_and_block_statistics_rebuild_the_powers(orc, n, B):
    """What the default search keeps in HBM instead of the per-bin powers: G[k] = (P[4k]+P[4k+1]) + (P[4k+2]+P[4k+3]) in
    float32, bit for bit, and per-block (a, inv, k) from which every P is rebuilt bit for bit with the same FMAs."""
    from paper_2406_15186_b200 import binding
    spec = noise_spectra(3, n, seed=n + B)
    spec[1] = spec[1] * 1e-3 + (5.0 - 2.0j)
    plan = binding.Plan(n, 3, min(8, n - 1), 16, 6.0, norm_block=B)
    plan.attach("cuda")
    P = plan.normalise_power(spec)
    G, st = plan.normalise_group_sums(spec, B)
    plan.destroy()
    Pp = torch.zeros((3, 4 * ((n + 3) // 4)), dtype=torch.float32, device="cuda")
    Pp[:, :n] = P
    q = Pp.view(3, -1, 4)
    want = (q[:, :, 0] + q[:, :, 1]) + (q[:, :, 2] + q[:, :, 3])
    assert torch.equal(G, want)
    nb = max(1, n // B)
    blk = torch.clamp(torch.arange(n, device="cuda") // B, max=nb - 1)
    a0, i0, k0, a1, i1, k1 = (st[:, :, c][:, blk].double() for c in range(6))
    x = (spec.real.float() - a0.float()).double() * i0 + k0         # fma = one rounding of the exact product-sum: emulate in double
    y = (spec.imag.float() - a1.float()).double() * i1 + k1
    x, y = x.float().double(), y.float().double()
    rebuilt = (x * x + (y * y).float().double()).float()
    assert torch.equal(rebuilt, P)
    ref = orc.normalise_power(spec[0].cpu().numpy(), B)              # and the statistics are the paper's: median and κ·MAD
    assert np.all(np.abs(P[0].cpu().numpy() - ref) <= 1e-5 * ref + 1e-6)


@pytest.mark.parametrize("n,zmax,B,C,thr,tile", [
    (200001, 200, 4096, 200, 5.0, 0),        # 8448-bin tiles: one scan pass of 9 quads per thread, group-sum input
    (200001, 1200, 8192, 1200, 5.0, 0),      # 9472-bin tiles: one pass of 11 quads per thread
    (200001, 3000, 8192, 1024, 5.0, 16384),  # 16384-bin tiles + halo: several passes of 5 quads per thread
    (60001, 100, 2048, 100, 5.0, 2048),      # small tiles: one pass of 5
])
def test_sweep_second_look_and_scan_variants(orc, n, zmax, B, C, thr, tile):
    """The sweep's own second look at a flagged cell (half-group covers, boxcar_sweep.cuh sweep_confirm_cell) only removes
    cells that cannot hold a window above threshold: the candidates equal those of a plan built without it (and the oracle's),
    while fewer cells reach the refine kernel; run for every quads-per-thread variant of the tile scan."""
    spec = noise_spectra(2, n, seed=n + zmax)
    bump(spec, 0, n // 3, min(zmax, 150), 1.5)
    bump(spec, 1, n // 2, 9, 2.5)
    got, stats = gpu_search(spec, zmax, B, C, thr, tile=tile)
    assert stats[9] >= stats[2] > 0 and stats[3] == 0        # flagged ≥ listed after the second look; nothing dropped
    from paper_2406_15186_b200 import binding
    ref, rstats = gpu_search(spec, zmax, B, C, thr, tile=tile, variants={binding.VARIANT_SWEEP_SECOND_LOOK: 0})
    assert np.array_equal(got, ref) and len(got) > 0
    assert rstats[2] == rstats[9] >= stats[2]                 # without the τ_h tables every flagged cell is listed
    assert_same_candidates(got, oracle_search(orc, spec, zmax, B, C, thr), f"zmax={zmax} tile={tile}")


# ---- exact ties (R14: "lowest such i"; Alg. 4 L696-712 scans start bins in ascending order and replaces on `>` only)
TIE_CASES = [
    # n, zmax, B, C, thr, block, offset of the first pulse, offset of the second          kernel (c) geometry
    (5000, 2, 1024, 64, 4.0, 3, 8, 10),         # both start bins inside one 4 x 4 register tile; no window covers both
    (5000, 7, 1024, 500, 4.0, 1, 13, 400),      # small zmax: the start bins of a block are split over lanes (lg_split > 0)
    (30011, 4096, 8192, 2000, 4.0, 1, 100, 1500),   # zmax·C = 8.2 M: the widths of a block are dealt to 2 CTAs (parts > 1)
]


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("n,zmax,B,C,thr,blk,o1,o2", TIE_CASES)
def test_exact_ties_go_to_the_lowest_bin(orc, mode, n, zmax, B, C, thr, blk, o1, o2):
    """Two bins of one normalisation block and one candidate block hold the same complex value: their float32 powers are
    bit-identical, S(i, 1) ties exactly in kernel (c)'s double sums, and the block's record must name the LOWER bin (R14),
    as the oracle's does.  The pulses are strong enough for width 1 to win the block and far enough apart (or zmax small
    enough) that no wider window beats it by covering both."""
    from paper_2406_15186_b200 import binding
    spec = noise_spectra(1, n, seed=31 * n + zmax)
    i1, i2 = blk * C + o1, blk * C + o2
    assert i1 // B == i2 // B and i1 // C == i2 // C == blk
    for i in (i1, i2):
        spec[0, i - 2:i + 3] *= 0.05                                  # quiet neighbours: width 1 wins at the pulse
    for i in (i1, i2):
        spec[0, i] = complex(17.0 * 50.0, -17.0 * 50.0)                # P = 17² ≈ 290 in mean-1 units
    plan = binding.Plan(n, 1, zmax, C, thr, norm_block=B)
    P = plan.normalise_power(spec).cpu().numpy()
    plan.destroy()
    assert P[0, i1] == P[0, i2] and P[0, i1] > 200                     # an exact float32 tie
    ref = oracle_search(orc, spec, zmax, B, C, thr)
    hit = ref[(ref["bin"] // C == blk)]
    assert len(hit) == 1 and hit["bin"][0] == i1 and hit["width"][0] == 1, hit   # the oracle resolves the tie downwards
    got, _ = gpu_search(spec, zmax, B, C, thr, mode=mode)
    assert_same_candidates(got, ref, f"tie at bins {i1}, {i2} mode={mode}")


@pytest.mark.parametrize("which,value", [(2, 5), (3, 0), (3, 1), (4, 0), (4, 37), (5, 0), (6, 1)])
def test_kernel_variants_never_change_results(orc, which, value):
    """pulscan_plan_set_variant switches kernel variants and the workspace layout, never a candidate."""
    n, zmax, B, C, thr = 60001, 100, 2048, 100, 4.5
    spec = noise_spectra(2, n, seed=99)
    bump(spec, 0, n // 3, 60, 1.6)
    bump(spec, 1, n // 2, 5, 3.0)
    base, _ = gpu_search(spec, zmax, B, C, thr)
    got, _ = gpu_search(spec, zmax, B, C, thr, variants={which: value})
    assert np.array_equal(base, got) and len(got) > 0
    assert_same_candidates(got, oracle_search(orc, spec, zmax, B, C, thr), f"variant {which} = {value}")


# ---- candidate blocks too long for one shared-memory prefix array: kernel (c) walks them in segments
def _long_block_spectrum(n, zmax, seed):
    """Noise + pulses in several segments of block 0 (segments are ≈ 15-25 k start bins), one in the last ragged block, and
    two identical single-bin pulses in one normalisation block that fall in different segments when the block is cut at
    25216 start bins (zmax 256): an exact tie across segments, which must go to the lower bin (R14)."""
    spec = noise_spectra(1, n, seed=seed)
    bump(spec, 0, 3000, min(zmax, 20), 1.9)
    bump(spec, 0, 29000, min(zmax, 60), 1.6)
    bump(spec, 0, n - 1500, 9, 2.2)
    for i in (25000, 26000):
        spec[0, i - 2:i + 3] *= 0.05
    for i in (25000, 26000):
        spec[0, i] = complex(12.0 * 50.0, 12.0 * 50.0)
    return spec


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("n,zmax,B,C,thr,r_block", [
    (200001, 256, 8192, 32768, 4.5, True),     # the paper's R-Block setting (Table 3): 2 segments per block
    (200001, 256, 8192, 32768, 4.5, False),
    (100001, 4096, 8192, 30000, 4.5, False),   # 2 segments of 15616 start bins, the widths of a block dealt to 8 CTAs
    (70001, 100, 4096, 70001, 4.0, False),     # one block = the whole spectrum, 3 segments
])
def test_long_candidate_blocks_are_walked_in_segments(orc, mode, n, zmax, B, C, thr, r_block):
    from paper_2406_15186_b200 import binding
    spec = _long_block_spectrum(n, zmax, seed=n + zmax)
    plan = binding.Plan(n, 1, zmax, C, thr, norm_block=B)
    assert "1 segment(s)" not in plan.describe().split("exact:")[1]
    P = plan.normalise_power(spec).cpu().numpy()
    plan.destroy()
    assert P[0, 25000] == P[0, 26000] > 100
    ref = oracle_search(orc, spec, zmax, B, C, thr, r_block=r_block)
    got, _ = gpu_search(spec, zmax, B, C, thr, mode=mode, r_block=r_block)
    assert len(ref) >= 1
    assert_same_candidates(got, ref, f"C={C} zmax={zmax} mode={mode} r_block={r_block}")


def test_long_candidate_blocks_tie_across_segments_and_per_width_emission(orc):
    """Every width's maximum is carried over the segments before ln p is taken: per-(block, width) emission gives exactly one record per (block, width), and the width-1 record of block 0 names bin 25000,
    the lower of the two tied bins, which sit in different segments."""
    from paper_2406_15186_b200 import binding
    n, zmax, B, C, thr = 120001, 64, 8192, 32768, 4.0
    spec = _long_block_spectrum(n, zmax, seed=5)
    ora = orc.search_harmonics(spec.cpu().numpy(), zmax, B, C, thr, 1, per_width=True)
    ora = ora[np.lexsort((ora["width"], ora["bin"], ora["spectrum"]))]
    plan = binding.Plan(n, 1, zmax, C, thr, norm_block=B, per_width_capacity=len(ora) + 16)
    plan.attach("cuda")
    plan.search(spec)
    got = plan.candidates()
    plan.destroy()
    assert plan.last_count == len(ora) == len(got)
    assert_same_candidates(got, ora, "per-width emission over segmented blocks")
    w1 = got[(got["width"] == 1) & (got["bin"] // C == 0)]
    assert len(w1) == 1 and w1["bin"][0] == 25000


def test_long_candidate_blocks_with_polynomial_logp(orc):
    """Alg. 3's ln p is not monotone in the power: it must be taken at the block maximum of a width, not per segment."""
    from paper_2406_15186_b200 import binding
    n, zmax, B, C, thr = 100001, 90, 8192, 32768, 6.0
    spec = _long_block_spectrum(n, zmax, seed=8)
    plan = binding.Plan(n, 1, zmax, C, thr, norm_block=B, poly_logp=True)
    plan.attach("cuda")
    plan.search_harmonics(spec)
    gpu = plan.hcandidates()
    plan.destroy()
    ora = orc.search_harmonics(spec.cpu().numpy(), zmax, B, C, thr, 1, poly_logp=True)
    assert len(ora) >= 2
    _assert_same_hcandidates(gpu, ora, "Alg. 3 over segmented blocks")
