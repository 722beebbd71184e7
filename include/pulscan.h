/*
 * pulscan.h — C ABI of libpulscan: the data-parallel hot path of Pulscan (White et al., arXiv 2406.15186),
 * the unmatched-filter (boxcar) acceleration search over the Fourier spectrum of a dedispersed observation,
 * as hand-written sm_100a CUDA.  Citations are PAPER.md line numbers; "R<n>" are the readings in DESIGN.md §3.
 *
 * What one search computes, per spectrum of a batch (§2.2.3-2.2.5):
 *   1. per normalisation block, per component (re, im independently): v' = (v − median)/(κ·MAD), κ = 1/Φ⁻¹(¾)
 *      (L140-148, Eq. 8); exact medians; the last block absorbs n_bins mod norm_block (R6); MAD = 0 → block = 0 (R7)
 *   2. power P = (re'² + im'²)/2 (L150; halved so that noise has mean 1, R2)
 *   3. boxcar sums S(i,w) = Σ_{j<w} P[i+j] for every width w in [1, zmax] and every bin i with i + w ≤ n_bins
 *      (L152, L169-199; R9-R11)
 *   4. per candidate block c = [c·block_width, (c+1)·block_width) of start bins and per width: the maximum and
 *      its lowest arg-max (Alg. 4; R12, R14)
 *   5. ln p = ln Q(w, S): χ² survival with 2w degrees of freedom at 2S (L154-158, Eq. 9), plus ln n_trials
 *      (Bonferroni, L158, R15); σ = the Gaussian-equivalent significance (L114, L158; R16)
 *   6. per block the width with the smallest ln p (largest σ; smallest width on ties, R13); the candidate
 *      (spectrum, bin, width, power, sigma) is emitted iff σ ≥ sigma_threshold (L342-344, L361; R17)
 * so at most one candidate per (spectrum, candidate block).
 *
 * Conventions.  All `d_` pointers are DEVICE pointers, all `h_` pointers are HOST pointers; the library never
 * takes ownership of either and owns no device memory of its own (its small threshold tables live in the caller's
 * workspace).  Every function returns PULSCAN_OK (0) or a negative error code and never throws;
 * pulscan_last_error() describes the last failure on the calling thread.  There is no CPU fallback: without a
 * CUDA device of compute capability 10.x pulscan_plan_set_workspace returns PULSCAN_ECUDA / PULSCAN_EARCH.
 *
 * Life of a plan.  (1) configure: pulscan_plan_create and the pulscan_plan_set_* calls are host-only and touch no CUDA
 * device.  (2) finalise: pulscan_plan_set_workspace checks the device, uploads the tables into the workspace (synchronous
 * copies), sets the kernels' shared-memory attributes on the CURRENT device and fixes the launch shapes — the only place
 * besides the launches that calls the CUDA runtime.  (3) search: pulscan_search / pulscan_search_harmonics allocate
 * nothing and never synchronise, from their first call on (the first search of a fresh plan can be captured into a CUDA
 * graph).  A setter that changes derived state or the workspace layout (every setter except _set_r_block, and
 * _set_emission without host staging) returns the plan to step (1): searches then fail with PULSCAN_ENOWORKSPACE until
 * pulscan_plan_set_workspace is called again (pulscan_plan_workspace_bytes may have changed).
 *
 * One search at a time per plan.  The counters, the block bitmap, the cell and block lists, the intermediate arrays and the
 * profiling slots all live in the plan's one workspace: two searches of the SAME plan that can overlap on the GPU (two streams)
 * or that are enqueued from two host threads at once race with each other.  Searches on one stream, one after the other, are
 * the supported use; for concurrent searches create one plan (and workspace) per stream.  Different plans are independent,
 * except for pulscan_normalise_power_static, whose calls share one array per device.
 */
#ifndef PULSCAN_H
#define PULSCAN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PULSCAN_OK 0
#define PULSCAN_EINVAL (-1)       /* bad argument (range, null, alignment, plan state)                   */
#define PULSCAN_ENOWORKSPACE (-2) /* no workspace attached, or it is too small                           */
#define PULSCAN_ECUDA (-3)        /* a CUDA runtime call or kernel launch failed                         */
#define PULSCAN_EARCH (-4)        /* the current device is not compute capability 10.x (B200, sm_100a)   */

/* Limits of this build (PULSCAN_EINVAL beyond them). */
#define PULSCAN_MAX_ZMAX 4096
#define PULSCAN_MAX_NORM_BLOCK 16384
#define PULSCAN_MAX_BLOCK_WIDTH (1 << 24) /* candidate blocks with block_width + zmax > 24576 are evaluated in segments */

typedef struct pulscan_plan pulscan_plan; /* opaque */

/* One candidate: 20 bytes, no padding.  `bin` is the first bin of the window (R10), `width` = w (the paper's
 * drift z = w − 1, R9), `power` = S(bin, width) in mean-1 units, `sigma` single-precision (R21). */
typedef struct {
    int32_t spectrum;
    int32_t bin;
    int32_t width;
    float power;
    float sigma;
} pulscan_candidate;

/* One candidate of the harmonic-summed search (pulscan_search_harmonics): 24 bytes, no padding.  `numharm` = H, the number
 * of harmonics summed into the spectrum Y_H the candidate was found in (1 = the plain power spectrum); `bin` is a bin of
 * Y_H, i.e. of the fundamental (L218 "aligned so the 0th bin of each spectrum is summed"); `power` = the boxcar sum of Y_H
 * in mean-1 units (mean H(H+1)/2 per bin in noise). */
typedef struct {
    int32_t spectrum;
    int32_t bin;
    int32_t width;
    int32_t numharm;
    float power;
    float sigma;
} pulscan_hcandidate;

/* Create a plan for `batch` spectra of `n_bins` complex64 bins each, boxcar widths 1..zmax, candidate blocks of
 * `block_width` start bins (Alg. 4's chunk_size; L224 "block width is a user defined parameter") and a
 * Gaussian-σ threshold (L361).  Host-only: touches no CUDA device.  Defaults: norm_block = next power of two
 * ≥ 16·block_width clamped to [1024, 8192]; n_trials = 1; pitch = n_bins.
 * Returns NULL on error (n_bins < 2, batch < 1, zmax < 1 or ≥ n_bins or > PULSCAN_MAX_ZMAX, block_width < 1,
 * or > PULSCAN_MAX_BLOCK_WIDTH, sigma_threshold ≤ 0 or not finite, batch·blocks ≥ 2³¹). */
pulscan_plan* pulscan_plan_create(int64_t n_bins, int32_t batch, int32_t zmax, int32_t block_width,
                                  float sigma_threshold);

/* Normalisation block B in bins (L142 "the input data is divided into blocks"): 2 ≤ B ≤ PULSCAN_MAX_NORM_BLOCK. */
int pulscan_plan_set_norm_block(pulscan_plan* plan, int32_t norm_block);

/* Bonferroni trial count N ≥ 1 (L158): p_adj = min(1, N·p).  Default 1 = single-trial σ (R15). */
int pulscan_plan_set_trials(pulscan_plan* plan, double n_trials);

/* Row stride of the input in complex64 bins, ≥ n_bins.  Default n_bins (dense rows). */
int pulscan_plan_set_pitch(pulscan_plan* plan, int64_t pitch_bins);

/* Search mode: 0 = pruned sweep (default; exact — cover-sum upper bounds only discard windows that cannot reach
 * their width's power threshold), 1 = exhaustive sweep (every (bin, width) evaluated; the cross-check; it keeps the
 * float32 power of every bin in the workspace, so the workspace grows and must be attached again). */
int pulscan_plan_set_mode(pulscan_plan* plan, int32_t mode);

/* Which boxcar widths are SEARCHED for candidates; all widths are still summed (L152 "the user can select the step size to
 * determine which boxcar filtered spectra are searched").  With drift z = width − 1 (R9): z_step ≥ 1 searches z = 0,
 * z_step, 2·z_step, … (Alg. 4: remainder(z / z_step) = 0); logarithmic ≠ 0 searches z = 0, 1, 2, 4, 8, … instead
 * (L411 "z = 1, 2, 4, 8, ... z-max", the paper's GPU default; z = 0, the unfiltered spectrum, is kept: reading R28) and
 * ignores z_step.  Default: z_step = 1, every width (north_star).  The reduction over widths (step 6) then runs over the
 * searched widths only; pulscan_plan_get_thresholds() reports +inf for the others. */
int pulscan_plan_set_width_sampling(pulscan_plan* plan, int32_t z_step, int32_t logarithmic);

/* "Pulscan R-Block" (L222-226 §2.4): save only the block index of a candidate, "an approximate frequency location".
 * enable ≠ 0: a record's `bin` is the first bin of its candidate block, block index × block_width (Table 3:
 * 360448 = 11 × 32768); width, power and sigma are unchanged.  Default 0: the exact first bin of the window.
 * The paper's own setting, block_width = 32768 (L224 "the default value of 32768 was used for all Pulscan R-Block tests"), is
 * within range: kernel (c) walks such a block in segments. */
int pulscan_plan_set_r_block(pulscan_plan* plan, int32_t enable);

/* Harmonic sum (L201-220 §2.3; `-numharm`): numharm ∈ [1, 4].  pulscan_search_harmonics() then also searches the summed
 * spectra Y_H(r) = Σ_{h≤H} Σ_{j<h} P[h·r + j], r < floor(n_bins/H) (R29), H = 2..numharm, each "boxcar filtered as
 * previously described" with χ² of H(H+1)·width degrees of freedom (L220).  Needs zmax < floor(n_bins/numharm).  Changes
 * pulscan_plan_workspace_bytes().  Default 1.  pulscan_search() is not affected. */
int pulscan_plan_set_harmonics(pulscan_plan* plan, int32_t numharm);
/* Capacity the caller must give d_hcandidates: Σ_{H ≤ numharm} batch · ceil(floor(n_bins/H) / block_width) records. */
int64_t pulscan_plan_max_hcandidates(const pulscan_plan* plan);
/* pulscan_search on Y_1 (the power spectrum) … Y_numharm: same contract as pulscan_search (device pointers, asynchronous, no
 * allocation); at most one record per candidate block of each Y_H; *d_count is zeroed first and ends as the total. */
int pulscan_search_harmonics(pulscan_plan* plan, const void* d_spectra, pulscan_hcandidate* d_hcandidates, uint32_t* d_count,
                             void* cuda_stream);

/* Normalisation method.  0 (default): exact median and MAD per block and component (L140-148, Eq. 8).  1: the paper's GPU
 * method, Algorithm 1 "Median of Medians Normalisation" (L624-650; §2.5) — an approximation: the median of a chunk is
 * estimated by recursively taking the median of 4 strided elements, the MAD likewise, scale factor 1.4826 (L648).  Needs
 * norm_block = a power of two in [256, 16384] (set it first) and n_bins ≥ norm_block; the n_bins mod norm_block bins after
 * the last chunk use the last chunk's statistics (reading R30).  Powers come out ≈ 12 % low in noise (the median of 4
 * over-estimates the median of the skewed |deviation| distribution), so it is a fast mode, not the parity path. */
int pulscan_plan_set_normalisation(pulscan_plan* plan, int32_t mode);

/* Significance function.  0 (default): the exact χ² tail, ln p = ln Q(shape, S) (L154-158, Eq. 9).  1: the paper's GPU method,
 * Algorithm 3 "Power to Log Probability Calculation" (L656-662; §2.6 Eq. 10-12): ln p ≈ pow·f(x)/1500 with
 * x = 1500·dof/pow, f the printed degree-16 polynomial, and ln p = 0 when dof ≥ 1.05·pow; called with the paper's units
 * pow = 2S, dof = 2·shape (R31).  The reduction over widths, the threshold and sigma then use that value, and the per-width
 * power thresholds of the sweep follow it.  An APPROXIMATION, error-profiled in DESIGN.md §9: 0 … 4.5 nats less significant
 * than the exact tail while x ≲ 1000 (widths ≲ 150 at σ 6), divergent beyond (the printed 8-digit coefficients no longer
 * determine f): a fast mode, not the parity path.  The plan must be attached again afterwards. */
int pulscan_plan_set_significance(pulscan_plan* plan, int32_t mode);

/* What is emitted per candidate block.  per_width = 0 (default): the width with the largest σ (step 6 above, R13), at most
 * one record per block.  per_width = 1: the paper's GPU output, one record per (block, searched width) whose maximum reaches
 * the threshold (Alg. 4 "write out local candidate", ranked by σ afterwards, L322) — `capacity` records must then
 * be provided for d_candidates / d_hcandidates (pulscan_plan_max_candidates() returns it); *d_count reports the number
 * found and only the first `capacity` of them are written. */
int pulscan_plan_set_emission(pulscan_plan* plan, int32_t per_width, int64_t capacity);

/* Tuning of the pruned sweep: tile_bins (multiple of 512, 1024..16384; 0 = default) and the per-cover false-flag
 * probability in noise as log10 (−1 … −9; 0 = default).  Affects speed only, never results. */
int pulscan_plan_set_tuning(pulscan_plan* plan, int32_t tile_bins, double log10_p_flag);

/* Kernel variants: comparison and tuning switches that change which kernel variant runs or how the workspace is laid out,
 * NEVER a result (the GPU tests run the parity suite's cases with them).  They replace the environment variables the library
 * read until round 2; the only one left is PULSCAN_DEBUG_SYNC (any value: cudaDeviceSynchronize after every launch so that a
 * device fault is reported by the launch that caused it; a debugging aid, never on a timed or captured path).
 *   PULSCAN_VARIANT_SWEEP_SECOND_LOOK      1 (default) / 0: the sweep re-tests a flagged cell against half-group thresholds itself
 *   PULSCAN_VARIANT_SCAN_QUADS             0 (default: 5, 9 or 11 quads per thread by tile length) / 5: the multi-pass scan
 *   PULSCAN_VARIANT_NORM_KEEP_INDICES      -1 (default: by norm_block) / 0 / 1: kernel (a) keeps bucket indices in registers
 *   PULSCAN_VARIANT_NORM_L2_AHEAD          -1 (default: 4 x SMs) / n >= 0: CTAs of L2 look-ahead of kernel (a), 0 = off
 *   PULSCAN_VARIANT_NORM_SINGLE_HISTOGRAM  1 (default) / 0: every normalisation block through the general select kernel
 *   PULSCAN_VARIANT_KEEP_POWER             0 (default) / 1: keep the float32 power of every bin in the workspace (4 B/bin)
 *                                          even where the sums of 4-bin groups would do
 * Like every setter that changes derived state: the workspace must be attached again (its size may change). */
#define PULSCAN_VARIANT_SWEEP_SECOND_LOOK 1
#define PULSCAN_VARIANT_SCAN_QUADS 2
#define PULSCAN_VARIANT_NORM_KEEP_INDICES 3
#define PULSCAN_VARIANT_NORM_L2_AHEAD 4
#define PULSCAN_VARIANT_NORM_SINGLE_HISTOGRAM 5
#define PULSCAN_VARIANT_KEEP_POWER 6
int pulscan_plan_set_variant(pulscan_plan* plan, int32_t which, int32_t value);

/* Capacity (in cells, 8 bytes each) of the list that carries flagged cover cells from the sweep to its refine kernel;
 * 0 = default (max(65536, batch·n_bins/256): ≈ 25× what noise flags at the default p_flag).  When the list is full the
 * sweep marks every candidate block of the affected tile instead, so the setting affects speed only, never results.
 * Changes pulscan_plan_workspace_bytes(). */
int pulscan_plan_set_cell_capacity(pulscan_plan* plan, int64_t cells);

/* Capacity the caller must give d_candidates: batch · ceil(n_bins / block_width) records. */
int64_t pulscan_plan_max_candidates(const pulscan_plan* plan);

/* Scratch the caller must provide (device memory, 256-byte aligned): the sums of 4-bin groups of the power spectrum
 * [batch][group_pitch] and 32 bytes per normalisation block (or, in exhaustive mode / with levels finer than 4 bins / for
 * the harmonic search / with the Alg. 1 normalisation, the float32 power of every bin [batch][power_pitch]), the
 * flagged-cell and flagged-block lists, counters and the threshold tables.  With host staging enabled it also holds a
 * device copy of the input for pulscan_search_host.  pulscan_plan_set_workspace FINALISES the plan (see "Life of a plan"):
 * it is synchronous, must be called with the target device current, and again after any setter that changes the plan. */
size_t pulscan_plan_workspace_bytes(const pulscan_plan* plan);
int pulscan_plan_enable_host_staging(pulscan_plan* plan, int32_t enable);
int pulscan_plan_set_workspace(pulscan_plan* plan, void* d_workspace, size_t bytes);

/* Run the whole path on the device.  d_spectra: complex64 [batch][pitch] (interleaved re, im float32; 8-byte
 * aligned; read-only; it must stay valid until the search has finished: flagged spans are rebuilt from it).
 * d_candidates: pulscan_plan_max_candidates() records.  d_count: one uint32, zeroed by the call, then the number of
 * candidates.  Enqueues memsets and kernels on `cuda_stream` (a cudaStream_t; NULL = default stream) and nothing else:
 * no allocation, no synchronisation, no other runtime call — on every call, the first included (CUDA-graph capturable);
 * the order of the records is unspecified (R19).  PULSCAN_ENOWORKSPACE if the plan is not finalised. */
int pulscan_search(pulscan_plan* plan, const void* d_spectra, pulscan_candidate* d_candidates, uint32_t* d_count,
                   void* cuda_stream);

/* The same search from HOST buffers: copies h_spectra (complex64 [batch][pitch]; pinned memory recommended) to
 * the staging area of the workspace, searches, copies the count and the records back to h_count /
 * h_candidates (capacity pulscan_plan_max_candidates()) and synchronises the stream before returning.
 * Requires pulscan_plan_enable_host_staging(plan, 1) before the workspace was sized and attached. */
int pulscan_search_host(pulscan_plan* plan, const void* h_spectra, pulscan_candidate* h_candidates,
                        uint32_t* h_count, void* cuda_stream);

/* Steps 1-2 only (normalise + power), for unit tests and profiling: d_power receives float32
 * [batch][pulscan_plan_power_pitch()] (bins ≥ n_bins of a row are unspecified). */
int pulscan_normalise_power(pulscan_plan* plan, const void* d_spectra, float* d_power, void* cuda_stream);
int64_t pulscan_plan_power_pitch(const pulscan_plan* plan);

/* Steps 1-2 (L140-150, Eq. 8: exact median/MAD normalisation, then the power) for a caller that cannot allocate device memory.
 * Who that is: a stage of a telescope back-end whose device memory was all handed out as ring buffers when the pipeline
 * started, a plug-in inside a host application that owns the allocator and passes the plug-in nothing but its input and
 * output buffers, code on a latency-critical path where cudaMalloc's device-wide synchronisation is not acceptable.  Such a
 * caller has no workspace to give pulscan_plan_set_workspace, and without one pulscan_normalise_power falls back to its slower
 * general kernels.  This entry point runs the same fast kernels as pulscan_search; the scratch they need (the list of blocks
 * handed to the general kernel, a few counters) is a fixed array inside the library image instead of caller memory.
 *   - It calls no cudaMalloc / cudaFree and no library routine that allocates; the plan needs NO workspace (an attached one is
 *     ignored).  The caller passes d_spectra and d_power exactly as for pulscan_normalise_power (same layout, alignment, result).
 *   - Limit: batch · max(1, n_bins div norm_block) ≤ PULSCAN_STATIC_MAX_NORM_BLOCKS, else PULSCAN_EINVAL (checked on the host
 *     before anything is enqueued).  The array is 4 bytes per block + 256 bytes ≈ 1 MiB and stays resident on every GPU the
 *     process uses with this library until the process exits, whether or not this function is ever called.
 *   - The first call on each device looks the array's device address up and sets kernel attributes on that device (with the
 *     target device current, as for every call).  Make that first call outside any stream capture; later calls only enqueue
 *     one 256-byte memset and the kernels on `cuda_stream`.
 *   - All calls on one device share the one array.  Every call zeroes the counters it needs before its kernels run, so
 *     back-to-back calls on one stream are fine whatever the previous call left behind; two calls that can overlap on the GPU
 *     (different streams, different host threads, different plans) race on it and corrupt each other's output.  Serialise them.
 *   - PULSCAN_EINVAL for a plan set to the Alg. 1 normalisation: that kernel needs no scratch, pulscan_normalise_power already
 *     allocates nothing for it. */
#define PULSCAN_STATIC_MAX_NORM_BLOCKS 262144
int pulscan_normalise_power_static(pulscan_plan* plan, const void* d_spectra, float* d_power, void* cuda_stream);

/* Steps 1-2 in the form the default search keeps them in HBM (for unit tests and profiling): instead of the power of every
 * bin, d_group_sums receives float32 [batch][pulscan_plan_group_pitch()] with G[k] = (P[4k] + P[4k+1]) + (P[4k+2] + P[4k+3])
 * (bins ≥ n_bins count as 0; entries ≥ ceil(n_bins/4) are unspecified), and d_block_stats float32
 * [batch][max(1, n_bins div norm_block)][8] with, per normalisation block, (a, inv, k) of the real parts then of the imaginary
 * parts (two unused floats): x' = fma(v − a, inv, k) is the normalised component ((v − median)/(κ·MAD)/√2: a = the lower central
 * value, k = −(median − a)·inv) and P = fma(x', x', y'·y').  Needs norm_block % 4 = 0, the exact normalisation and an
 * attached workspace; both arrays 32-byte aligned. */
int pulscan_normalise_group_sums(pulscan_plan* plan, const void* d_spectra, float* d_group_sums, float* d_block_stats,
                                 void* cuda_stream);
int64_t pulscan_plan_group_pitch(const pulscan_plan* plan);

/* Introspection (host only).  thresholds: h_T[w−1] = the power at which width w reaches the σ threshold
 * (zmax doubles).  describe: a human-readable dump of the plan (levels of the pruned sweep, sizes); returns the
 * number of bytes needed including the terminator.  stats: after the stream has been synchronised, h_stats[0] =
 * candidate blocks flagged by the sweep in the last search, h_stats[1] = normalisation blocks the fast kernel handed
 * to the general path, h_stats[2] = cover cells the sweep listed for its refine kernel (after its own second look),
 * h_stats[3] = cells dropped because the list was full (their tiles' blocks are all marked),
 * h_stats[4..8] = why blocks were handed over (geometry, search window, list capacity, verification,
 * degenerate sample), h_stats[9] = cover cells flagged by the sweep's cover sums before its second look,
 * h_stats[10] = flagged lanes of the sweep whose blocks were marked directly (strong signals), h_stats[11..15] reserved.  h_stats must hold 16 values. */
int pulscan_plan_get_thresholds(const pulscan_plan* plan, double* h_T);
int64_t pulscan_plan_describe(const pulscan_plan* plan, char* h_buf, int64_t buf_bytes);
int pulscan_plan_get_stats(pulscan_plan* plan, uint32_t* h_stats, void* cuda_stream);
/* Kernels one pulscan_search() enqueues for this plan (memsets not counted). */
int32_t pulscan_plan_launches_per_search(const pulscan_plan* plan);

/* Per-kernel timing.  set_profiling(n_slots > 0) creates 5·n_slots CUDA events (needs a current device) and makes every pulscan_search record them on its stream
 * around its stages into slot (search index mod n_slots); get_profile waits for that search and returns
 * h_ms[0..3] = milliseconds of {workspace memsets, kernel (a) normalise+power, kernel (b) sweep, kernel (c) exact
 * evaluation + significance + compaction}.  n_slots = 0 (default) records nothing. */
int pulscan_plan_set_profiling(pulscan_plan* plan, int32_t n_slots);
int pulscan_plan_get_profile(pulscan_plan* plan, int32_t slot, float* h_ms);

int pulscan_plan_destroy(pulscan_plan* plan);

const char* pulscan_last_error(void);
const char* pulscan_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PULSCAN_H */
