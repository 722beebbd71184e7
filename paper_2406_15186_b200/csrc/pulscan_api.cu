// pulscan_api.cu — the C ABI of libpulscan (include/pulscan.h): plan construction (host only), workspace layout,
// and the enqueue of the three kernels of one search.  No PyTorch, no allocation and no synchronisation on the
// search path; there is no CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/pulscan.h"
#include "block_exact.cuh"
#include "boxcar_sweep.cuh"
#include "harmonic_sum.cuh"
#include "norm_power.cuh"
#include "norm_power_mom.cuh"
#include "norm_power_v2.cuh"
#include "significance.cuh"

using namespace pulscan;

namespace {

thread_local std::string g_last_error;

int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_last_error = buf;
    return code;
}

#define CUDA_TRY(expr)                                                                                       \
    do {                                                                                                     \
        cudaError_t e_ = (expr);                                                                             \
        if (e_ != cudaSuccess) return fail(PULSCAN_ECUDA, "%s failed: %s", #expr, cudaGetErrorString(e_));  \
    } while (0)

// PULSCAN_DEBUG_SYNC=1 in the environment: synchronise after every launch so that a device fault is reported by the
// launch that caused it (debugging aid; never set on a timed path).
int debug_sync(const char* what) {
    static const bool on = std::getenv("PULSCAN_DEBUG_SYNC") != nullptr;
    if (!on) return PULSCAN_OK;
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return fail(PULSCAN_ECUDA, "%s: %s", what, cudaGetErrorString(e));
    return PULSCAN_OK;
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline int pow2_ceil(int x) { int p = 1; while (p < x) p <<= 1; return p; }

} // namespace

// Per-cover false-flag probability of the pruned sweep in noise, log10.  Measured on a B200 with the sweep's own second look
// in place (sweep + refine, ms): cfg 3 -3: 1.156, -3.25: 1.128, -3.5: 1.111, -3.75: 1.112, -4: 2.20 (levels finer than 4 bins);
// cfg 4: 0.510 / 0.520 / 0.526 / 0.544 / 1.34; cfg 5: 1.876 / 1.816 / 1.771 / 1.735 / 1.780.
constexpr double kDefaultLog10PFlag = -3.25;

struct pulscan_plan {
    // user parameters
    int64_t n = 0;
    int32_t batch = 0, zmax = 0, C = 0, B = 0;
    double sigma_thr = 0, n_trials = 1.0;
    int64_t pitch = 0;
    int32_t mode = 0;
    int32_t per_width = 0;                   // emit one candidate per (block, searched width) instead of the best width per block
    unsigned out_capacity = 0xFFFFFFFFu;     // records the output array can hold (per-width emission only; otherwise never exceeded)
    int64_t user_capacity = 0;
    int32_t norm_mode = 0;                   // 0 exact median/MAD; 1 the paper's median-of-medians approximation (Alg. 1)
    int32_t signif_mode = 0;                 // 0 exact χ² tail (Eq. 9); 1 the paper's polynomial ln p (Alg. 3)
    int32_t numharm = 1;                     // harmonic-summed spectra searched by pulscan_search_harmonics (L201-220)
    int32_t shape_mult = 1;                  // H(H+1)/2 of the spectrum this plan searches: a width-w sum is Gamma(w·shape_mult)
    int32_t numharm_tag = 1;                 // the H written into pulscan_hcandidate records by this plan
    bool is_child = false;                   // a plan for one Y_H, owned by the plan the user created; it never normalises
    std::vector<pulscan_plan*> harm;         // children for H = 2..numharm
    size_t off_child = 0, child_ws_bytes = 0;
    std::vector<size_t> child_off;           // offset of each child's region inside [off_child, off_child + child_ws_bytes)
    int32_t r_block = 0;                     // report the candidate block's first bin instead of the exact bin (L222-226)
    int32_t z_step = 1, log_sampling = 0;   // which widths are searched (all are summed): Alg. 4
    int32_t tile_user = 0;
    double log10_p_flag = kDefaultLog10PFlag;
    bool host_staging = false;
    // kernel variants (pulscan_plan_set_variant): comparison and tuning switches, none of which changes a result
    int32_t v_second_look = 1;   // the sweep's second look at a flagged cell (half-group thresholds)
    int32_t v_scan_quads = 0;    // 0 = automatic, 5 = the multi-pass scan of 5 quads per thread
    int32_t v_keepidx = -1;      // single-histogram kernel keeps its bucket indices in registers: -1 = automatic, 0, 1
    int32_t v_l2_ahead = -1;     // its L2 look-ahead in CTAs: -1 = automatic (4 x SMs), 0 = off
    int32_t v_single_hist = 1;   // 0: every normalisation block goes through the general kernel
    int32_t v_keep_power = 0;    // 1: the float32 power of every bin stays in the workspace even where the group sums would do
    // derived (host)
    bool dirty = true;         // derived tables need (re)building
    int64_t nblk = 0;          // candidate blocks per spectrum
    int32_t nb = 0;            // normalisation blocks per spectrum
    int64_t pitchP = 0;
    int64_t pitchG = 0;        // row pitch of the group-sum array G (floats): ceil(n/4) rounded up to 4
    bool keep_P = false;       // the per-bin power array stays in the workspace (see derive); otherwise G + statistics only
    double lnp_thr = 0, ln_trials = 0;
    std::vector<double> T;     // T_w
    std::vector<float> Tp;     // conservative float thresholds for the float32 sweep
    std::vector<float> tau;    // per-level cover thresholds
    SweepParams sp{};
    int tiles_per_row = 0;
    bool sweep_fine = false;   // some level has g < 4: the sweep keeps the full-resolution prefix sum
    std::string pruned_error;  // non-empty: the pruned sweep could not be sized for this plan (mode 1 still works)
    int refine_grid = 0;
    int sweep_grid = 0;        // persistent CTAs of the pruned sweep: SM count × resident CTAs per SM
    size_t smem_sweep = 0, smem_refine = 0, smem_exh = 0, smem_exact = 0;
    unsigned cell_cap_user = 0;
    unsigned cell_cap = 0;     // capacity of the flagged-cell list between the sweep and its refine kernel
    int exh_len = 0;
    int exact_lg_split = 0;    // kernel (c): 2^lg lanes share the start bins of a width
    int exact_parts = 1;       // kernel (c): CTAs that share the widths of one marked block
    int exact_seg = 0;         // kernel (c): start bins per segment of a candidate block (= C unless the block is too long for shared memory)
    unsigned exact_slots = 0;  // marked blocks that can be split (size of the partial-result scratch)
    size_t off_partial = 0, off_done = 0;
    // normalisation launch shapes
    int ept_main = 0, nt_main = 0, ept_tail = 0, nt_tail = 0, main_blocks_per_row = 0;
    bool has_tail = false;
    int norm_nt = 256;         // threads per CTA of the single-histogram kernel
    unsigned norm_l2_ahead = 0; // single-histogram kernel: bulk-prefetch into L2 the block of the CTA this many launches ahead
    bool norm_staged = false;  // single-histogram kernel variant: block staged in shared memory by TMA, or read from global
    bool norm_keepidx = true;  // single-histogram kernel keeps the bucket indices in registers for its gather (else: re-reads the block)
    bool use_fast = false;     // full blocks of exactly ept_main·256 bins go through norm_power_v2_kernel + redo list
    // workspace (device, caller-owned)
    void* ws = nullptr;
    size_t ws_bytes = 0;
    size_t off_P = 0, off_G = 0, off_stats = 0, off_bitmap = 0, off_flagged = 0, off_counters = 0, off_redo = 0, off_cells = 0, off_stage_in = 0, off_stage_cand = 0,
           off_stage_count = 0, bitmap_bytes = 0, need_bytes = 0;
    // device tables: T_w (double), T'_w and τ (float); they live in the caller's workspace (off_tables) and are uploaded by
    // pulscan_plan_set_workspace, so that the plan owns no device memory at all
    size_t off_tables = 0;
    double* d_T = nullptr;
    float* d_Tp = nullptr;
    float* d_tau = nullptr;
    bool finalized = false;    // workspace attached, tables uploaded, launch shapes fixed for the current device
    int device = -1;           // the device the plan was finalized on
    int sm_count = 148;
    // optional per-kernel timing: 5 events per slot (start, memsets done, (a) done, (b) done, (c) done)
    int prof_slots = 0, prof_next = 0;
    std::vector<cudaEvent_t> prof_events;
};

extern "C" pulscan_plan* pulscan_plan_create(int64_t, int32_t, int32_t, int32_t, float);
extern "C" int pulscan_plan_destroy(pulscan_plan*);

namespace {

// ---------------------------------------------------------------- host-side plan derivation
float round_down_float(double x) {
    float f = (float)x;
    if ((double)f > x) f = std::nextafterf(f, -INFINITY);
    return f;
}

// Conservative float32 threshold for a sum of `terms` non-negative float32 addends that must not miss a true
// (double-precision) sum ≥ T: any summation order loses at most (terms−1)·2⁻²⁴ relative; 2e-6 covers the
// float32 rounding of the addends themselves.
float conservative_threshold(double T, int terms) {
    return round_down_float(T * (1.0 - 2.0 * (double)terms * 5.9604644775390625e-8 - 2e-6));
}

void attach_children(pulscan_plan& p) {
    for (size_t k = 0; k < p.harm.size(); ++k) {
        p.harm[k]->ws = static_cast<char*>(p.ws) + p.off_child + p.child_off[k];
        p.harm[k]->ws_bytes = align_up(p.harm[k]->need_bytes, 256);
    }
}

// First cover length of a level's first step: the largest m ≤ m_lo with m ≡ 0 or 1 (mod 4), see sweep_step.
int sweep_m_start(int m_lo) { return (m_lo & 3) >= 1 ? (m_lo & ~3) + 1 : m_lo; }

int derive(pulscan_plan& p) {
    if (!p.dirty) return PULSCAN_OK;
    p.nblk = (p.n + p.C - 1) / p.C;
    p.nb = (int32_t)std::max<int64_t>(1, p.n / p.B);
    p.pitchP = (int64_t)align_up((size_t)p.n, 4);
    p.pitchG = (int64_t)align_up((size_t)((p.n + 3) / 4), 4);
    p.lnp_thr = ln_sf(p.sigma_thr);
    p.ln_trials = std::log(p.n_trials);
    const double lnp_target = p.lnp_thr - p.ln_trials; // ln p_adj ≤ lnp_thr ⇔ ln p ≤ lnp_thr − ln N  (R15, R17)
    p.T.resize(p.zmax);
    p.Tp.resize(p.zmax);
    // A width that is not searched gets an infinite threshold: no cover, window or block maximum of it can pass, so every
    // later stage skips it without knowing about the sampling.
    auto searched = [&](int w) {
        const int z = w - 1;
        return p.log_sampling ? (z == 0 || (z & (z - 1)) == 0) : (z % p.z_step == 0);
    };
    p.pruned_error.clear();
    for (int w = 1; w <= p.zmax; ++w) {
        p.T[w - 1] = !searched(w) ? INFINITY
                     : p.signif_mode ? power_threshold_poly(w * p.shape_mult, lnp_target) : power_threshold(w * p.shape_mult, lnp_target);
        p.Tp[w - 1] = searched(w) ? conservative_threshold(p.T[w - 1], w) : INFINITY;
    }

    // ---- sweep tile
    // the group-sum input needs a quarter of the landing space: 8192-bin tiles halve the barriers per bin and balance the
    // warp-tasks better (measured at cfg 3: sweep 1.55 -> 1.43 ms; cfg 5: 2.42 -> 2.22 ms)
    const bool likely_from_g = !p.is_child && p.mode == 0 && p.numharm == 1 && p.norm_mode == 0 && (p.B & 3) == 0;
    int tile = p.tile_user ? p.tile_user : ((p.zmax <= 512 && !likely_from_g) ? 4096 : 8192);
    // ---- group size per width: the largest g = 2^lg whose worst cover (w + 2g − 2 bins) of pure noise passes the
    //      width's threshold with probability ≤ p_flag; made non-decreasing in w by a suffix minimum.
    //      Levels with g < 4 (narrow widths of harmonic-summed spectra, very low σ thresholds) make the sweep use its
    //      full-resolution scan (boxcar_sweep_kernel<true>).  If the width range needs more than kMaxLevels levels,
    //      p_flag is relaxed tenfold at a time: it affects speed only.
    const int lg_cap = 6;
    std::vector<int> lgw(p.zmax + 2, 0);
    std::vector<SweepLevel> lvls;
    int lgmax = 0;
    for (double l10 = p.log10_p_flag;; l10 += 1.0) {
        const double ln_pflag = l10 * 2.302585092994046;
        for (int w = 1; w <= p.zmax; ++w) {
            int best = 0;                 // g = 1: the cover is the window itself
            for (int lg = 1; lg <= lg_cap; ++lg) {
                const int g = 1 << lg, Lc = w + 2 * g - 2;
                if ((tile >> lg) % kSweepR != 0) break;
                if (l10 >= 0.0 || !std::isfinite(p.T[w - 1]) ||
                    ln_q(Lc * p.shape_mult, (double)conservative_threshold(p.T[w - 1], Lc)) <= ln_pflag) best = lg; else break;
            }
            lgw[w] = (w > 1 && !std::isfinite(p.T[w - 1])) ? lgw[w - 1] : best;   // a width that is not searched follows its neighbour
        }
        for (int w = p.zmax - 1; w >= 1; --w) lgw[w] = std::min(lgw[w], lgw[w + 1]);
        lvls.clear();
        lgmax = 0;
        bool fits = true;
        int ntasks_all = 0;
        for (int w = 1; w <= p.zmax && fits;) {
            const int lg = lgw[w], g = 1 << lg;
            auto m_range = [&](int w2, int& m_lo, int& m_hi) {
                if (g == 1) { m_lo = w; m_hi = w2; }
                else { m_lo = (w + g - 1) / g; m_hi = (w2 >= 2) ? (w2 - 2) / g + 2 : 1; }
            };
            int w2 = w, m_lo = 0, m_hi = 0;
            while (w2 + 1 <= p.zmax && lgw[w2 + 1] == lg) {   // extend the run while the m range fits 32 steps of 4
                m_range(w2 + 1, m_lo, m_hi);                  // (sweep_task's hit mask has 32 bits)
                if ((m_hi - sweep_m_start(m_lo) + 4) / 4 > 32) break;
                ++w2;
            }
            m_range(w2, m_lo, m_hi);
            if ((int)lvls.size() >= kMaxLevels) { fits = false; break; }
            SweepLevel lv{};
            lv.lg = lg; lv.wlo = w; lv.whi = w2; lv.m_lo = m_lo; lv.m_hi = m_hi;
            lv.m_start = sweep_m_start(m_lo);
            lv.nsteps = (m_hi - lv.m_start + 4) / 4;
            lv.nk = tile >> lg;
            lv.nwt = (lv.nk + 32 * kSweepR - 1) / (32 * kSweepR);
            if (lv.nsteps > 32) return fail(PULSCAN_EINVAL, "internal: sweep level with %d steps (limit 32)", lv.nsteps);
            ntasks_all += lv.nwt;
            lvls.push_back(lv);
            lgmax = std::max(lgmax, lg);
            w = w2 + 1;
        }
        if (fits && ntasks_all > kMaxWarpTasks) fits = false;   // too many fine levels for one tile: coarser groups
        if (fits) {   // shared memory of the two tile buffers + one decimated array per distinct group size
            const int len = tile + (int)align_up((size_t)(p.zmax + 2 * (1 << lgmax)), 64);
            size_t fl = kSweepBufs * ((size_t)len + kScanTail + 4);
            std::vector<int> seen;
            for (const SweepLevel& lv : lvls)
                if (std::find(seen.begin(), seen.end(), lv.lg) == seen.end()) {
                    seen.push_back(lv.lg);
                    fl += (size_t)(len >> lv.lg) + 1 + kPadG + 3;
                }
            if (fl * 4 + sizeof(SweepCtl) + 2048 <= 227 * 1024) break;
        }
        if (l10 >= 0.0) {   // cannot happen inside the documented parameter ranges; the exhaustive mode does not need the levels
            char msg[256];
            snprintf(msg, sizeof msg, "zmax = %d with tile = %d does not fit the pruned sweep (shared memory or %d warp-tasks per tile)",
                     p.zmax, tile, kMaxWarpTasks);
            p.pruned_error = msg;
            lvls.clear(); lgmax = 0;
            break;
        }
    }
    SweepParams& sp = p.sp;
    std::memset(&sp, 0, sizeof sp);
    p.tau.clear();
    std::stable_sort(lvls.begin(), lvls.end(), [](const SweepLevel& a, const SweepLevel& b) { return a.nsteps > b.nsteps; });
    sp.nlevels = (int)lvls.size();
    sp.tile = tile;
    const int halo = (int)align_up((size_t)(p.zmax + 2 * (1 << lgmax)), 64);
    sp.len = tile + halo;
    if (sp.len > kMaxSweepLen)   // the rounding bound of the scan (scan_roundings, boxcar_sweep.cuh) is asserted for this length
        return fail(PULSCAN_EINVAL, "internal: sweep landing buffer of %d bins exceeds %d", sp.len, kMaxSweepLen);
    int off = 0, task = 0;
    for (int l = 0; l < sp.nlevels; ++l) {
        SweepLevel& lv = lvls[l];
        int a = 0;
        while (a < sp.narr && sp.arr_lg[a] != lv.lg) ++a;
        if (a == sp.narr) {
            sp.arr_lg[a] = lv.lg; sp.arr_off[a] = off;
            off += (int)align_up((size_t)((sp.len >> lv.lg) + 1 + kPadG), 4);
            ++sp.narr;
        }
        lv.pg_off = sp.arr_off[a];
        lv.tau_off = (int)p.tau.size();
        const int g = 1 << lv.lg;
        for (int m = lv.m_start; m < lv.m_start + 4 * lv.nsteps; ++m) {
            if (m < lv.m_lo || m > lv.m_hi) { p.tau.push_back(INFINITY); continue; }
            const int wmin = (g == 1) ? m : (m == 1 ? 1 : (m - 2) * g + 2);
            // the lowest threshold among the level's searched widths whose windows have a cover of exactly m groups
            // (widths wmin … m·g; the exact T_w grows with w, Alg. 3's need not); +inf if there is none
            const int wtop = std::min(lv.whi, m * g);
            double tmin = INFINITY;
            for (int wq = std::min(std::max(lv.wlo, wmin), lv.whi); wq <= wtop; ++wq) tmin = std::min(tmin, p.T[wq - 1]);
            p.tau.push_back(std::isfinite(tmin) ? conservative_threshold(tmin, m * g) : INFINITY);
        }
        // with sparse width sampling whole 4-wide steps can be dead (τ = +inf): trim them off both ends
        {
            auto dead = [&](int st) {
                for (int q = 0; q < 4; ++q)
                    if (std::isfinite(p.tau[lv.tau_off + 4 * st + q])) return false;
                return true;
            };
            int first = 0, last = lv.nsteps - 1;
            while (first <= last && dead(first)) ++first;
            while (last >= first && dead(last)) --last;
            lv.m_start += 4 * first; lv.tau_off += 4 * first; lv.nsteps = last - first + 1;
            if (lv.nsteps == 0) lv.nwt = 0;
        }
        lv.wt_off = task;
        task += lv.nwt;
        sp.lv[l] = lv;
    }
    sp.ntasks = task;
    for (int lg = 0; lg < 8; ++lg) sp.off_lg[lg] = -1;
    for (int a = 0; a < sp.narr; ++a) sp.off_lg[sp.arr_lg[a]] = sp.arr_off[a];
    // τ_h tables: thresholds of covers of mh half-groups (g/2 bins), per level with g ≥ 8: the refine kernel's second look
    for (int l = 0; l < sp.nlevels; ++l) {
        SweepLevel& lv = sp.lv[l];
        lv.tauh_off = 0; lv.mh_start = 0; lv.nmh = 0;
        if (lv.lg < 3 || lv.nsteps == 0 || !p.v_second_look) continue;
        const int gh = 1 << (lv.lg - 1);
        lv.mh_start = std::max(0, 2 * lv.m_start - 2);
        const int mh_end = 2 * (lv.m_start + 4 * lv.nsteps - 1);
        lv.nmh = mh_end - lv.mh_start + 1;
        lv.tauh_off = (int)p.tau.size();
        for (int mh = lv.mh_start; mh <= mh_end; ++mh) {
            const int wmin = (mh <= 1) ? 1 : (mh - 2) * gh + 2, wtop = std::min(lv.whi, mh * gh);
            double tmin = INFINITY;
            for (int wq = std::max(lv.wlo, wmin); wq <= wtop; ++wq) tmin = std::min(tmin, p.T[wq - 1]);
            p.tau.push_back(std::isfinite(tmin) && mh >= 1 ? conservative_threshold(tmin, mh * gh) : INFINITY);
        }
    }
    p.sweep_fine = false;
    for (int a = 0; a < sp.narr; ++a) p.sweep_fine = p.sweep_fine || sp.arr_lg[a] < 2;
    // Does the float32 power of every bin have to exist in HBM?  Not on the default path: kernel (a) then leaves only the sums
    // of aligned groups of four bins (G, a quarter of the bytes) and six numbers per normalisation block, and the rare-path
    // kernels rebuild the spans they need from the input spectrum (power_source.cuh).  It stays for: a child plan (its
    // "power" is the harmonic-summed spectrum Y_H), the exhaustive cross-check mode, levels finer than four bins
    // (full-resolution sweep), the harmonic search (Y_H is summed from P), the Alg. 1 normalisation kernel, and
    // normalisation blocks that are not a multiple of four bins.  PULSCAN_VARIANT_KEEP_POWER forces it (comparison runs).
    p.keep_P = p.is_child || p.mode == 1 || p.sweep_fine || p.numharm > 1 || p.norm_mode == 1 || (p.B & 3) != 0 || p.v_keep_power;
    sp.z_floats = p.keep_P ? (int)align_up((size_t)(sp.len + kScanTail), 4) : (int)align_up((size_t)(sp.len / 4 + kScanTail / 4), 4);
    // quads per thread per scan pass: a whole tile + halo in one pass where it fits 9 or 11 quads per thread (the
    // full-resolution scan keeps three more values per quad in registers and stays at 5)
    sp.scan_nq = (p.sweep_fine || sp.len <= 20 * kSweepThreads) ? 5 : (sp.len <= 36 * kSweepThreads ? 9 : (sp.len <= 44 * kSweepThreads && !p.keep_P ? 11 : 5));
    if (p.v_scan_quads == 5) sp.scan_nq = 5;
    sp.npass = (sp.len + 4 * sp.scan_nq * kSweepThreads - 1) / (4 * sp.scan_nq * kSweepThreads);
    if (task > kMaxWarpTasks) return fail(PULSCAN_EINVAL, "sweep tile of %d bins needs %d warp-tasks (limit %d)", tile, task, kMaxWarpTasks);
    sp.ntau = (int)p.tau.size();
    sp.smem_floats = kSweepBufs * sp.z_floats + off;
    p.tiles_per_row = (int)((p.n + tile - 1) / tile);
    const size_t flag_bytes = align_up((size_t)(tile / p.C + 3), 16);
    sp.zmax = p.zmax;
    sp.tp_monotone = 1;
    for (int w = 1; w <= p.zmax; ++w)
        if (!std::isfinite(p.Tp[w - 1]) || (w > 1 && p.Tp[w - 1] < p.Tp[w - 2])) sp.tp_monotone = 0;
    // strong-signal shortcut of the sweep: only where noise practically never flags that many lanes of one warp-task (at the
    // harmonic children's 10^-2.5 it marked noise blocks: numharm 4 at cfg 3 10.97 -> 12.06 ms)
    sp.dense_lanes = p.log10_p_flag <= -3.0 ? kSweepDenseLanes : 33;
    sp.ref_span = 0;
    for (int l = 0; l < sp.nlevels; ++l)
        sp.ref_span = std::max(sp.ref_span, (sp.lv[l].m_start + 4 * sp.lv[l].nsteps + 6) << sp.lv[l].lg);
    p.smem_sweep = (size_t)sp.smem_floats * 4 + align_up((size_t)sp.ntau, 4) * 4 + sizeof(SweepCtl);
    p.smem_refine = (size_t)(kRefineThreads / 32) * (sp.ref_span + 1) * sizeof(double);
    if (p.smem_refine > 227 * 1024) return fail(PULSCAN_EINVAL, "refine span of %d bins does not fit shared memory", sp.ref_span);
    if (p.smem_sweep > 227 * 1024) return fail(PULSCAN_EINVAL, "sweep tile needs %zu bytes of shared memory", p.smem_sweep);
    p.exh_len = tile + (int)align_up((size_t)p.zmax, 64);
    p.smem_exh = (size_t)p.exh_len * 4 + align_up((size_t)p.zmax, 4) * 4 + 16 + flag_bytes;
    {   // kernel (c) holds the prefix sum of a candidate block + halo in shared memory as doubles; a block too long for that
        // (the paper's R-Block width 32768, L224) is walked in segments, with the per-width running maxima carried in
        // (zmax + 1)·12 further bytes
        constexpr long long kDyn = 227 * 1024;
        if (p.C + p.zmax <= 24576) p.exact_seg = p.C;
        else {
            const long long room = (kDyn - (long long)sizeof(ExactSmemHdr) - (long long)(p.zmax + 1) * 12 - 16) / 8 - p.zmax - 2;
            p.exact_seg = (int)(room / 64 * 64);
            if (p.exact_seg < 1024) return fail(PULSCAN_EINVAL, "internal: no room for a segment of block_width = %d at zmax = %d", p.C, p.zmax);
        }
        const int cs = std::min(p.C, p.exact_seg);
        p.smem_exact = sizeof(ExactSmemHdr) + (size_t)((cs + p.zmax + 2) & ~1) * 8 + (p.exact_seg < p.C ? (size_t)(p.zmax + 1) * 12 : 0);
    }
    {   // kernel (c): a thread owns four consecutive widths; the start bins of a block are split over 2^lg adjacent lanes.  One
        // block costs zmax·C window sums on ONE SM (issue-bound: double-precision compare and select) plus ≈ 45 µs of
        // barrier-separated set-up per CTA (prefix sum rebuilt from the spectrum, ln p of the passing widths): only when the
        // window sums are several times that (measured at cfg 4, 1.44 M sums per block: 1 CTA 0.245 ms, 8 CTAs 0.387 ms) are
        // the widths of a block dealt to several CTAs; lg is then chosen to give that many rounds of kExactThreads threads.
        const long long nquads = p.zmax / 4 + 1;
        const long long want_parts = std::min<long long>(8, std::max<long long>(1, (long long)p.zmax * p.C / 3000000));
        long long best = -1;
        for (int lg = 0; lg <= 5; ++lg) {
            const long long rounds = (nquads * (1 << lg) + kExactThreads - 1) / kExactThreads;
            // a round costs its 4 x 4 tiles plus eight barriers and the ln p evaluations (worth ~48 tiles)
            long long cost = ((rounds + want_parts - 1) / want_parts) * ((((p.C + (1 << lg) - 1) >> lg) + 3) / 4 + 48) + lg;
            if (rounds < want_parts) cost += 1000000;          // cannot be split that far
            if (best < 0 || cost < best) { best = cost; p.exact_lg_split = lg; }
        }
        const int rounds = (int)((nquads * (1 << p.exact_lg_split) + kExactThreads - 1) / kExactThreads);
        p.exact_parts = (int)std::min<long long>(rounds, want_parts);
        p.exact_slots = p.exact_parts > 1 ? (unsigned)std::min<long long>((long long)p.batch * p.nblk, 16384) : 0u;
    }

    // ---- normalisation launch shapes (a child plan searches a spectrum that its parent has normalised and summed)
    if (p.is_child) { p.main_blocks_per_row = 0; p.has_tail = false; p.use_fast = false; }
    else {
    const int64_t len_last = p.n - (int64_t)(p.nb - 1) * p.B;
    if (p.B <= 8192) { p.nt_main = 256; p.ept_main = pow2_ceil((p.B + 255) / 256); }
    else { p.nt_main = 1024; p.ept_main = pow2_ceil((p.B + 1023) / 1024); }
    p.has_tail = len_last > (int64_t)p.ept_main * p.nt_main || p.nb == 1;
    if (p.has_tail) {
        p.nt_tail = len_last <= 256 * 32 ? 256 : 1024;
        p.ept_tail = pow2_ceil((int)((len_last + p.nt_tail - 1) / p.nt_tail));
        if (p.ept_tail > 32) return fail(PULSCAN_EINVAL, "last normalisation block too long (%lld bins)", (long long)len_last);
        p.main_blocks_per_row = p.nb - 1;
    } else {
        p.main_blocks_per_row = p.nb;
    }

    p.norm_staged = false;   // the TMA-staged variant lost its measurement (round 1) and is no longer dispatched
    // Bucket indices kept in registers between the histogram pass and the gather, or recomputed from a re-read of the block
    // (40 instead of 64 registers: more blocks per SM, one more read pass).  Measured (kernel (a), ms; kept / recomputed):
    // cfg 3 (B 4096, 128 threads, 8 -> 10 CTAs) 3.05 / 3.58; cfg 5 (B 2048) 7.53 / 8.05; cfg 4 (B 8192, 256 threads,
    // 4 -> 6 CTAs) 0.864 / 0.830 — recomputed for blocks of 8192 bins only.  PULSCAN_VARIANT_NORM_KEEP_INDICES overrides.
    p.norm_keepidx = p.v_keepidx >= 0 ? p.v_keepidx != 0 : p.B < 8192;
    // Fewer warps per CTA: the warp-serial phases keep two warps busy and idle the rest.  Measured: cfg 3 (B = 4096)
    // 256 threads 3.71 ms, 128 threads 3.41 ms; cfg 5 (B = 2048) 128 threads 9.06 ms, 64 threads 10.5 ms.
    p.norm_nt = (p.B >= 512 && p.B <= 4096) ? 128 : 256;
    p.use_fast = p.nt_main == 256 && p.B == p.ept_main * 256 && p.ept_main >= 2 && p.main_blocks_per_row > 0 && p.v_single_hist;
    }

    // ---- workspace layout
    size_t o = 0;
    p.off_P = o; o += p.keep_P ? align_up((size_t)p.batch * p.pitchP * 4, 256) : 0;
    p.off_G = o; o += p.keep_P ? 0 : align_up((size_t)p.batch * p.pitchG * 4, 256);
    p.off_stats = o; o += p.keep_P ? 0 : align_up((size_t)p.batch * p.nb * 8 * sizeof(float), 256);
    p.bitmap_bytes = align_up((size_t)((p.batch * p.nblk + 31) / 32) * 4, 256);
    p.off_bitmap = o; o += p.bitmap_bytes;
    p.off_flagged = o; o += align_up((size_t)p.batch * p.nblk * 4, 256);
    p.off_counters = o; o += 256;
    p.off_redo = o; o += align_up((size_t)p.batch * p.nb * 4, 256);
    // noise flags ≈ 0.6 cells per 4096 bins at the default p_flag; room for 16 per 4096 bins (then tiles fall back to
    // marking all their blocks)
    p.cell_cap = (unsigned)std::min<unsigned long long>(1ull << 28, std::max<unsigned long long>(65536, (unsigned long long)p.batch * p.n / 256));
    if (p.cell_cap_user) p.cell_cap = p.cell_cap_user;
    p.off_cells = o; o += align_up((size_t)p.cell_cap * sizeof(SweepCell), 256);
    p.off_partial = o; o += align_up((size_t)p.exact_slots * p.exact_parts * sizeof(ExactPartial), 256);
    p.off_done = o; o += align_up((size_t)p.exact_slots * sizeof(unsigned), 256);
    p.off_tables = o;
    o += align_up(p.T.size() * sizeof(double), 256) + align_up(p.Tp.size() * sizeof(float), 256) +
         align_up(std::max<size_t>(1, p.tau.size()) * sizeof(float), 256);
    if (p.host_staging) {
        p.off_stage_in = o; o += align_up((size_t)p.batch * p.pitch * 8, 256);
        // per-width emission writes up to the caller's capacity, which may exceed one record per block
        const size_t recs = std::max<size_t>((size_t)p.batch * p.nblk, (size_t)p.user_capacity);
        p.off_stage_cand = o; o += align_up(recs * sizeof(pulscan_candidate), 256);
        p.off_stage_count = o; o += 256;
    }
    // ---- harmonic-summed spectra: one child plan per H = 2..numharm, each with its own region of the workspace (a child's
    //      "power" buffer is Y_H)
    for (pulscan_plan* c : p.harm) pulscan_plan_destroy(c);
    p.harm.clear();
    p.off_child = o; p.child_ws_bytes = 0; p.child_off.clear();
    for (int H = 2; H <= p.numharm && !p.is_child; ++H) {
        const int64_t nH = p.n / H;
        if ((int64_t)p.zmax >= nH) return fail(PULSCAN_EINVAL, "zmax = %d must be < floor(n_bins / %d) = %lld", p.zmax, H, (long long)nH);
        pulscan_plan* c = pulscan_plan_create(nH, p.batch, p.zmax, p.C, (float)p.sigma_thr);
        if (!c) return PULSCAN_EINVAL;
        c->is_child = true; c->shape_mult = H * (H + 1) / 2; c->numharm_tag = H; c->sigma_thr = p.sigma_thr; c->n_trials = p.n_trials;
        c->signif_mode = p.signif_mode; c->mode = p.mode;   // the mode is checked against the child's sweep levels at finalisation
        c->z_step = p.z_step; c->log_sampling = p.log_sampling; c->tile_user = p.tile_user;
        // a harmonic-summed spectrum has H(H+1)/2 of noise in every bin of a cover's slack: coarser groups at a higher flag rate
        // pay there (numharm 4, log-spaced widths, cfg 3: 8.92 ms at -3.25, 8.25 at -2.5, 8.35 at -2)
        c->log10_p_flag = (p.log10_p_flag == kDefaultLog10PFlag) ? -2.5 : p.log10_p_flag;
        c->cell_cap_user = p.cell_cap_user; c->B = p.B;
        c->v_second_look = p.v_second_look; c->v_scan_quads = p.v_scan_quads;
        p.harm.push_back(c);
        const int rc = derive(*c);
        if (rc) return rc;
        p.child_off.push_back(p.child_ws_bytes);                   // every Y_H keeps its own buffer: one decimation pass writes all
        p.child_ws_bytes += align_up(c->need_bytes, 256);
    }
    o += p.child_ws_bytes;
    p.need_bytes = o;
    p.dirty = false;
    if (p.ws && p.ws_bytes >= p.need_bytes) attach_children(p);
    return PULSCAN_OK;
}

// Everything pulscan_search needs from the CUDA runtime besides launches, done once when the workspace is attached: device
// check, upload of the three small tables into the workspace, dynamic shared-memory limits of the kernels (an attribute of the
// function ON THE CURRENT DEVICE, so it is set at every finalisation rather than once per process), launch shapes from the
// occupancy API.  Synchronous; never called from pulscan_search.
int set_kernel_attributes(const pulscan_plan& p);

using SweepFn = void (*)(const SweepParams, const float*, long long, long long, int, long long, int, long long, const float*,
                         SweepCell*, unsigned, unsigned*, unsigned*, unsigned*);
SweepFn sweep_function(const pulscan_plan& p) {
    const int nq = p.sp.scan_nq;
    if (!p.keep_P) return nq == 9 ? boxcar_sweep_kernel<false, true, 9> : nq == 11 ? boxcar_sweep_kernel<false, true, 11> : boxcar_sweep_kernel<false, true, 5>;
    if (p.sweep_fine) return boxcar_sweep_kernel<true, false, 5>;
    return nq == 9 ? boxcar_sweep_kernel<false, false, 9> : boxcar_sweep_kernel<false, false, 5>;
}

int finalize_device(pulscan_plan& p) {
    p.finalized = false;
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10)
        return fail(PULSCAN_EARCH, "device %s is compute capability %d.%d; libpulscan is built for sm_100a only", prop.name,
                    prop.major, prop.minor);
    // all validation happens here ("Life of a plan"): a plan whose pruned sweep could not be sized must not get as far as a
    // search (which would fail at enqueue time, possibly inside a stream capture)
    if (p.mode == 0 && !p.pruned_error.empty())
        return fail(PULSCAN_EINVAL, "%s; use mode 1 (exhaustive)", p.pruned_error.c_str());
    p.device = dev;
    p.sm_count = prop.multiProcessorCount;
    char* ws = static_cast<char*>(p.ws);
    p.d_T = reinterpret_cast<double*>(ws + p.off_tables);
    p.d_Tp = reinterpret_cast<float*>(ws + p.off_tables + align_up(p.T.size() * sizeof(double), 256));
    p.d_tau = reinterpret_cast<float*>(reinterpret_cast<char*>(p.d_Tp) + align_up(p.Tp.size() * sizeof(float), 256));
    CUDA_TRY(cudaMemcpy(p.d_T, p.T.data(), p.T.size() * sizeof(double), cudaMemcpyHostToDevice));
    CUDA_TRY(cudaMemcpy(p.d_Tp, p.Tp.data(), p.Tp.size() * sizeof(float), cudaMemcpyHostToDevice));
    if (!p.tau.empty()) CUDA_TRY(cudaMemcpy(p.d_tau, p.tau.data(), p.tau.size() * sizeof(float), cudaMemcpyHostToDevice));
    constexpr int kMaxDynSmem = 227 * 1024;
    if (p.smem_sweep > (size_t)kMaxDynSmem || p.smem_exh > (size_t)kMaxDynSmem || p.smem_exact > (size_t)kMaxDynSmem)
        return fail(PULSCAN_EINVAL, "plan needs more shared memory than an SM has (sweep %zu, exhaustive %zu, exact %zu bytes)",
                    p.smem_sweep, p.smem_exh, p.smem_exact);
    int rc = set_kernel_attributes(p);
    if (rc) return rc;
    const SweepFn sweep_fn = sweep_function(p);
    int occ = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, sweep_fn, kSweepThreads, p.smem_sweep));
    if (occ < 1) return fail(PULSCAN_ECUDA, "boxcar_sweep_kernel does not fit an SM with %zu bytes of shared memory", p.smem_sweep);
    p.sweep_grid = (int)std::min<long long>((long long)p.tiles_per_row * p.batch, (long long)p.sm_count * occ);
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, sweep_refine_kernel, kRefineThreads, p.smem_refine));
    if (occ < 1) return fail(PULSCAN_ECUDA, "sweep_refine_kernel does not fit an SM with %zu bytes of shared memory", p.smem_refine);
    p.refine_grid = p.sm_count * std::min(occ, 16);
    {   // look-ahead of the single-histogram kernel's L2 prefetch in CTAs (short blocks only, see kV2L2Ahead): half a wave of
        // resident CTAs measured best (592 and 1184: 7.61 ms at cfg 5; 2368: 8.0; off: 8.25); PULSCAN_VARIANT_NORM_L2_AHEAD overrides
        p.norm_l2_ahead = p.v_l2_ahead >= 0 ? (unsigned)p.v_l2_ahead : (unsigned)p.sm_count * 4u;
    }
    p.finalized = true;
    return PULSCAN_OK;
}

void release_profiling(pulscan_plan& p) {
    for (cudaEvent_t e : p.prof_events)
        if (e) cudaEventDestroy(e);
    p.prof_events.clear();
    p.prof_next = 0;
}

// A setter changed something the derived tables or the workspace layout depend on: the plan must be finalised again
// (pulscan_plan_set_workspace) before the next search.  Host only: the plan owns no device memory.
void invalidate(pulscan_plan& p) {
    p.dirty = true;
    p.finalized = false;
    for (pulscan_plan* c : p.harm) c->finalized = false;
}

// Dynamic shared-memory limits above 48 KB are an attribute of (function, device): set for every kernel that may need one,
// each time a plan is finalised on a device (idempotent, host-side, cheap).
int set_kernel_attributes(const pulscan_plan& p) {
    (void)p;
    constexpr int kMaxDynSmem = 227 * 1024;
    CUDA_TRY(cudaFuncSetAttribute(boxcar_sweep_kernel<false, false, 5>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem));
    CUDA_TRY(cudaFuncSetAttribute(boxcar_sweep_kernel<false, false, 9>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem));
    CUDA_TRY(cudaFuncSetAttribute(boxcar_sweep_kernel<true, false, 5>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem));
    CUDA_TRY(cudaFuncSetAttribute(boxcar_sweep_kernel<false, true, 5>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem));
    CUDA_TRY(cudaFuncSetAttribute(boxcar_sweep_kernel<false, true, 9>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem));
    CUDA_TRY(cudaFuncSetAttribute(boxcar_sweep_kernel<false, true, 11>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem));
    CUDA_TRY(cudaFuncSetAttribute(sweep_refine_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem));
    CUDA_TRY(cudaFuncSetAttribute(boxcar_exhaustive_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem));
    CUDA_TRY(cudaFuncSetAttribute(block_exact_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem));
    return PULSCAN_OK;
}

template <int NT>
int launch_norm(int ept, int grid, cudaStream_t st, const float2* spectra, long long pitch_in, long long n, int B, int nb,
                int first_block, int blocks_per_row, const NormOut& out) {
#define PULSCAN_NORM_CASE(E)                                                                                      \
    case E:                                                                                                       \
        norm_power_kernel<E, NT><<<grid, NT, 0, st>>>(spectra, pitch_in, n, B, nb, first_block, blocks_per_row, out); \
        break;
    switch (ept) {
        PULSCAN_NORM_CASE(1)
        PULSCAN_NORM_CASE(2)
        PULSCAN_NORM_CASE(4)
        PULSCAN_NORM_CASE(8)
        PULSCAN_NORM_CASE(16)
        PULSCAN_NORM_CASE(32)
        default: return fail(PULSCAN_EINVAL, "internal: unsupported elements-per-thread %d", ept);
    }
#undef PULSCAN_NORM_CASE
    CUDA_TRY(cudaGetLastError());
    char what[64];
    snprintf(what, sizeof what, "norm_power_kernel<%d,%d> grid %d", ept, NT, grid);
    return debug_sync(what);
}

constexpr int kRedoGrid = 148;

// Fast kernel for the full blocks + redo kernel (general path) for the blocks it declined.
int launch_norm_fast(pulscan_plan& p, int grid, cudaStream_t st, const float2* spec, const NormOut& out, unsigned* redo,
                     unsigned* redo_count) {
    const char* lim_lo = reinterpret_cast<const char*>(spec);
    const char* lim_hi = lim_lo + ((size_t)(p.batch - 1) * p.pitch + p.n) * 8;
#define PULSCAN_V2_LAUNCH(E, NT_, ST)                                                                                 \
    {                                                                                                                 \
        if (!ST && !p.norm_keepidx && (E) >= 16)                                                                       \
            norm_power_v2_kernel<E, NT_, false, false><<<grid, NT_, v2_smem_bytes<E, NT_, false>(), st>>>(            \
                spec, p.pitch, p.main_blocks_per_row, p.nb, out, redo, redo_count, lim_lo, lim_hi, p.norm_l2_ahead);  \
        else                                                                                                          \
            norm_power_v2_kernel<E, NT_, ST><<<grid, NT_, v2_smem_bytes<E, NT_, ST>(), st>>>(                          \
                spec, p.pitch, p.main_blocks_per_row, p.nb, out, redo, redo_count, lim_lo, lim_hi, p.norm_l2_ahead);  \
    }
#define PULSCAN_V2_REDO(E)                                                                                            \
    norm_power_redo_kernel<E, 256><<<kRedoGrid, 256, 0, st>>>(spec, p.pitch, p.B, p.nb, p.main_blocks_per_row, out, redo, \
                                                              redo_count);
    // key = threads per CTA · 64 + values per thread of the single-histogram kernel (B = their product)
    switch (p.norm_nt * 64 + p.B / p.norm_nt) {
        case 256 * 64 + 2: PULSCAN_V2_LAUNCH(2, 256, false) break;
        case 256 * 64 + 4: PULSCAN_V2_LAUNCH(4, 256, false) break;
        case 256 * 64 + 8: PULSCAN_V2_LAUNCH(8, 256, false) break;
        case 256 * 64 + 16: PULSCAN_V2_LAUNCH(16, 256, false) break;
        case 256 * 64 + 32: PULSCAN_V2_LAUNCH(32, 256, false) break;
        case 128 * 64 + 32: PULSCAN_V2_LAUNCH(32, 128, false) break;
        case 128 * 64 + 16: PULSCAN_V2_LAUNCH(16, 128, false) break;
        case 128 * 64 + 8: PULSCAN_V2_LAUNCH(8, 128, false) break;
        case 128 * 64 + 4: PULSCAN_V2_LAUNCH(4, 128, false) break;
        default: return fail(PULSCAN_EINVAL, "internal: no single-histogram kernel for %d threads x %d values", p.norm_nt, p.B / p.norm_nt);
    }
    switch (p.ept_main) {
        case 2: PULSCAN_V2_REDO(2) break;
        case 4: PULSCAN_V2_REDO(4) break;
        case 8: PULSCAN_V2_REDO(8) break;
        case 16: PULSCAN_V2_REDO(16) break;
        case 32: PULSCAN_V2_REDO(32) break;
        default: return fail(PULSCAN_EINVAL, "internal: unsupported elements-per-thread %d", p.ept_main);
    }
#undef PULSCAN_V2_REDO
#undef PULSCAN_V2_LAUNCH
    CUDA_TRY(cudaGetLastError());
    return debug_sync("fast normalisation kernel + norm_power_redo_kernel");
}

// d_scratch: the redo list and its counter (inside the workspace for pulscan_search; a temporary for the stand-alone
// pulscan_normalise_power, which has no workspace).  redo_count must be zero on entry.
int enqueue_norm(pulscan_plan& p, const void* d_spectra, const NormOut& out, cudaStream_t st, unsigned* d_redo,
                 unsigned* d_redo_count) {
    float* d_power = out.P;
    const float2* spec = reinterpret_cast<const float2*>(d_spectra);
    int rc = PULSCAN_OK;
    if (p.norm_mode == 1) {   // Alg. 1: one kernel for every chunk, the last one of a row included
        if (!d_power) return fail(PULSCAN_EINVAL, "internal: the Alg. 1 kernel writes the per-bin power array");
        const long long grid = (long long)p.nb * p.batch;
        if (grid > 2147483647LL) return fail(PULSCAN_EINVAL, "too many normalisation blocks for one launch");
#define PULSCAN_MOM_CASE(E, NT_)                                                                                      \
    case (E) * (NT_):                                                                                                 \
        norm_power_mom_kernel<E, NT_><<<(int)grid, NT_, 0, st>>>(spec, p.pitch, p.n, p.nb, d_power, p.pitchP);       \
        break;
        switch (p.B) {
            PULSCAN_MOM_CASE(4, 64)
            PULSCAN_MOM_CASE(4, 128)
            PULSCAN_MOM_CASE(8, 128)
            PULSCAN_MOM_CASE(16, 128)
            PULSCAN_MOM_CASE(32, 128)
            PULSCAN_MOM_CASE(32, 256)
            PULSCAN_MOM_CASE(64, 256)
            default: return fail(PULSCAN_EINVAL, "median-of-medians normalisation needs norm_block = 256 … 16384, a power of two");
        }
#undef PULSCAN_MOM_CASE
        CUDA_TRY(cudaGetLastError());
        return debug_sync("norm_power_mom_kernel");
    }
    if (p.main_blocks_per_row > 0) {
        const long long grid = (long long)p.main_blocks_per_row * p.batch;
        if (grid > 2147483647LL) return fail(PULSCAN_EINVAL, "too many normalisation blocks for one launch");
        if (p.use_fast && d_redo)
            rc = launch_norm_fast(p, (int)grid, st, spec, out, d_redo, d_redo_count);
        else
            rc = (p.nt_main == 256)
                     ? launch_norm<256>(p.ept_main, (int)grid, st, spec, p.pitch, p.n, p.B, p.nb, 0, p.main_blocks_per_row, out)
                     : launch_norm<1024>(p.ept_main, (int)grid, st, spec, p.pitch, p.n, p.B, p.nb, 0, p.main_blocks_per_row, out);
        if (rc) return rc;
    }
    if (p.has_tail) {
        rc = (p.nt_tail == 256)
                 ? launch_norm<256>(p.ept_tail, p.batch, st, spec, p.pitch, p.n, p.B, p.nb, p.nb - 1, 1, out)
                 : launch_norm<1024>(p.ept_tail, p.batch, st, spec, p.pitch, p.n, p.B, p.nb, p.nb - 1, 1, out);
    }
    return rc;
}

// Kernels (b) and (c) on a power (or harmonic-summed) spectrum that is ready in d_P; the plan's bitmap and counters must
// have been zeroed on the stream.  Exactly one of d_candidates / d_hcandidates is non-null.
// d_in: what the sweep streams — the per-bin array (P or Y_H, pitchP) or, for a plan that does not keep one, the group sums G
// (pitchG).  src: where the rare-path kernels read a bin's power (power_source.cuh).
int enqueue_sweep_exact(pulscan_plan& p, const float* d_in, const PowerSource& src, pulscan_candidate* d_candidates,
                        pulscan_hcandidate* d_hcandidates, uint32_t* d_count, cudaStream_t st, cudaEvent_t* ev) {
    const bool from_g = !p.keep_P;
    const long long pitch_in = from_g ? p.pitchG : p.pitchP;
    int rc = PULSCAN_OK;
    char* ws = static_cast<char*>(p.ws);
    unsigned* d_bitmap = reinterpret_cast<unsigned*>(ws + p.off_bitmap);
    unsigned* d_flagged = reinterpret_cast<unsigned*>(ws + p.off_flagged);
    unsigned* d_counters = reinterpret_cast<unsigned*>(ws + p.off_counters);
    const long long grid_b = (long long)p.tiles_per_row * p.batch;                 // (b)
    if (grid_b > 2147483647LL) return fail(PULSCAN_EINVAL, "too many sweep tiles for one launch");
    if (p.mode == 0) {
        if (!p.pruned_error.empty()) return fail(PULSCAN_EINVAL, "%s; use mode 1 (exhaustive)", p.pruned_error.c_str());
        SweepCell* d_cells = reinterpret_cast<SweepCell*>(ws + p.off_cells);
        sweep_function(p)<<<p.sweep_grid, kSweepThreads, p.smem_sweep, st>>>(p.sp, d_in, pitch_in, p.n, p.tiles_per_row, grid_b, p.C,
                                                                             p.nblk, p.d_tau, d_cells, p.cell_cap, d_bitmap, d_flagged,
                                                                             d_counters);
        CUDA_TRY(cudaGetLastError());
        if ((rc = debug_sync("boxcar_sweep_kernel"))) return rc;
        sweep_refine_kernel<<<p.refine_grid, kRefineThreads, p.smem_refine, st>>>(p.sp, src, from_g ? d_in : nullptr, p.pitchG, p.n, p.tiles_per_row, p.C,
                                                                                  p.nblk, p.d_tau, p.d_Tp, d_cells, p.cell_cap,
                                                                                  d_bitmap, d_flagged, d_counters);
    } else {
        if (from_g) return fail(PULSCAN_EINVAL, "internal: the exhaustive sweep needs the per-bin power array");
        boxcar_exhaustive_kernel<<<(int)grid_b, kSweepThreads, p.smem_exh, st>>>(p.sp.tile, p.exh_len, p.zmax, d_in, p.pitchP,
                                                                                p.n, p.tiles_per_row, p.C, p.nblk, p.d_Tp,
                                                                                d_bitmap, d_flagged, d_counters);
    }
    CUDA_TRY(cudaGetLastError());
    if ((rc = debug_sync(p.mode ? "boxcar_exhaustive_kernel" : "sweep_refine_kernel"))) return rc;
    if (ev) CUDA_TRY(cudaEventRecord(ev[3], st));

    const long long total_blocks = (long long)p.batch * p.nblk;                    // (c)
    const int grid_c = (int)std::min<long long>(total_blocks * p.exact_parts, (long long)p.sm_count * 4);
    if (p.exact_slots) CUDA_TRY(cudaMemsetAsync(ws + p.off_done, 0, (size_t)p.exact_slots * sizeof(unsigned), st));
    block_exact_kernel<<<grid_c, kExactThreads, p.smem_exact, st>>>(src, p.n, p.zmax, p.C, p.nblk, p.d_T, p.ln_trials,
                                                                   p.lnp_thr, p.r_block, p.shape_mult, p.signif_mode, p.numharm_tag, d_hcandidates, p.per_width, p.out_capacity, p.exact_lg_split, p.exact_parts, p.exact_seg,
                                                                   p.exact_slots, reinterpret_cast<ExactPartial*>(ws + p.off_partial),
                                                                   reinterpret_cast<unsigned*>(ws + p.off_done),
                                                                   d_flagged, d_counters, d_candidates, d_count);
    CUDA_TRY(cudaGetLastError());
    return PULSCAN_OK;
}

// What kernel (a) writes for this plan, what the sweep streams, and where the rare-path kernels read powers.
NormOut norm_outputs(const pulscan_plan& p) {
    char* ws = static_cast<char*>(p.ws);
    if (p.keep_P) return NormOut{reinterpret_cast<float*>(ws + p.off_P), p.pitchP, nullptr, 0, nullptr};
    return NormOut{nullptr, 0, reinterpret_cast<float*>(ws + p.off_G), p.pitchG, reinterpret_cast<float*>(ws + p.off_stats)};
}
const float* sweep_input(const pulscan_plan& p) {
    char* ws = static_cast<char*>(p.ws);
    return reinterpret_cast<const float*>(ws + (p.keep_P ? p.off_P : p.off_G));
}
PowerSource power_source(const pulscan_plan& p, const void* d_spectra) {
    char* ws = static_cast<char*>(p.ws);
    PowerSource s{};
    s.P = p.keep_P ? reinterpret_cast<const float*>(ws + p.off_P) : nullptr;
    s.pitchP = p.pitchP;
    s.spectra = reinterpret_cast<const float2*>(d_spectra);
    s.pitch = p.pitch;
    s.stats = p.keep_P ? nullptr : reinterpret_cast<const float*>(ws + p.off_stats);
    s.B = p.B; s.nb = p.nb;
    return s;
}

// The search entry points only look at host state here: no CUDA call, no allocation.
int check_plan_ready(pulscan_plan* plan) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (!plan->ws) return fail(PULSCAN_ENOWORKSPACE, "no workspace attached (pulscan_plan_set_workspace)");
    if (plan->dirty || !plan->finalized)
        return fail(PULSCAN_ENOWORKSPACE, "the plan was changed after pulscan_plan_set_workspace: attach the workspace again "
                                          "(pulscan_plan_workspace_bytes may have changed)");
    return PULSCAN_OK;
}

} // namespace

// ---------------------------------------------------------------------------------------------------- C ABI
extern "C" {

pulscan_plan* pulscan_plan_create(int64_t n_bins, int32_t batch, int32_t zmax, int32_t block_width,
                                  float sigma_threshold) {
    auto bad = [](const char* fmt, auto... a) -> pulscan_plan* { fail(PULSCAN_EINVAL, fmt, a...); return nullptr; };
    if (n_bins < 2 || n_bins > 2147483647LL - 65536) return bad("n_bins = %lld out of range [2, 2^31 - 2^16)", (long long)n_bins);
    if (batch < 1) return bad("batch = %d < 1", batch);
    if (zmax < 1 || zmax > PULSCAN_MAX_ZMAX) return bad("zmax = %d out of range [1, %d]", zmax, PULSCAN_MAX_ZMAX);
    if ((int64_t)zmax >= n_bins) return bad("zmax = %d must be < n_bins = %lld", zmax, (long long)n_bins);
    if (block_width < 1) return bad("block_width = %d < 1", block_width);
    if (block_width > PULSCAN_MAX_BLOCK_WIDTH) return bad("block_width = %d exceeds %d", block_width, PULSCAN_MAX_BLOCK_WIDTH);
    if (!(sigma_threshold > 0.f) || !std::isfinite(sigma_threshold)) return bad("sigma_threshold must be finite and > 0");
    const int64_t nblk = (n_bins + block_width - 1) / block_width;
    if (nblk * batch >= 2147483648LL) return bad("batch · candidate blocks = %lld ≥ 2^31", (long long)(nblk * batch));
    pulscan_plan* p = new (std::nothrow) pulscan_plan;
    if (!p) return bad("out of host memory");
    p->n = n_bins; p->batch = batch; p->zmax = zmax; p->C = block_width; p->sigma_thr = sigma_threshold;
    p->pitch = n_bins;
    int nbk = pow2_ceil(16 * block_width);
    p->B = std::min(8192, std::max(1024, nbk));
    g_last_error.clear();
    return p;
}

int pulscan_plan_set_norm_block(pulscan_plan* plan, int32_t norm_block) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (norm_block < 2 || norm_block > PULSCAN_MAX_NORM_BLOCK)
        return fail(PULSCAN_EINVAL, "norm_block = %d out of range [2, %d]", norm_block, PULSCAN_MAX_NORM_BLOCK);
    plan->B = norm_block; invalidate(*plan);
    return PULSCAN_OK;
}

int pulscan_plan_set_trials(pulscan_plan* plan, double n_trials) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (!(n_trials >= 1.0) || !std::isfinite(n_trials)) return fail(PULSCAN_EINVAL, "n_trials must be finite and ≥ 1");
    plan->n_trials = n_trials; invalidate(*plan);
    return PULSCAN_OK;
}

int pulscan_plan_set_pitch(pulscan_plan* plan, int64_t pitch_bins) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (pitch_bins < plan->n) return fail(PULSCAN_EINVAL, "pitch = %lld < n_bins = %lld", (long long)pitch_bins, (long long)plan->n);
    plan->pitch = pitch_bins; invalidate(*plan);
    return PULSCAN_OK;
}

int pulscan_plan_set_mode(pulscan_plan* plan, int32_t mode) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (mode != 0 && mode != 1) return fail(PULSCAN_EINVAL, "mode must be 0 (pruned) or 1 (exhaustive)");
    if (plan->mode != mode) invalidate(*plan);   // the exhaustive sweep needs the per-bin power array in the workspace
    plan->mode = mode;
    return PULSCAN_OK;
}

int pulscan_plan_set_width_sampling(pulscan_plan* plan, int32_t z_step, int32_t logarithmic) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (z_step < 1) return fail(PULSCAN_EINVAL, "z_step = %d < 1", z_step);
    plan->z_step = z_step; plan->log_sampling = logarithmic != 0;
    invalidate(*plan);
    return PULSCAN_OK;
}

int pulscan_plan_set_r_block(pulscan_plan* plan, int32_t enable) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    plan->r_block = enable != 0;
    return PULSCAN_OK;
}

int pulscan_plan_set_normalisation(pulscan_plan* plan, int32_t mode) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (mode != 0 && mode != 1) return fail(PULSCAN_EINVAL, "mode must be 0 (exact median/MAD) or 1 (median of medians, Alg. 1)");
    if (mode == 1) {
        const int B = plan->B;
        if (B < 256 || B > 16384 || (B & (B - 1)) != 0)
            return fail(PULSCAN_EINVAL, "median-of-medians normalisation needs norm_block = 256 … 16384, a power of two (it is %d)", B);
        if (plan->n < B) return fail(PULSCAN_EINVAL, "median-of-medians normalisation needs n_bins >= norm_block");
    }
    if (plan->norm_mode != mode) invalidate(*plan);
    plan->norm_mode = mode;
    return PULSCAN_OK;
}

int pulscan_plan_set_significance(pulscan_plan* plan, int32_t mode) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (mode != 0 && mode != 1) return fail(PULSCAN_EINVAL, "mode must be 0 (exact chi-squared tail) or 1 (polynomial ln p, Alg. 3)");
    plan->signif_mode = mode;
    invalidate(*plan);       // the per-width power thresholds follow the significance function
    return PULSCAN_OK;
}

int pulscan_plan_set_emission(pulscan_plan* plan, int32_t per_width, int64_t capacity) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (per_width != 0 && per_width != 1) return fail(PULSCAN_EINVAL, "per_width must be 0 or 1");
    if (per_width && (capacity < 1 || capacity > 0x7FFFFFFFll)) return fail(PULSCAN_EINVAL, "per-width emission needs a capacity in [1, 2^31)");
    plan->per_width = per_width;
    plan->user_capacity = per_width ? capacity : 0;
    plan->out_capacity = per_width ? (unsigned)capacity : 0xFFFFFFFFu;
    if (plan->host_staging) invalidate(*plan);   // the staging area for the records is sized from the capacity
    return PULSCAN_OK;
}

int pulscan_plan_set_tuning(pulscan_plan* plan, int32_t tile_bins, double log10_p_flag) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (tile_bins != 0 && (tile_bins < 1024 || tile_bins > 16384 || tile_bins % 512 != 0))
        return fail(PULSCAN_EINVAL, "tile_bins must be 0 or a multiple of 512 in [1024, 16384]");
    if (log10_p_flag != 0.0 && !(log10_p_flag <= -1.0 && log10_p_flag >= -9.0))
        return fail(PULSCAN_EINVAL, "log10_p_flag must be 0 or in [-9, -1]");
    plan->tile_user = tile_bins;
    plan->log10_p_flag = (log10_p_flag == 0.0) ? kDefaultLog10PFlag : log10_p_flag;
    invalidate(*plan);
    return PULSCAN_OK;
}

int pulscan_plan_set_variant(pulscan_plan* plan, int32_t which, int32_t value) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    switch (which) {
        case PULSCAN_VARIANT_SWEEP_SECOND_LOOK:
            if (value != 0 && value != 1) return fail(PULSCAN_EINVAL, "PULSCAN_VARIANT_SWEEP_SECOND_LOOK takes 0 or 1");
            plan->v_second_look = value; break;
        case PULSCAN_VARIANT_SCAN_QUADS:
            if (value != 0 && value != 5) return fail(PULSCAN_EINVAL, "PULSCAN_VARIANT_SCAN_QUADS takes 0 (automatic) or 5");
            plan->v_scan_quads = value; break;
        case PULSCAN_VARIANT_NORM_KEEP_INDICES:
            if (value < -1 || value > 1) return fail(PULSCAN_EINVAL, "PULSCAN_VARIANT_NORM_KEEP_INDICES takes -1 (automatic), 0 or 1");
            plan->v_keepidx = value; break;
        case PULSCAN_VARIANT_NORM_L2_AHEAD:
            if (value < -1 || value > (1 << 20)) return fail(PULSCAN_EINVAL, "PULSCAN_VARIANT_NORM_L2_AHEAD takes -1 (automatic) or 0 … 2^20 CTAs");
            plan->v_l2_ahead = value; break;
        case PULSCAN_VARIANT_NORM_SINGLE_HISTOGRAM:
            if (value != 0 && value != 1) return fail(PULSCAN_EINVAL, "PULSCAN_VARIANT_NORM_SINGLE_HISTOGRAM takes 0 or 1");
            plan->v_single_hist = value; break;
        case PULSCAN_VARIANT_KEEP_POWER:
            if (value != 0 && value != 1) return fail(PULSCAN_EINVAL, "PULSCAN_VARIANT_KEEP_POWER takes 0 or 1");
            plan->v_keep_power = value; break;
        default: return fail(PULSCAN_EINVAL, "unknown variant %d", which);
    }
    invalidate(*plan);
    return PULSCAN_OK;
}

int pulscan_plan_set_cell_capacity(pulscan_plan* plan, int64_t cells) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (cells < 0 || cells > (1ll << 28)) return fail(PULSCAN_EINVAL, "cell capacity out of range [0, 2^28]");
    plan->cell_cap_user = (unsigned)cells; invalidate(*plan);
    return PULSCAN_OK;
}

int64_t pulscan_plan_max_candidates(const pulscan_plan* plan) {
    if (!plan) { fail(PULSCAN_EINVAL, "null plan"); return -1; }
    if (plan->per_width) return plan->user_capacity;
    return (int64_t)plan->batch * ((plan->n + plan->C - 1) / plan->C);
}

size_t pulscan_plan_workspace_bytes(const pulscan_plan* plan) {
    if (!plan) { fail(PULSCAN_EINVAL, "null plan"); return 0; }
    if (derive(*const_cast<pulscan_plan*>(plan))) return 0;
    return plan->need_bytes;
}

int pulscan_plan_enable_host_staging(pulscan_plan* plan, int32_t enable) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    plan->host_staging = enable != 0; invalidate(*plan);
    return PULSCAN_OK;
}

int pulscan_plan_set_workspace(pulscan_plan* plan, void* d_workspace, size_t bytes) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    int rc = derive(*plan);
    if (rc) return rc;
    if (!d_workspace) return fail(PULSCAN_EINVAL, "null workspace");
    if (reinterpret_cast<uintptr_t>(d_workspace) & 255) return fail(PULSCAN_EINVAL, "workspace must be 256-byte aligned");
    if (bytes < plan->need_bytes)
        return fail(PULSCAN_ENOWORKSPACE, "workspace too small: %zu bytes given, %zu needed", bytes, plan->need_bytes);
    plan->ws = d_workspace; plan->ws_bytes = bytes;
    attach_children(*plan);
    for (pulscan_plan* c : plan->harm)
        if ((rc = finalize_device(*c))) return rc;
    return finalize_device(*plan);
}

int64_t pulscan_plan_power_pitch(const pulscan_plan* plan) {
    if (!plan) { fail(PULSCAN_EINVAL, "null plan"); return -1; }
    return (int64_t)align_up((size_t)plan->n, 4);
}

int pulscan_normalise_power(pulscan_plan* plan, const void* d_spectra, float* d_power, void* cuda_stream) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    int rc = derive(*plan);
    if (rc) return rc;
    if (!d_spectra || !d_power) return fail(PULSCAN_EINVAL, "null pointer");
    if (reinterpret_cast<uintptr_t>(d_spectra) & 7) return fail(PULSCAN_EINVAL, "d_spectra must be 8-byte aligned");
    if (reinterpret_cast<uintptr_t>(d_power) & 15) return fail(PULSCAN_EINVAL, "d_power must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (plan->ws && plan->finalized) { // workspace attached: same kernels as pulscan_search
        char* ws = static_cast<char*>(plan->ws);
        unsigned* d_counters = reinterpret_cast<unsigned*>(ws + plan->off_counters);
        CUDA_TRY(cudaMemsetAsync(d_counters, 0, 256, st));
        return enqueue_norm(*plan, d_spectra, NormOut{d_power, plan->pitchP, nullptr, 0, nullptr}, st,
                            reinterpret_cast<unsigned*>(ws + plan->off_redo), d_counters + 1);
    }
    return enqueue_norm(*plan, d_spectra, NormOut{d_power, plan->pitchP, nullptr, 0, nullptr}, st, nullptr, nullptr); // no workspace: general kernels only
}

int64_t pulscan_plan_group_pitch(const pulscan_plan* plan) {
    if (!plan) { fail(PULSCAN_EINVAL, "null plan"); return -1; }
    return (int64_t)align_up((size_t)((plan->n + 3) / 4), 4);
}

int pulscan_normalise_group_sums(pulscan_plan* plan, const void* d_spectra, float* d_group_sums, float* d_block_stats,
                                 void* cuda_stream) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    int rc = derive(*plan);
    if (rc) return rc;
    if (!d_spectra || !d_group_sums || !d_block_stats) return fail(PULSCAN_EINVAL, "null pointer");
    if (reinterpret_cast<uintptr_t>(d_spectra) & 7) return fail(PULSCAN_EINVAL, "d_spectra must be 8-byte aligned");
    if ((reinterpret_cast<uintptr_t>(d_group_sums) | reinterpret_cast<uintptr_t>(d_block_stats)) & 31)
        return fail(PULSCAN_EINVAL, "d_group_sums / d_block_stats must be 32-byte aligned");
    if (plan->B & 3) return fail(PULSCAN_EINVAL, "group sums need norm_block to be a multiple of 4 (it is %d)", plan->B);
    if (plan->norm_mode == 1) return fail(PULSCAN_EINVAL, "group sums are written by the exact normalisation kernels only");
    if (!plan->ws || !plan->finalized) return fail(PULSCAN_ENOWORKSPACE, "no workspace attached (pulscan_plan_set_workspace)");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    char* ws = static_cast<char*>(plan->ws);
    unsigned* d_counters = reinterpret_cast<unsigned*>(ws + plan->off_counters);
    CUDA_TRY(cudaMemsetAsync(d_counters, 0, 256, st));
    return enqueue_norm(*plan, d_spectra, NormOut{nullptr, 0, d_group_sums, plan->pitchG, d_block_stats}, st,
                        reinterpret_cast<unsigned*>(ws + plan->off_redo), d_counters + 1);
}

int pulscan_search(pulscan_plan* plan, const void* d_spectra, pulscan_candidate* d_candidates, uint32_t* d_count,
                   void* cuda_stream) {
    int rc = check_plan_ready(plan);
    if (rc) return rc;
    if (!d_spectra || !d_candidates || !d_count) return fail(PULSCAN_EINVAL, "null pointer");
    if (reinterpret_cast<uintptr_t>(d_spectra) & 7) return fail(PULSCAN_EINVAL, "d_spectra must be 8-byte aligned");
    if (reinterpret_cast<uintptr_t>(d_candidates) & 3 || reinterpret_cast<uintptr_t>(d_count) & 3)
        return fail(PULSCAN_EINVAL, "d_candidates / d_count must be 4-byte aligned");
    pulscan_plan& p = *plan;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    char* ws = static_cast<char*>(p.ws);
    unsigned* d_bitmap = reinterpret_cast<unsigned*>(ws + p.off_bitmap);
    unsigned* d_counters = reinterpret_cast<unsigned*>(ws + p.off_counters);

    cudaEvent_t* ev = nullptr;
    if (p.prof_slots > 0) {
        ev = &p.prof_events[(size_t)(p.prof_next % p.prof_slots) * 5];
        ++p.prof_next;
        CUDA_TRY(cudaEventRecord(ev[0], st));
    }
    CUDA_TRY(cudaMemsetAsync(d_bitmap, 0, p.bitmap_bytes, st));
    CUDA_TRY(cudaMemsetAsync(d_counters, 0, 256, st));
    CUDA_TRY(cudaMemsetAsync(d_count, 0, sizeof(uint32_t), st));

    if (ev) CUDA_TRY(cudaEventRecord(ev[1], st));
    rc = enqueue_norm(p, d_spectra, norm_outputs(p), st, reinterpret_cast<unsigned*>(ws + p.off_redo), d_counters + 1); // (a)
    if (rc) return rc;
    if (ev) CUDA_TRY(cudaEventRecord(ev[2], st));

    rc = enqueue_sweep_exact(p, sweep_input(p), power_source(p, d_spectra), d_candidates, nullptr, d_count, st, ev);
    if (rc) return rc;
    if (ev) CUDA_TRY(cudaEventRecord(ev[4], st));
    return debug_sync("block_exact_kernel");
}

int pulscan_plan_set_harmonics(pulscan_plan* plan, int32_t numharm) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (numharm < 1 || numharm > 4) return fail(PULSCAN_EINVAL, "numharm = %d out of range [1, 4]", numharm);
    if ((int64_t)plan->zmax >= plan->n / numharm)
        return fail(PULSCAN_EINVAL, "zmax = %d must be < floor(n_bins / numharm) = %lld", plan->zmax, (long long)(plan->n / numharm));
    plan->numharm = numharm; invalidate(*plan);
    return PULSCAN_OK;
}

int64_t pulscan_plan_max_hcandidates(const pulscan_plan* plan) {
    if (!plan) { fail(PULSCAN_EINVAL, "null plan"); return -1; }
    if (plan->per_width) return plan->user_capacity;
    int64_t total = 0;
    for (int H = 1; H <= plan->numharm; ++H) total += (int64_t)plan->batch * ((plan->n / H + plan->C - 1) / plan->C);
    return total;
}

int pulscan_search_harmonics(pulscan_plan* plan, const void* d_spectra, pulscan_hcandidate* d_hcandidates, uint32_t* d_count,
                             void* cuda_stream) {
    int rc = check_plan_ready(plan);
    if (rc) return rc;
    if (!d_spectra || !d_hcandidates || !d_count) return fail(PULSCAN_EINVAL, "null pointer");
    if (reinterpret_cast<uintptr_t>(d_spectra) & 7) return fail(PULSCAN_EINVAL, "d_spectra must be 8-byte aligned");
    if (reinterpret_cast<uintptr_t>(d_hcandidates) & 3 || reinterpret_cast<uintptr_t>(d_count) & 3)
        return fail(PULSCAN_EINVAL, "d_hcandidates / d_count must be 4-byte aligned");
    pulscan_plan& p = *plan;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    char* ws = static_cast<char*>(p.ws);
    float* d_P = reinterpret_cast<float*>(ws + p.off_P);
    unsigned* d_counters = reinterpret_cast<unsigned*>(ws + p.off_counters);
    CUDA_TRY(cudaMemsetAsync(ws + p.off_bitmap, 0, p.bitmap_bytes, st));
    CUDA_TRY(cudaMemsetAsync(d_counters, 0, 256, st));
    CUDA_TRY(cudaMemsetAsync(d_count, 0, sizeof(uint32_t), st));
    rc = enqueue_norm(p, d_spectra, norm_outputs(p), st, reinterpret_cast<unsigned*>(ws + p.off_redo), d_counters + 1);   // (a)
    if (rc) return rc;
    if ((rc = enqueue_sweep_exact(p, sweep_input(p), power_source(p, d_spectra), nullptr, d_hcandidates, d_count, st, nullptr)))
        return rc;                                                                                              // Y_1 = P
    if (!p.harm.empty() && !p.keep_P) return fail(PULSCAN_EINVAL, "internal: the harmonic sum needs the per-bin power array");
    if (!p.harm.empty()) {                                                                                      // Y_2 … in one pass
        HarmonicOut ho{};
        for (size_t k = 0; k < p.harm.size(); ++k) {
            pulscan_plan& c = *p.harm[k];
            ho.Y[k] = reinterpret_cast<float*>(static_cast<char*>(c.ws) + c.off_P);
            ho.pitch[k] = c.pitchP; ho.nH[k] = c.n;
        }
        const long long total = (long long)p.batch * ho.nH[0];
        const int grid = (int)std::min<long long>((total + kHarmThreads - 1) / kHarmThreads, (long long)p.sm_count * 16);
        switch ((int)p.harm.size() + 1) {
            case 2: harmonic_sum_kernel<2><<<grid, kHarmThreads, 0, st>>>(d_P, p.pitchP, ho, total); break;
            case 3: harmonic_sum_kernel<3><<<grid, kHarmThreads, 0, st>>>(d_P, p.pitchP, ho, total); break;
            default: harmonic_sum_kernel<4><<<grid, kHarmThreads, 0, st>>>(d_P, p.pitchP, ho, total); break;
        }
        CUDA_TRY(cudaGetLastError());
        if ((rc = debug_sync("harmonic_sum_kernel"))) return rc;
    }
    for (pulscan_plan* cp : p.harm) {
        pulscan_plan& c = *cp;
        c.mode = p.mode; c.r_block = p.r_block; c.per_width = p.per_width; c.out_capacity = p.out_capacity;
        char* cws = static_cast<char*>(c.ws);
        CUDA_TRY(cudaMemsetAsync(cws + c.off_bitmap, 0, c.bitmap_bytes, st));
        CUDA_TRY(cudaMemsetAsync(cws + c.off_counters, 0, 256, st));
        if ((rc = enqueue_sweep_exact(c, sweep_input(c), power_source(c, nullptr), nullptr, d_hcandidates, d_count, st, nullptr))) return rc;
    }
    return PULSCAN_OK;
}

int pulscan_search_host(pulscan_plan* plan, const void* h_spectra, pulscan_candidate* h_candidates, uint32_t* h_count,
                        void* cuda_stream) {
    int rc = check_plan_ready(plan);
    if (rc) return rc;
    if (!plan->host_staging) return fail(PULSCAN_EINVAL, "host staging not enabled (pulscan_plan_enable_host_staging)");
    if (!h_spectra || !h_candidates || !h_count) return fail(PULSCAN_EINVAL, "null pointer");
    pulscan_plan& p = *plan;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    char* ws = static_cast<char*>(p.ws);
    void* d_in = ws + p.off_stage_in;
    pulscan_candidate* d_cand = reinterpret_cast<pulscan_candidate*>(ws + p.off_stage_cand);
    uint32_t* d_cnt = reinterpret_cast<uint32_t*>(ws + p.off_stage_count);
    CUDA_TRY(cudaMemcpyAsync(d_in, h_spectra, (size_t)p.batch * p.pitch * 8, cudaMemcpyHostToDevice, st));
    rc = pulscan_search(plan, d_in, d_cand, d_cnt, cuda_stream);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpyAsync(h_count, d_cnt, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    // per-width emission: *h_count is the number FOUND; only the first `capacity` records exist (and fit h_candidates)
    const size_t ncopy = std::min<size_t>(*h_count, p.per_width ? (size_t)p.user_capacity : (size_t)*h_count);
    if (ncopy)
        CUDA_TRY(cudaMemcpyAsync(h_candidates, d_cand, ncopy * sizeof(pulscan_candidate), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return PULSCAN_OK;
}

int pulscan_plan_get_thresholds(const pulscan_plan* plan, double* h_T) {
    if (!plan || !h_T) return fail(PULSCAN_EINVAL, "null pointer");
    int rc = derive(*const_cast<pulscan_plan*>(plan));
    if (rc) return rc;
    std::memcpy(h_T, plan->T.data(), plan->T.size() * sizeof(double));
    return PULSCAN_OK;
}

int64_t pulscan_plan_describe(const pulscan_plan* plan, char* h_buf, int64_t buf_bytes) {
    if (!plan) { fail(PULSCAN_EINVAL, "null plan"); return -1; }
    if (derive(*const_cast<pulscan_plan*>(plan))) return -1;
    const pulscan_plan& p = *plan;
    std::string s;
    char line[512];
    snprintf(line, sizeof line,
             "pulscan plan: n_bins=%lld batch=%d zmax=%d block_width=%d norm_block=%d sigma_threshold=%g n_trials=%g pitch=%lld mode=%s\n",
             (long long)p.n, p.batch, p.zmax, p.C, p.B, p.sigma_thr, p.n_trials, (long long)p.pitch, p.mode ? "exhaustive" : "pruned");
    s += line;
    snprintf(line, sizeof line, "options: widths searched = %s, location = %s, normalisation = %s, significance = %s, numharm = %d\n",
             p.log_sampling ? "z = 0, 1, 2, 4, ... (L411)" : (p.z_step == 1 ? "every width" : "every z_step-th drift (L152)"),
             p.r_block ? "R-Block (L222-226)" : "exact bin", p.norm_mode ? "median of medians (Alg. 1)" : "exact median/MAD",
             p.signif_mode ? "polynomial ln p (Alg. 3)" : "exact chi-squared tail", p.numharm);
    s += line;
    snprintf(line, sizeof line, "norm: %d blocks/row, main %s<EPT=%d,NT=%d> x %d/row%s\n", p.nb, p.use_fast ? "single-histogram" : "general",
             p.use_fast ? p.B / p.norm_nt : p.ept_main, p.use_fast ? p.norm_nt : p.nt_main, p.main_blocks_per_row,
             p.has_tail ? "" : " (no tail launch)");
    s += line;
    if (p.has_tail) { snprintf(line, sizeof line, "norm tail: <EPT=%d,NT=%d> x 1/row\n", p.ept_tail, p.nt_tail); s += line; }
    auto sweep_lines = [&](const pulscan_plan& q, const char* tag) {
        double evals = 0;
        for (int l = 0; l < q.sp.nlevels; ++l) {
            const SweepLevel& lv = q.sp.lv[l];
            const double ev = 4.0 * lv.nsteps / (double)(1 << lv.lg);
            evals += ev;
            snprintf(line, sizeof line,
                     "sweep%s level %d: g=%d widths [%d,%d] covers m=[%d,%d] steps=%d warp-tasks/tile=%d  (%.3f cover sums per bin)\n", tag, l,
                     1 << lv.lg, lv.wlo, lv.whi, lv.m_lo, lv.m_hi, lv.nsteps, lv.nwt, ev);
            s += line;
        }
        snprintf(line, sizeof line,
                 "sweep%s: tile=%d len=%d tiles/row=%d smem=%zu B, %.3f cover sums per bin (exhaustive: %d), p_flag=1e%g, scan: %d quads per thread x %d pass(es)%s\n",
                 tag, q.sp.tile, q.sp.len, q.tiles_per_row, q.smem_sweep, evals, q.zmax, q.log10_p_flag, q.sp.scan_nq, q.sp.npass,
                 q.sweep_fine ? ", full resolution" : "");
        s += line;
    };
    if (!p.pruned_error.empty()) {
        snprintf(line, sizeof line, "pruned sweep unavailable (pulscan_plan_set_workspace fails in mode 0): %s\n", p.pruned_error.c_str());
        s += line;
    }
    sweep_lines(p, "");
    for (size_t h = 0; h < p.harm.size(); ++h) {
        char tag[16];
        snprintf(tag, sizeof tag, " Y_%d", (int)h + 2);
        if (!derive(*p.harm[h])) sweep_lines(*p.harm[h], tag);
    }
    snprintf(line, sizeof line, "intermediate in HBM: %s\n",
             p.keep_P ? "float32 power of every bin (4 B/bin)" : "sums of 4-bin groups (1 B/bin) + 32 B per normalisation block");
    s += line;
    snprintf(line, sizeof line, "exact: 4 widths per thread, start bins split over %d lanes, widths of a block dealt to %d CTA(s), %d segment(s) of %d start bins per block\n",
             1 << p.exact_lg_split, p.exact_parts, (p.C + p.exact_seg - 1) / p.exact_seg, std::min(p.C, p.exact_seg));
    s += line;
    snprintf(line, sizeof line, "exact: smem=%zu B; workspace=%zu B; T_1=%.4f T_zmax=%.4f\n", p.smem_exact, p.need_bytes, p.T.front(), p.T.back());
    s += line;
    const int64_t need = (int64_t)s.size() + 1;
    if (h_buf && buf_bytes > 0) {
        const size_t ncopy = (size_t)std::min<int64_t>(buf_bytes - 1, (int64_t)s.size());
        std::memcpy(h_buf, s.data(), ncopy);
        h_buf[ncopy] = 0;
    }
    return need;
}

int pulscan_plan_get_stats(pulscan_plan* plan, uint32_t* h_stats, void* cuda_stream) {
    int rc = check_plan_ready(plan);
    if (rc) return rc;
    if (!h_stats) return fail(PULSCAN_EINVAL, "null pointer");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    CUDA_TRY(cudaMemcpyAsync(h_stats, static_cast<char*>(plan->ws) + plan->off_counters, 16 * sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return PULSCAN_OK;
}

int32_t pulscan_plan_launches_per_search(const pulscan_plan* plan) {
    if (!plan) { fail(PULSCAN_EINVAL, "null plan"); return -1; }
    if (derive(*const_cast<pulscan_plan*>(plan))) return -1;
    const int norm = plan->norm_mode == 1 ? 1 : (plan->main_blocks_per_row > 0 ? (plan->use_fast ? 2 : 1) : 0) + (plan->has_tail ? 1 : 0);
    return norm + (plan->mode == 0 ? 3 : 2);
}

int pulscan_plan_set_profiling(pulscan_plan* plan, int32_t n_slots) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    if (n_slots < 0 || n_slots > 65536) return fail(PULSCAN_EINVAL, "n_slots out of range [0, 65536]");
    release_profiling(*plan);
    plan->prof_slots = 0;
    plan->prof_events.resize((size_t)n_slots * 5);
    for (cudaEvent_t& e : plan->prof_events) {
        e = nullptr;
        const cudaError_t err = cudaEventCreate(&e);
        if (err != cudaSuccess) {
            release_profiling(*plan);
            return fail(PULSCAN_ECUDA, "cudaEventCreate failed: %s", cudaGetErrorString(err));
        }
    }
    plan->prof_slots = n_slots;
    return PULSCAN_OK;
}

int pulscan_plan_get_profile(pulscan_plan* plan, int32_t slot, float* h_ms) {
    if (!plan || !h_ms) return fail(PULSCAN_EINVAL, "null pointer");
    if (slot < 0 || slot >= plan->prof_slots || plan->prof_events.empty() || slot >= plan->prof_next)
        return fail(PULSCAN_EINVAL, "profiling slot %d not recorded", slot);
    cudaEvent_t* ev = &plan->prof_events[(size_t)slot * 5];
    CUDA_TRY(cudaEventSynchronize(ev[4]));
    for (int k = 0; k < 4; ++k) CUDA_TRY(cudaEventElapsedTime(&h_ms[k], ev[k], ev[k + 1]));
    return PULSCAN_OK;
}

int pulscan_plan_destroy(pulscan_plan* plan) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    for (pulscan_plan* c : plan->harm) pulscan_plan_destroy(c);
    release_profiling(*plan);
    delete plan;
    return PULSCAN_OK;
}

// ------------------------------------------------------------------------------------ static-scratch entry point
// pulscan_normalise_power_static: steps 1-2 for callers that have no device memory to give beyond their input and output.
// The exact normalisation's fast kernel needs a little scratch: a list of the blocks it hands to the general kernel and a few
// counters.  Everywhere else in this library that scratch is part of the caller's workspace; here it is the array below, which
// is part of the loaded library image on every GPU (≈ 1 MiB, held until the process exits).
//
// g_static_scratch is only a device address inside device code.  In the host code of this file the name is a handle for the
// runtime, so the real address is asked for once per device (cudaGetSymbolAddress, with that device current) and remembered.
namespace {

constexpr unsigned kStaticCounterWords = 64;   // [1] = entries in the list, [4..8] = why blocks were handed over; 256 bytes
static __device__ __align__(256) unsigned g_static_scratch[kStaticCounterWords + PULSCAN_STATIC_MAX_NORM_BLOCKS];

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
unsigned* g_static_addr[kStaticMaxDevices] = {};   // per device ordinal; nullptr = not set up yet

// Set-up on first use per device: architecture check, kernel attributes, address of the array on the CURRENT device.
int static_scratch_on_current_device(unsigned** out) {
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(PULSCAN_EINVAL, "device ordinal %d beyond the %d this entry point tracks", dev, kStaticMaxDevices);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        int major = 0;
        CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        if (major != 10) return fail(PULSCAN_EARCH, "device %d is compute capability %d.x; libpulscan is built for sm_100a only", dev, major);
        pulscan_plan none;
        const int rc = set_kernel_attributes(none);
        if (rc) return rc;
        unsigned* addr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&addr), g_static_scratch);
        if (e != cudaSuccess || !addr)
            return fail(PULSCAN_ECUDA, "cudaGetSymbolAddress(g_static_scratch) failed on device %d: %s", dev, cudaGetErrorString(e));
        g_static_addr[dev] = addr;
    }
    *out = g_static_addr[dev];
    return PULSCAN_OK;
}

} // namespace

int pulscan_normalise_power_static(pulscan_plan* plan, const void* d_spectra, float* d_power, void* cuda_stream) {
    if (!plan) return fail(PULSCAN_EINVAL, "null plan");
    int rc = derive(*plan);
    if (rc) return rc;
    if (plan->norm_mode == 1)
        return fail(PULSCAN_EINVAL, "the Alg. 1 normalisation uses no scratch: call pulscan_normalise_power (it allocates nothing either)");
    const long long blocks = (long long)plan->batch * plan->nb;
    if (blocks > (long long)PULSCAN_STATIC_MAX_NORM_BLOCKS)
        return fail(PULSCAN_EINVAL, "batch x normalisation blocks per spectrum = %lld exceeds PULSCAN_STATIC_MAX_NORM_BLOCKS = %d: "
                                    "pass fewer spectra per call or use a longer norm_block", blocks, (int)PULSCAN_STATIC_MAX_NORM_BLOCKS);
    if (!d_spectra || !d_power) return fail(PULSCAN_EINVAL, "null pointer");
    if (reinterpret_cast<uintptr_t>(d_spectra) & 7) return fail(PULSCAN_EINVAL, "d_spectra must be 8-byte aligned");
    if (reinterpret_cast<uintptr_t>(d_power) & 15) return fail(PULSCAN_EINVAL, "d_power must be 16-byte aligned");
    unsigned* scratch = nullptr;
    if ((rc = static_scratch_on_current_device(&scratch))) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // the array still holds the previous call's counters and list: the counters must start at zero, the list is only read up
    // to the new count
    CUDA_TRY(cudaMemsetAsync(scratch, 0, kStaticCounterWords * sizeof(unsigned), st));
    return enqueue_norm(*plan, d_spectra, NormOut{d_power, plan->pitchP, nullptr, 0, nullptr}, st, scratch + kStaticCounterWords,
                        scratch + 1);
}

const char* pulscan_last_error(void) { return g_last_error.c_str(); }
const char* pulscan_version(void) { return "pulscan-b200 0.1.0 (sm_100a)"; }

} // extern "C"
