// boxcar_sweep.cuh — kernel (b): the boxcar sweep over the float32 power spectrum.
//
// What must be found (§2.2.5; Alg. 4): for every start bin i and every width
// w ≤ zmax the sum S(i,w) = Σ_{j<w} P[i+j], and per candidate block the maxima.  A window can only become a candidate
// if S(i,w) ≥ T_w, the power at which width w reaches the σ threshold (L342-344: "compared with precomputed
// threshold values").  In noise that happens for ~1e-9 of all (i,w), so this stage is a FILTER: it marks the
// candidate blocks that contain at least one window with S ≥ T_w·(1−ε) and kernel (c) then evaluates exactly those
// blocks in double precision.  Nothing a marked block could emit is lost and an unmarked block cannot emit.
//
// The paper's kernel (Alg. 4) does one shared-memory add per (bin, width) — issue-bound, ~2·zmax instructions per
// bin.  Here the work is split in two kernels:
//
//  boxcar_sweep_kernel (streaming, every bin): persistent CTAs stride over tiles; a tile (+ zmax halo) lands in one of
//    two shared-memory buffers by a TMA bulk copy issued a whole tile ahead.  Each thread sums its 5 quads of powers and
//    a CTA scan turns the quad sums into PG4[k] = PP[4k] (PP[i] = Σ_{j<i} P[j]) and its decimations PG8, PG16, …
//    COVER SUMS: P ≥ 0, so a window of width w is bounded above by the sum of the aligned g-bin groups that cover it,
//    U(k0,m) = PG_g[k0+m] − PG_g[k0].  For a level (g, [wlo, whi]) a thread holds PG at 8 consecutive group starts in
//    registers and slides over m: one FADD + half an FMNMX3 per cover sum, (n/g)·(whi/g+2) cover sums instead of
//    n·(whi−wlo+1) window sums.  g ∈ {4, 8, 16, …} grows like √w (chosen on the host so that a cover of pure noise
//    passes with probability ≤ p_flag), which makes every level cost O(n).  A cell (8 group starts × 4 cover lengths)
//    with a passing cover is appended to a global list — ≈ 0.6 cells per 4096-bin tile in noise.
//  sweep_refine_kernel (rare path, one warp per listed cell): re-reads the cell's span of P, builds its prefix sum in
//    double, re-tests the 32 covers and sums the ≤ g² windows of each passing cover against their own T'_w; blocks
//    with a window that reaches T'_w are marked (bitmap + list).
//
// Float safety of the streaming kernel.  Every PG entry carries at most D = scan_roundings(NQ, passes) roundings of magnitude
// ≤ 2⁻²⁴·PP[len] (counted step by step at scan_roundings below: 26 for the one-pass scans of 11 quads per thread, 28 for five
// passes of 5 quads), so a cover sum, the rounded difference of two entries, is off by at most (2·D + 1)·2⁻²⁴·PP[len] ≤ slack =
// kSlackUlps·2⁻²⁴·PP[len] from the exact sum of the float32 powers (scan_tile asserts it for every NQ it is compiled for); the
// cover test adds the slack on the keeping side.  The refine kernel works in double and compares with T'_w, which
// the host rounds down by 2w·2⁻²⁴ + 2·10⁻⁶ relative.
//
// Exhaustive mode (the cross-check) evaluates every (i, w) by the paper's recursion instead.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "power_source.cuh"

namespace pulscan {

constexpr int kMaxLevels = 8;
constexpr int kSweepThreads = 256;
constexpr int kSweepR = 8;                 // consecutive group starts per thread
constexpr int kScanTail = 48;              // zeros kept after a landing buffer's len powers (12 after its len/4 group sums): the
                                           // last scanning thread's run of ≤ 11 quads may start before len and end after it
#ifndef PULSCAN_SWEEP_BUFS
#define PULSCAN_SWEEP_BUFS 2
#endif
#ifndef PULSCAN_SWEEP_OCC
#define PULSCAN_SWEEP_OCC 4
#endif
constexpr int kSweepBufs = PULSCAN_SWEEP_BUFS;   // landing buffers per CTA (copies in flight ahead of the scan)
constexpr int kRefineThreads = 128;        // sweep_refine_kernel: 4 warps, one listed cell per warp at a time
constexpr int kMaxWarpTasks = 128;         // warp-tasks per tile (8 levels of at most tile/(256·g) each)
constexpr int kPadG = 16;                  // replicated entries after each decimated prefix array (window over-read)
#ifndef PULSCAN_SWEEP_DENSE_LANES
#define PULSCAN_SWEEP_DENSE_LANES 5   /* cfg 4, sweep+refine / kernel (c) ms: 8: 0.398/0.193, 5: 0.355/0.202, 4: 0.348/0.258, 3: 0.320/0.490 (noise cells marked) */
#endif
constexpr int kSweepDenseLanes = PULSCAN_SWEEP_DENSE_LANES;        // flagged lanes of a warp-task from which its blocks are marked without listing cells
constexpr float kSlackUlps = 96.f;         // ≥ 2·scan_roundings(NQ, passes) + 1, asserted in scan_tile
// Longest landing buffer a plan can ask for: a 16384-bin tile + halo of zmax ≤ 4096 and two groups of ≤ 128 bins, rounded to 64.
constexpr int kMaxSweepLen = 16384 + 4096 + 2 * 128 + 64;
// Roundings on the way from the float32 powers to one entry PG[k] = PP[k·g] of scan_tile, each of magnitude ≤ 2⁻²⁴·PP[len]
// (roundings of disjoint partial sums count once: each is relative to its own part of the total):
//   3       the quad sum (((a + b) + c) + d in the full-resolution scan; (a + b) + (c + d), formed by kernel (a) as a group sum
//           G or here, is 2)
//   NQ − 1  the thread's serial prefix over its quads
//   5       the warp's shuffle scan
//   1       excl = incl − s[NQ−1]
//   3       the butterfly sum of the totals of the warps below
//   2       off = carry + (wbase + excl)
//   1       s[q] += off
//   1       the full-resolution entries x[3q+t] += s[q−1]
//   2       per further pass: the carry, an entry of the pass before, goes through off and s[q] += off again
constexpr int scan_roundings(int nq, int passes) { return 3 + (nq - 1) + 5 + 1 + 3 + 2 + 1 + 1 + 2 * (passes - 1); }

struct SweepLevel {
    int lg;        // log2 of the group size g
    int wlo, whi;  // widths this level answers for
    int m_lo;      // smallest number of groups a cover of a width-wlo window has
    int m_hi;      // largest number of groups a cover of a width-whi window has
    int m_start;   // first cover length of the first step: ≡ 0 or 1 (mod 4), ≤ m_lo (the sliding window's vector loads start at
                   // m_start rounded down to a multiple of 4, and its 12 entries reach one length further, see sweep_step)
    int nsteps;    // 4-wide steps over m: m_start + 4·nsteps > m_hi; ≤ 32; τ = +inf below m_lo and above m_hi
    int tau_off;   // offset of τ[m_start ..] in the τ table (4·nsteps entries)
    int pg_off;    // offset (floats) of this level's decimated prefix array PG[k] = PP[k·g] in shared memory
    int nk;        // group starts per tile = tile / g
    int wt_off;    // first warp-task of this level; a warp-task is 32 lanes × 8 group starts
    int nwt;       // warp-tasks of this level
    // second look at a flagged cell with groups of half the size (sweep_refine_kernel, from the group sums); nmh = 0: none
    int tauh_off;  // offset of τ_h[mh − mh_start] in the τ table: thresholds of covers made of mh half-groups of g/2 bins
    int mh_start;  // first half-cover length in that table (= 2·m_start − 2, clamped at 0)
    int nmh;       // entries of that table
};

struct SweepParams {
    int nlevels;
    int tile;        // start bins per CTA
    int len;         // tile + halo, multiple of 64; halo ≥ zmax + 2·g_max
    int ntasks;      // warp-tasks per tile (levels are ordered by decreasing cost)
    int ntau;
    int zmax;
    int narr;        // decimated arrays: one per distinct group size
    int arr_lg[kMaxLevels];
    int arr_off[kMaxLevels];
    int off_lg[8];   // offset of the array with group size 2^lg, lg = 0..7; −1 if no level uses it
    int scan_nq;     // quads per thread per scan pass (5, 9 or 11: the kernel's NQ); a pass covers 4·NQ·256 bins
    int npass;       // scan passes per tile = ceil(len / (4·NQ·256)): 1 when NQ = 9 or 11
    int z_floats;    // floats of ONE landing buffer: len + kScanTail zeros (len/4 + kScanTail/4 for group-sum input)
    int smem_floats; // two landing buffers + decimated arrays
    int ref_span;    // longest span of bins a listed cell covers (sweep_refine_kernel's shared memory per warp)
    int tp_monotone; // T'_w is finite and non-decreasing in w (every width searched, exact significance)
    int dense_lanes; // flagged lanes of a warp-task from which its blocks are marked without listing cells; 33 = never
    SweepLevel lv[kMaxLevels];
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// Stage `bytes` (multiple of 16, 16-byte aligned both sides) global → shared with one TMA bulk copy and wait for it.
__device__ __forceinline__ void tma_load_1d(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* mbar) {
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(mbar)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(mbar)), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                         smem_u32(smem_dst)),
                     "l"(gmem_src), "r"(bytes), "r"(smem_u32(mbar))
                     : "memory");
    }
    uint32_t done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(mbar))
            : "memory");
    }
}

// Load P[row][t0 .. t0+len) into sP (zeros beyond n), through TMA when the addresses allow it.
__device__ __forceinline__ void load_tile(float* sP, const float* __restrict__ Prow, long long t0, long long n,
                                          long long pitchP, int len, uint64_t* mbar) {
    const long long avail = pitchP - t0;                       // floats left in the row's allocation
    const int ncopy = (int)(avail < (long long)len ? avail : (long long)len);
    const bool aligned = ((reinterpret_cast<uintptr_t>(Prow + t0) & 15) == 0) && ((ncopy & 3) == 0) && ncopy > 0;
    const long long nv = n - t0;                               // valid bins from t0
    const int first_pad = (int)(nv < 0 ? 0 : (nv < (long long)len ? nv : (long long)len));
    if (aligned) {
        tma_load_1d(sP, Prow + t0, (uint32_t)ncopy * 4u, mbar); // every thread returns after the bytes have landed
        for (int i = first_pad + threadIdx.x; i < len; i += blockDim.x) sP[i] = 0.f;
    } else {
        for (int i = threadIdx.x; i < len; i += blockDim.x) sP[i] = (i < first_pad) ? __ldg(Prow + t0 + i) : 0.f;
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------------------------------------------
// Quad-sum scan.  raw[i] = P[t0+i] for i < len and 0 for len ≤ i < len + kScanTail.  Each thread owns NQ consecutive quads
// (4·NQ powers; NQ odd: 16·NQ-byte lane stride = conflict-free 16-byte loads, 4·NQ bytes for group sums), so PP at the
// multiples of 4 it owns, PP[4(u+q)] with u = i0/4 + 1, q = 0..NQ−1, are its running quad sums plus the scanned offset,
// and the multiples of g among them follow a fixed pattern: the decimated arrays PG_lg[k] = PP[k << lg], k ∈ [0, len >> lg],
// lg ≥ 2, are written straight from registers.  NQ = 9 or 11 scans a whole tile + halo in ONE pass (≤ 9216 / 11264 bins:
// two CTA barriers per tile instead of four and no half-idle second pass); NQ = 5 takes as many passes as the tile needs.
// Entries past len >> lg (written by the thread that straddles len, inside the kPadG pad) equal PP[len] because of the
// zeros after len; the other pad entries only ever meet τ = +inf and are zeroed once per kernel.  After the first barrier
// of the last pass nobody reads `raw` any more (`after_loads` runs there: the next TMA copy into this buffer).  Returns
// PP[len] in every thread.  Ends with a CTA barrier; the barrier inside a pass also orders the previous tile's cover sums
// before this tile's writes to the arrays.
struct ScanSmem {
    alignas(16) float wtot[kSweepThreads / 32 + 4];   // warp totals; [8] = the running total carried into the next pass
};

// The entries of the decimated array PG_LG (PG[k] = PP[k << LG]) among a thread's prefix values s[q] = PP[4(u + q)]: those
// with u + q ≡ 0 (mod 2^(LG−2)), i.e. q = q0, q0 + M, … with q0 = −u mod M; each is picked from its M candidates by selects.
template <int LG, int NQ>
__device__ __forceinline__ void scan_put(float* __restrict__ dst, int u, const float (&s)[NQ]) {
    if constexpr (LG == 2) {
#pragma unroll
        for (int q = 0; q < NQ; ++q) dst[u + q] = s[q];
    } else {
        constexpr int sh = LG - 2, M = 1 << sh;
        const int q0 = (-u) & (M - 1);
        float* d = dst + ((u + q0) >> sh);
#pragma unroll
        for (int j = 0; j * M < NQ; ++j) {
            float v = s[j * M];
#pragma unroll
            for (int t = 1; t < M && j * M + t < NQ; ++t) v = (q0 == t) ? s[j * M + t] : v;
            if (j * M + M - 1 < NQ) d[j] = v;                    // every q0 lands inside the thread's run
            else if (j * M + q0 < NQ) d[j] = v;
        }
    }
}

// FINE = true additionally keeps the prefix inside each quad (x[3q+t] = the quad's first t+1 powers) and writes the arrays
// with g = 1 and g = 2 (PG0 = PP itself, PG1): needed when a level's covers must be finer than 4 bins — harmonic-summed
// spectra, whose noise level per bin is H(H+1)/2, and very low σ thresholds.
// FROMG = true: `raw` holds the tile's group sums G[k] = P[4k] + … + P[4k+3] (written by kernel (a), norm_power.cuh)
// instead of the powers: a thread's NQ quad sums are NQ loads.
template <bool FINE, bool FROMG, int NQ, class AfterLoads>
__device__ __forceinline__ float scan_tile(const SweepParams& sp, const float* raw, float* sG, ScanSmem& ss,
                                           AfterLoads after_loads) {
    static_assert(!(FINE && FROMG), "levels finer than four bins need the powers themselves");
    static_assert(NQ % 2 == 1 && NQ <= kScanTail / 4, "odd lane stride; zeros after the landing buffer");
    constexpr int kPer = 4 * NQ, kPass = kPer * kSweepThreads;
    static_assert(2 * scan_roundings(NQ, (kMaxSweepLen + kPass - 1) / kPass) + 1 <= (int)kSlackUlps,
                  "the cover test's slack no longer bounds the scan's rounding error: raise kSlackUlps or scan fewer quads per thread");
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int len = sp.len;
    float carry = 0.f;
    for (int pass = 0; pass < sp.npass; ++pass) {
        const int i0 = pass * kPass + kPer * tid;
        const bool act = i0 < len;
        float s[NQ];
        float x[FINE ? 3 * NQ : 1];
        if (act && FROMG) {
            const float* gq = raw + (i0 >> 2);
#pragma unroll
            for (int q = 0; q < NQ; ++q) s[q] = gq[q];
#pragma unroll
            for (int q = 1; q < NQ; ++q) s[q] += s[q - 1];
        } else if (act) {
            const float4* zq = reinterpret_cast<const float4*>(raw) + (i0 >> 2);
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                const float4 v = zq[q];
                if (FINE) {
                    x[3 * q] = v.x; x[3 * q + 1] = v.x + v.y; x[3 * q + 2] = x[3 * q + 1] + v.z;
                    s[q] = x[3 * q + 2] + v.w;
                } else {
                    s[q] = (v.x + v.y) + (v.z + v.w);
                }
            }
#pragma unroll
            for (int q = 1; q < NQ; ++q) s[q] += s[q - 1];
        } else {
#pragma unroll
            for (int q = 0; q < NQ; ++q) s[q] = 0.f;
        }
        float incl = s[NQ - 1];
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const float t = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += t;
        }
        const float excl = incl - s[NQ - 1];
        if (lane == 31) ss.wtot[warp] = incl;
        __syncthreads();
        if (pass == sp.npass - 1) after_loads();
        // sum of the totals of the warps below this one: lane w < 8 holds total w, masked, three butterfly steps
        float wbase = (lane < warp) ? ss.wtot[lane & (kSweepThreads / 32 - 1)] : 0.f;
#pragma unroll
        for (int off = 4; off > 0; off >>= 1) wbase += __shfl_xor_sync(0xffffffffu, wbase, off);
        wbase = __shfl_sync(0xffffffffu, wbase, 0);
        if (act) {
            const float off = carry + (wbase + excl);
#pragma unroll
            for (int q = 0; q < NQ; ++q) s[q] += off;           // s[q] = PP[4(u+q)]
            const int u = (i0 >> 2) + 1;
            if (FINE) {                                         // x[3q+t] = PP[i0 + 4q + t + 1], t = 0..2
#pragma unroll
                for (int q = 0; q < NQ; ++q) {
                    const float oq = q ? s[q - 1] : off;
                    x[3 * q] += oq; x[3 * q + 1] += oq; x[3 * q + 2] += oq;
                }
                if (sp.off_lg[0] >= 0) {                        // PG0[i] = PP[i]: entries i0+1 … i0+4·NQ (the pad holds 16)
                    float* dst = sG + sp.off_lg[0];
#pragma unroll
                    for (int q = 0; q < NQ; ++q) {
                        float* d = dst + i0 + 4 * q + 1;
                        if (i0 + 4 * q + 4 <= len + kPadG) { d[0] = x[3 * q]; d[1] = x[3 * q + 1]; d[2] = x[3 * q + 2]; d[3] = s[q]; }
                    }
                }
                if (sp.off_lg[1] >= 0) {                        // PG1[k] = PP[2k]: entries i0/2+1 … i0/2+2·NQ
                    float* dst = sG + sp.off_lg[1];
#pragma unroll
                    for (int q = 0; q < NQ; ++q) { dst[(i0 >> 1) + 2 * q + 1] = x[3 * q + 1]; dst[(i0 >> 1) + 2 * q + 2] = s[q]; }
                }
            }
            // one store sequence per group size, the group size a compile-time constant in each (the branches are uniform)
            if (sp.off_lg[2] >= 0) scan_put<2, NQ>(sG + sp.off_lg[2], u, s);
            if (sp.off_lg[3] >= 0) scan_put<3, NQ>(sG + sp.off_lg[3], u, s);
            if (sp.off_lg[4] >= 0) scan_put<4, NQ>(sG + sp.off_lg[4], u, s);
            if (sp.off_lg[5] >= 0) scan_put<5, NQ>(sG + sp.off_lg[5], u, s);
            if (sp.off_lg[6] >= 0) scan_put<6, NQ>(sG + sp.off_lg[6], u, s);
            if (sp.off_lg[7] >= 0) scan_put<7, NQ>(sG + sp.off_lg[7], u, s);
        }
        // PP at the end of this pass = the last thread's running total: the carry of the next pass and, after the last pass,
        // PP[len] (the bound of every entry, which the caller's slack is scaled by)
        if (tid == kSweepThreads - 1) ss.wtot[kSweepThreads / 32] = act ? s[NQ - 1] : carry + (wbase + excl);
        __syncthreads();
        carry = ss.wtot[kSweepThreads / 32];
    }
    return carry;
}

// One 4-wide step over m for 8 group starts.  O is the rotation of the 12-entry window W (compile time, so that the window
// never moves between registers): W[(O + j) % 12] = PG[k0b + m_base + 4·step + j], j = 0..11 after the load below, where
// m_base = m_start − D is a multiple of 4 (16-byte alignment of the vector loads) and D ∈ {0, 1}: the step's cover lengths
// are m_start + 4·step + q, q = 0..3, whose ends are the entries D + q + r ≤ 11.  D = 1 lets a level start at m ≡ 1 (mod 4)
// without a dead cover length: the levels with 4-bin groups start at m = 1 and are the most expensive per step.
template <int O, int D>
__device__ __forceinline__ bool sweep_step(const float (&A)[kSweepR], float (&W)[12], const float* __restrict__ pg_next,
                                           const float* __restrict__ tau4) {
    const float4 nw = *reinterpret_cast<const float4*>(pg_next);
    W[(O + 8) % 12] = nw.x; W[(O + 9) % 12] = nw.y; W[(O + 10) % 12] = nw.z; W[(O + 11) % 12] = nw.w;
    const float4 t = *reinterpret_cast<const float4*>(tau4);
    const float tq[4] = {t.x, t.y, t.z, t.w};
    bool hit = false;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        float u[kSweepR];
#pragma unroll
        for (int r = 0; r < kSweepR; ++r) u[r] = W[(O + D + q + r) % 12] - A[r];
        const float m0 = fmaxf(fmaxf(u[0], u[1]), u[2]);
        const float m1 = fmaxf(fmaxf(u[3], u[4]), u[5]);
        const float m2 = fmaxf(fmaxf(u[6], u[7]), m0);
        hit = hit || (fmaxf(m1, m2) >= tq[q]);
    }
    return hit;
}

// All covers of one level for 8 consecutive group starts k0b..k0b+7: returns the bit mask of the 4-wide m steps in
// which some cover reached its threshold (slack already folded into A).
template <int D>
__device__ __forceinline__ unsigned sweep_task_d(const float* __restrict__ PG, int k0b, int m_base, int nsteps,
                                                 const float* __restrict__ tau, float slack) {
    float A[kSweepR], W[12];
    {
        const float4 a0 = *reinterpret_cast<const float4*>(PG + k0b);
        const float4 a1 = *reinterpret_cast<const float4*>(PG + k0b + 4);
        A[0] = a0.x - slack; A[1] = a0.y - slack; A[2] = a0.z - slack; A[3] = a0.w - slack;
        A[4] = a1.x - slack; A[5] = a1.y - slack; A[6] = a1.z - slack; A[7] = a1.w - slack;
        const float* p = PG + k0b + m_base;
        const float4 w0 = *reinterpret_cast<const float4*>(p);
        const float4 w1 = *reinterpret_cast<const float4*>(p + 4);
        W[0] = w0.x; W[1] = w0.y; W[2] = w0.z; W[3] = w0.w; W[4] = w1.x; W[5] = w1.y; W[6] = w1.z; W[7] = w1.w;
        W[8] = W[9] = W[10] = W[11] = 0.f;
    }
    unsigned mask = 0;
    const float* p = PG + k0b + m_base + 8;
    for (int s = 0; s < nsteps; s += 3) {
        if (sweep_step<0, D>(A, W, p, tau)) mask |= 1u << s;
        if (s + 1 < nsteps && sweep_step<4, D>(A, W, p + 4, tau + 4)) mask |= 2u << s;
        if (s + 2 < nsteps && sweep_step<8, D>(A, W, p + 8, tau + 8)) mask |= 4u << s;
        p += 12; tau += 12;
    }
    return mask;
}

__device__ __forceinline__ unsigned sweep_task(const float* __restrict__ PG, int k0b, int m_start, int nsteps,
                                               const float* __restrict__ tau, float slack) {
    return (m_start & 1) ? sweep_task_d<1>(PG, k0b, m_start - 1, nsteps, tau, slack)     // warp-uniform
                         : sweep_task_d<0>(PG, k0b, m_start, nsteps, tau, slack);
}

// Second look at a flagged cell before it is listed, by the whole warp (lane = 8·q + r looks at cover length m4 + q from group
// start k0b + r: the refine kernel's layout, and the same test as its look from the group sums, here on the tile's float32
// prefix arrays with the slack on the keeping side).  A window that reaches its T_w is covered by m groups of g bins and by
// mh = 2m − 1 + b − a half-groups of g/2 bins (start in half a of the first group, end in half b of the last); the half-cover
// is only g − 2 bins longer than its narrowest window, so its threshold τ_h[mh] rejects most of the noise flags that live off
// the 2g − 2 bins of slack of the full cover (cfg 3: 9 of 10 cells).  Needs the array PG_{lg−1} in shared memory (a level of
// that group size exists) and the level's τ_h table; otherwise the cell is kept.  Returns the same value in every lane.
__device__ __forceinline__ bool sweep_confirm_cell(const SweepParams& sp, const SweepLevel& lv, const float* __restrict__ sG,
                                                   const float* __restrict__ sTau, int k0b, int st, float slack) {
    if (lv.lg < 3 || lv.nmh <= 0) return true;
    const int offh = sp.off_lg[lv.lg - 1];
    if (offh < 0) return true;
    const int lane = threadIdx.x & 31;
    const float* PG = sG + lv.pg_off;
    const float* PH = sG + offh;
    const int q = lane >> 3, k = k0b + (lane & 7), m = lv.m_start + 4 * st + q;
    bool ok = false;
    if (PG[k + m] - (PG[k] - slack) >= sTau[lv.tau_off + 4 * st + q]) {
#pragma unroll
        for (int ab = 0; ab < 4; ++ab) {
            const int ha = ab & 1, hb = ab >> 1;
            const int mh = 2 * m - 1 + hb - ha, tt = mh - lv.mh_start;
            if (mh < 1 || tt < 0 || tt >= lv.nmh) continue;
            const int h0 = 2 * k + ha;
            if (PH[h0 + mh] - (PH[h0] - slack) >= sTau[lv.tauh_off + tt]) ok = true;
        }
    }
    return __any_sync(0xffffffffu, ok);
}

// Append the tile's marked candidate blocks to the global list, once each (bitmap test-and-set).
__device__ __forceinline__ void publish_flags(const unsigned char* sflag, int nblk_tile, long long c_first, long long nblk,
                                              long long row, unsigned* __restrict__ bitmap,
                                              unsigned* __restrict__ flagged, unsigned* __restrict__ counters) {
    for (int cb = threadIdx.x; cb < nblk_tile; cb += blockDim.x) {
        if (!sflag[cb]) continue;
        const long long c = c_first + cb;
        if (c >= nblk) continue;
        const unsigned long long gid = (unsigned long long)(row * nblk + c);
        const unsigned bit = 1u << (gid & 31);
        const unsigned old = atomicOr(bitmap + (gid >> 5), bit);
        if (!(old & bit)) flagged[atomicAdd(counters, 1u)] = (unsigned)gid;
    }
}

// A warp-task: the covers of one level for 32 × 8 consecutive group starts.  The list is the same for every tile, so it
// is built once per CTA; warp w runs tasks w, w + 8, … of every tile.
struct alignas(16) WarpTask {
    int pg_off, tau_off, m_start, nsteps;
    int level, kbase, nk, pad_;
};

// A flagged cell: tile `item` (= row·tiles_per_row + tile index), level, 4-wide step over m, first of 8 group starts.
struct SweepCell {
    unsigned item;
    unsigned code;   // level << 28 | step << 20 | (k0b >> 3)
};

struct SweepCtl {
    ScanSmem scan;
    alignas(8) uint64_t mbar[kSweepBufs];
    WarpTask task[kMaxWarpTasks];
};

// Mark candidate block gid = row·nblk + c once (bitmap test-and-set) and append it to the list kernel (c) works from.
__device__ __forceinline__ void mark_block(unsigned long long gid, unsigned* __restrict__ bitmap,
                                           unsigned* __restrict__ flagged, unsigned* __restrict__ counters) {
    const unsigned bit = 1u << (gid & 31);
    if (bitmap[gid >> 5] & bit) return;
    const unsigned old = atomicOr(bitmap + (gid >> 5), bit);
    if (!(old & bit)) flagged[atomicAdd(counters, 1u)] = (unsigned)gid;
}

// Thread 0: start the TMA copy of tile `item` into `dst`.  The copy is clipped to the row's allocation (pitchP), so it
// never touches the next spectrum (R11); P rows start 16-byte aligned and pitchP, tile and len are multiples of 4, so the
// copy always satisfies TMA's alignment rules.
template <bool FROMG>
__device__ __forceinline__ void sweep_issue_tile(const SweepParams& sp, long long item, const float* __restrict__ P,
                                                 long long pitchP, int tiles_per_row, float* dst, uint64_t* mbar) {
    const long long row = item / tiles_per_row;
    const long long t0 = ((item - row * tiles_per_row) * sp.tile) >> (FROMG ? 2 : 0);   // in elements of the input array
    const long long want = sp.len >> (FROMG ? 2 : 0);
    const long long avail = pitchP - t0;
    const uint32_t bytes = (uint32_t)(avail < want ? avail : want) * 4u;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");    // the buffer's earlier generic accesses precede the copy
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(mbar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(P + row * pitchP + t0), "r"(bytes), "r"(smem_u32(mbar))
                 : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t* mbar, uint32_t parity) {
    uint32_t done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(mbar)), "r"(parity)
            : "memory");
    }
}

// Streaming filter, persistent: gridDim.x CTAs (a multiple of the SM count) stride over the n_items = tiles_per_row ·
// batch tiles.  Two landing buffers: a tile's copy is issued as soon as the previous user of its buffer has read its
// powers into registers, i.e. a whole tile ahead.  Two CTA barriers per tile (both inside the scan).
// counters[2] = cells appended (the refine kernel's work count), counters[9] = cells flagged before the second look,
// counters[10] = flagged lanes whose blocks were marked directly (dense warp-tasks),
// (sweep_confirm_cell), counters[3] = cells dropped because the list was full
// (their tile's blocks are all marked instead, which is always allowed: kernel (c) decides).
// Dynamic shared memory: [kSweepBufs × z_floats landing buffers][decimated arrays][ntau τ][SweepCtl].
// FROMG = true: P / pitchP are the group-sum array G and its pitch (see scan_tile).
template <bool FINE, bool FROMG, int NQ>
__global__ void __launch_bounds__(kSweepThreads, PULSCAN_SWEEP_OCC)
boxcar_sweep_kernel(const __grid_constant__ SweepParams sp, const float* __restrict__ P, long long pitchP, long long n,
                    int tiles_per_row, long long n_items, int C, long long nblk, const float* __restrict__ tau_g,
                    SweepCell* __restrict__ cells, unsigned cell_cap, unsigned* __restrict__ bitmap,
                    unsigned* __restrict__ flagged, unsigned* __restrict__ counters) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* raw0 = reinterpret_cast<float*>(smem_raw);
    float* sG = raw0 + kSweepBufs * sp.z_floats;
    float* sTau = raw0 + sp.smem_floats;
    SweepCtl& ctl = *reinterpret_cast<SweepCtl*>(sTau + ((sp.ntau + 3) & ~3));
    const int tid = threadIdx.x, lane = tid & 31;
    const long long stride = gridDim.x;

    // ---- once per CTA: τ table, zeros after len and in the arrays (PG[0] = 0, pads), task list, the first two copies
    for (int i = tid; i < sp.ntau; i += kSweepThreads) sTau[i] = tau_g[i];
    for (int i = tid; i < sp.smem_floats - kSweepBufs * sp.z_floats; i += kSweepThreads) sG[i] = 0.f;
    {   // zeros after the copied elements (a thread's run of quads may start before and end after them)
        const int first = FROMG ? (sp.len >> 2) : sp.len, ntail = sp.z_floats - first;
        for (int i = tid; i < kSweepBufs * ntail; i += kSweepThreads) raw0[(i / ntail) * sp.z_floats + first + i % ntail] = 0.f;
    }
    for (int q = tid; q < sp.ntasks; q += kSweepThreads) {
        int L = 0;
        while (L + 1 < sp.nlevels && q >= sp.lv[L + 1].wt_off) ++L;
        const SweepLevel& lv = sp.lv[L];
        ctl.task[q] = WarpTask{lv.pg_off, lv.tau_off, lv.m_start, lv.nsteps, L, (q - lv.wt_off) * 32 * kSweepR, lv.nk, 0};
    }
    if (tid == 0) {
        for (int b = 0; b < kSweepBufs; ++b) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&ctl.mbar[b])));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        const long long i0 = blockIdx.x;
        for (int b = 0; b < kSweepBufs; ++b)
            if (i0 + b * stride < n_items)
                sweep_issue_tile<FROMG>(sp, i0 + b * stride, P, pitchP, tiles_per_row, raw0 + b * sp.z_floats, &ctl.mbar[b]);
    }

    // (row, tile index) of the current item, advanced without divisions
    long long row = blockIdx.x / tiles_per_row;
    int tix = (int)(blockIdx.x - row * tiles_per_row);
    const long long drow = stride / tiles_per_row;
    const int dtix = (int)(stride - drow * tiles_per_row);

    int it = 0;
    for (long long item = blockIdx.x; item < n_items; item += stride, ++it) {
        const int b = it % kSweepBufs;
        float* raw = raw0 + b * sp.z_floats;
        mbar_wait(&ctl.mbar[b], (uint32_t)(it / kSweepBufs) & 1u);
        const long long nv = n - (long long)tix * sp.tile;      // valid bins from the tile's first one
        if (nv < (long long)sp.len) {                            // last tile of a row: nothing beyond the spectrum's end
            // (group sums: the group holding the last bin is kept, kernel (a) added zeros for its missing bins)
            const int first = FROMG ? (int)((nv + 3) >> 2) : (int)nv, end = FROMG ? (sp.len >> 2) : sp.len;
            for (int i = first + tid; i < end; i += kSweepThreads) raw[i] = 0.f;
            __syncthreads();
        }
        const float pp_max = scan_tile<FINE, FROMG, NQ>(sp, raw, sG, ctl.scan, [&] {
            const long long nxt = item + kSweepBufs * stride;
            if (tid == 0 && nxt < n_items) sweep_issue_tile<FROMG>(sp, nxt, P, pitchP, tiles_per_row, raw, &ctl.mbar[b]);
        });
        const float slack = kSlackUlps * 5.9604644775390625e-8f * pp_max;

        // ---- cover sums: warp-tasks dealt round-robin, most expensive levels first
        for (int q = tid >> 5; q < sp.ntasks; q += kSweepThreads / 32) {
            const int4 ta = *reinterpret_cast<const int4*>(&ctl.task[q]);            // pg_off, tau_off, m_start, nsteps
            const int4 tb = *reinterpret_cast<const int4*>(&ctl.task[q].level);      // level, kbase, nk
            const int k0b = tb.y + lane * kSweepR;
            const unsigned mask = (k0b < tb.z) ? sweep_task(sG + ta.x, k0b, ta.z, ta.w, sTau + ta.y, slack) : 0u;
            unsigned lanes = __ballot_sync(0xffffffffu, mask != 0u);     // rare: 1.3 cells per tile in noise
            // Many flagged lanes in one warp-task are a strong signal, not noise: every flagged lane marks the candidate blocks
            // that own its 8·g start bins straight away (always allowed: kernel (c) decides) instead of the warp walking
            // through hundreds of cells one at a time while the rest of its CTA waits at the next barrier.
            if (lanes == 0u) continue;
            if (__popc(lanes) >= sp.dense_lanes && ((kSweepR << sp.lv[tb.x].lg) <= 16 * C)) {
                if (mask != 0u) {
                    const long long t0 = (long long)tix * sp.tile + ((long long)k0b << sp.lv[tb.x].lg);
                    const long long last = min(t0 + (kSweepR << sp.lv[tb.x].lg) - 1, n - 1);
                    for (long long c = t0 / C; c <= last / C; ++c) mark_block((unsigned long long)(row * nblk + c), bitmap, flagged, counters);
                }
                if (lane == 0) atomicAdd(counters + 10, (unsigned)__popc(lanes));
                continue;
            }
            while (lanes) {
                const int src = __ffs(lanes) - 1;
                lanes &= lanes - 1;
                unsigned ms = __shfl_sync(0xffffffffu, mask, src);
                const int kc = tb.y + src * kSweepR;
                while (ms) {
                    const int st = __ffs(ms) - 1;
                    ms &= ms - 1;
                    const bool keep = sweep_confirm_cell(sp, sp.lv[tb.x], sG, sTau, kc, st, slack);
                    if (lane == 0) {
                        atomicAdd(counters + 9, 1u);             // cells flagged by the cover sums, before the second look
                        const unsigned pos = keep ? atomicAdd(counters + 2, 1u) : 0u;
                        if (keep && pos < cell_cap) {
                            cells[pos] = SweepCell{(unsigned)item, ((unsigned)tb.x << 28) | ((unsigned)st << 20) | (unsigned)(kc >> 3)};
                        } else if (keep) {                       // list full: mark every block the tile's start bins touch
                            atomicAdd(counters + 3, 1u);
                            const long long t0 = (long long)tix * sp.tile;
                            const long long last = min(t0 + sp.tile - 1, n - 1);
                            for (long long c = t0 / C; c <= last / C; ++c) mark_block((unsigned long long)(row * nblk + c), bitmap, flagged, counters);
                        }
                    }
                }
            }
        }
        row += drow; tix += dtix;
        if (tix >= tiles_per_row) { tix -= tiles_per_row; ++row; }
    }
}

// Rare path: one warp per listed cell.  The cell covers group starts k0b..k0b+7 and cover lengths m4..m4+3 of its
// level, i.e. the bins [k0b·g, (k0b + m4 + 10)·g) of its tile; their prefix sum is rebuilt in double from P, the 32
// covers are re-tested against τ and the windows inside each passing cover (start in its first group, end in its last)
// are summed and compared with T'_w.  A window that passes marks the candidate block of its start bin.
// Dynamic shared memory: (kRefineThreads/32) × (ref_span + 1) doubles.
__global__ void __launch_bounds__(kRefineThreads)
sweep_refine_kernel(const __grid_constant__ SweepParams sp, const PowerSource src_pw, const float* __restrict__ G,
                    long long pitchG, long long n, int tiles_per_row, int C, long long nblk, const float* __restrict__ tau_g,
                    const float* __restrict__ Tp_g, const SweepCell* __restrict__ cells, unsigned cell_cap,
                    unsigned* __restrict__ bitmap, unsigned* __restrict__ flagged, unsigned* __restrict__ counters) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* pp = reinterpret_cast<double*>(smem_raw) + (size_t)warp * (sp.ref_span + 1);
    const unsigned ncell = min(counters[2], cell_cap);
    const unsigned nwarps = gridDim.x * (kRefineThreads / 32);
    for (unsigned e = blockIdx.x * (kRefineThreads / 32) + warp; e < ncell; e += nwarps) {
        const SweepCell cell = cells[e];
        const SweepLevel& lv = sp.lv[cell.code >> 28];
        const int step = (int)((cell.code >> 20) & 0xFFu), k0b = (int)(cell.code & 0xFFFFFu) << 3;
        const int lg = lv.lg, g = 1 << lg, m4 = lv.m_start + 4 * step;
        const long long row = cell.item / (unsigned)tiles_per_row;
        const long long base = (long long)(cell.item - (unsigned)(row * tiles_per_row)) * sp.tile + ((long long)k0b << lg);
        const int span = (m4 + 10) << lg;                        // ≤ ref_span
        const long long room = n - base;
        const int valid = (int)(room < (long long)span ? (room < 0 ? 0 : room) : (long long)span);
        // Nothing left to find if every candidate block that owns a start bin of this cell is already marked (a strong
        // signal flags many cells over the same few blocks; kernel (c) evaluates a marked block completely anyway).
        {
            const long long s_last = min(base + (8ll << lg), n) - 1;          // last start bin of the cell
            const long long c0 = base / C, c1 = s_last / C;
            if (s_last >= base && c1 - c0 < 32) {
                bool marked = true;
                if (c0 + lane <= c1) {
                    const unsigned long long gid = (unsigned long long)(row * nblk + c0 + lane);
                    marked = (__ldcg(bitmap + (gid >> 5)) >> (gid & 31)) & 1u;
                }
                if (__all_sync(0xffffffffu, marked)) continue;
            }
        }
        // ---- Second look, from the group sums (1 B/bin, no rebuild).  A cover of m groups of g bins is 2g − 2 bins longer than
        // the narrowest window it answers for, and most noise flags live off that slack.  The same window is also covered by
        // half-groups of g/2 bins — starts in half a of the first group, ends in half b of the last, mh = 2m − 1 + b − a
        // half-groups — and that cover is only g − 2 bins longer than its narrowest window: the four half-covers of every
        // passing cover are tested against their own thresholds τ_h[mh] (the lowest T'_w among the level's searched widths
        // (mh − 2)·g/2 + 2 … mh·g/2, rounded down like τ).  A window that reaches its T_w passes its half-cover for the same
        // reason it passes its cover (P ≥ 0; the group sums are float32 sums of four powers, 2·2⁻²⁴ relative, inside τ_h's
        // margin), so a cell without a passing half-cover holds nothing.  Needs g ≥ 8 (half-groups are whole group sums).
        if (G != nullptr && lg >= 3 && lv.nmh > 0) {
            const float* gsrc = G + row * pitchG + (base >> 2);
            const int nq = span >> 2, vq = (valid + 3) >> 2;
            for (int j = lane; j < nq; j += 32) pp[j + 1] = (j < vq) ? (double)__ldg(gsrc + j) : 0.0;
            if (lane == 0) pp[0] = 0.0;
            __syncwarp();
            {
                const int Lq = (nq + 31) >> 5;
                const int q0 = min(lane * Lq, nq), q1 = min(q0 + Lq, nq);
                double run = 0.0;
                for (int j = q0; j < q1; ++j) { run += pp[j + 1]; pp[j + 1] = run; }
                double incl = run;
#pragma unroll
                for (int off = 1; off < 32; off <<= 1) {
                    const double t = __shfl_up_sync(0xffffffffu, incl, off);
                    if (lane >= off) incl += t;
                }
                const double excl = incl - run;
                for (int j = q0; j < q1; ++j) pp[j + 1] += excl;
            }
            __syncwarp();
            const int r = lane & 7, m = m4 + (lane >> 3), lq = lg - 2, lhq = lg - 3;   // group / half-group size in quads: 2^lq, 2^lhq
            bool confirmed = false;
            if (pp[(r + m) << lq] - pp[r << lq] >= (double)__ldg(tau_g + lv.tau_off + 4 * step + (lane >> 3)) * (1.0 - 1e-6)) {
#pragma unroll
                for (int ab = 0; ab < 4; ++ab) {
                    const int ha = ab & 1, hb = ab >> 1;
                    const int mh = 2 * m - 1 + hb - ha, t = mh - lv.mh_start;
                    if (mh < 1 || t < 0 || t >= lv.nmh) continue;
                    const int h0 = 2 * r + ha;
                    if (pp[(h0 + mh) << lhq] - pp[h0 << lhq] >= (double)__ldg(tau_g + lv.tauh_off + t) * (1.0 - 1e-6)) confirmed = true;
                }
            }
            unsigned live = __ballot_sync(0xffffffffu, confirmed);
            // Third look, wide groups only: the 4 × 4 sub-covers (g/4 starts × g/4 ends, whole group sums for g ≥ 16) of every cover
            // that passed, against the threshold of their narrowest searched width — the test the rebuilt span would meet
            // further down, taken here from the group sums so that a cell of noise is dropped before ≈ (m + 10)·g bins of
            // the input spectrum are read and normalised for it.
            if (live && lg >= 4 && sp.tp_monotone) {
                const int lh = lg - 2, h = 1 << lh, sa = lane & 3, sb = (lane >> 2) & 3;
                unsigned todo = live;
                live = 0u;
                while (todo) {
                    const int srcl = __ffs(todo) - 1;
                    todo &= todo - 1;
                    const int rr = srcl & 7, mm = m4 + (srcl >> 3);
                    const int i0 = rr << lg, e0 = (rr + mm - 1) << lg;
                    const int fs = i0 + (sa << lh), le1 = min(e0 + ((sb + 1) << lh), valid);          // first start, one past the last end
                    const int w_lo = max((e0 + (sb << lh)) - (fs + h - 1) + 1, max(lv.wlo, 1)), w_hi = min(le1 - fs, lv.whi);
                    const bool sub = lane < 16 && w_lo <= w_hi &&
                                     pp[(le1 + 3) >> 2] - pp[fs >> 2] >= (double)__ldg(Tp_g + (w_lo - 1)) * (1.0 - 1e-6);
                    if (__any_sync(0xffffffffu, sub)) { live = 1u; break; }
                }
            }
            __syncwarp();
            if (!live) continue;
        }
        PowerSource::Row src(src_pw, row);
        // ---- prefix sum in double: stage the span (coalesced loads, several in flight), then each lane scans its own
        //      chunk of L consecutive bins and the chunk totals are scanned across the warp
        for (int j = lane; j < span; j += 32) pp[j + 1] = (j < valid) ? (double)src(base + j) : 0.0;
        if (lane == 0) pp[0] = 0.0;
        __syncwarp();
        const int L = (span + 31) >> 5;
        const int c0 = min(lane * L, span), c1 = min(c0 + L, span);
        double run = 0.0;
        for (int j = c0; j < c1; ++j) { run += pp[j + 1]; pp[j + 1] = run; }
        double incl = run;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const double t = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += t;
        }
        const double excl = incl - run;
        for (int j = c0; j < c1; ++j) pp[j + 1] += excl;
        __syncwarp();
        // ---- re-test the 32 covers (lane = 8·(m − m4) + (k0 − k0b)), then the windows of those that pass
        const int r = lane & 7, m = m4 + (lane >> 3);
        const bool live = pp[(r + m) << lg] - pp[r << lg] >= (double)__ldg(tau_g + lv.tau_off + 4 * step + (lane >> 3)) * (1.0 - 1e-6);
        unsigned hits = __ballot_sync(0xffffffffu, live);
        while (hits) {
            const int srcl = __ffs(hits) - 1;
            hits &= hits - 1;
            const int rr = srcl & 7, mm = m4 + (srcl >> 3);
            const int i0 = rr << lg, e0 = (rr + mm - 1) << lg;
            if (g <= C) {   // nothing left to find if the (one or two) blocks owning the cover's start bins are already marked
                const unsigned long long ga = (unsigned long long)(row * nblk + (base + i0) / C);
                const unsigned long long gb = (unsigned long long)(row * nblk + min(base + i0 + g - 1, n - 1) / C);
                const unsigned wa = __ldcg(bitmap + (ga >> 5)), wb = __ldcg(bitmap + (gb >> 5));
                if ((wa >> (ga & 31) & 1u) && (wb >> (gb & 31) & 1u)) continue;
            }
            if (g >= 8 && g <= C) {   // 32 windows spread over the cover first: a real signal passes here and marks its block(s)
                const int i = i0 + ((lane << lg) >> 5), ee = e0 + ((((lane * 11) & 31) << lg) >> 5);
                const int w = ee - i + 1;
                if (w >= 1 && w >= lv.wlo && w <= lv.whi && ee < valid && pp[ee + 1] - pp[i] >= (double)__ldg(Tp_g + (w - 1)))
                    mark_block((unsigned long long)(row * nblk + (base + i) / C), bitmap, flagged, counters);
                __syncwarp();
                const unsigned long long ga = (unsigned long long)(row * nblk + (base + i0) / C);
                const unsigned long long gb = (unsigned long long)(row * nblk + min(base + i0 + g - 1, n - 1) / C);
                const unsigned wa = __ldcg(bitmap + (ga >> 5)), wb = __ldcg(bitmap + (gb >> 5));
                if ((wa >> (ga & 31) & 1u) && (wb >> (gb & 31) & 1u)) continue;
            }
            if (lg >= 4 && sp.tp_monotone) {
                // Wide groups: cut the cover's g × g (start, end) pairs into 4 × 4 sub-covers of h = g/4 starts and ends.  The
                // sum from a sub-cover's first start to its last end bounds all its windows, and (T'_w non-decreasing in w)
                // the threshold of its narrowest searched width bounds theirs from below: only sub-covers that pass that test
                // (a few in noise) have their h² windows summed.
                const int lh = lg - 2, h = 1 << lh, sa = lane & 3, sb = (lane >> 2) & 3;
                const int fs = i0 + (sa << lh), le = min(e0 + ((sb + 1) << lh) - 1, valid - 1);   // first start, last (valid) end
                const int w_lo = max((e0 + (sb << lh)) - (fs + h - 1) + 1, max(lv.wlo, 1)), w_hi = min(le - fs + 1, lv.whi);
                const bool sub_live = lane < 16 && w_lo <= w_hi && pp[le + 1] - pp[fs] >= (double)__ldg(Tp_g + (w_lo - 1));
                unsigned subs = __ballot_sync(0xffffffffu, sub_live);
                while (subs) {
                    const int sl = __ffs(subs) - 1;
                    subs &= subs - 1;
                    const int is = i0 + ((sl & 3) << lh), es = e0 + (((sl >> 2) & 3) << lh);
                    for (int idx = lane; idx < h * h; idx += 32) {
                        const int i = is + (idx >> lh), ee = es + (idx & (h - 1));
                        const int w = ee - i + 1;
                        if (w < 1 || w < lv.wlo || w > lv.whi || ee >= valid) continue;
                        if (pp[ee + 1] - pp[i] >= (double)__ldg(Tp_g + (w - 1)))
                            mark_block((unsigned long long)(row * nblk + (base + i) / C), bitmap, flagged, counters);
                    }
                }
                continue;
            }
            for (int idx = lane; idx < g * g; idx += 32) {
                const int i = i0 + (idx >> lg), ee = e0 + (idx & (g - 1));
                const int w = ee - i + 1;
                if (w < 1 || w < lv.wlo || w > lv.whi || ee >= valid) continue;
                if (pp[ee + 1] - pp[i] >= (double)__ldg(Tp_g + (w - 1)))
                    mark_block((unsigned long long)(row * nblk + (base + i) / C), bitmap, flagged, counters);
            }
        }
        __syncwarp();
    }
}

// Exhaustive sweep (cross-check mode): thread per start bin, the paper's recursion S(i,w) = S(i,w−1) + P[i+w−1]
// over every width, compared with T'_w.  Same outputs as the pruned kernel.  Dynamic shared memory:
//   [len floats][zmax T'][mbarrier][nblk_tile flag bytes].
__global__ void __launch_bounds__(kSweepThreads)
boxcar_exhaustive_kernel(int tile, int len, int zmax, const float* __restrict__ P, long long pitchP, long long n,
                         int tiles_per_row, int C, long long nblk, const float* __restrict__ Tp_g,
                         unsigned* __restrict__ bitmap, unsigned* __restrict__ flagged,
                         unsigned* __restrict__ counters) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* sP = reinterpret_cast<float*>(smem_raw);
    float* sT = sP + len;
    uint64_t* mbar = reinterpret_cast<uint64_t*>(sT + ((zmax + 3) & ~3));
    unsigned char* sflag = reinterpret_cast<unsigned char*>(mbar + 2);

    const int tid = threadIdx.x;
    const long long row = blockIdx.x / tiles_per_row;
    const long long t0 = (long long)(blockIdx.x % tiles_per_row) * tile;
    const long long c_first = t0 / C;
    long long last_start = t0 + tile - 1;
    if (last_start > n - 1) last_start = n - 1;
    const int nblk_tile = (int)(last_start / C - c_first) + 1;

    for (int i = tid; i < zmax; i += kSweepThreads) sT[i] = Tp_g[i];
    for (int i = tid; i < nblk_tile; i += kSweepThreads) sflag[i] = 0;
    load_tile(sP, P + row * pitchP, t0, n, pitchP, len, mbar);

    for (int i = tid; i < tile && t0 + i < n; i += kSweepThreads) {
        float s = 0.f;
        bool hit = false;
        const long long room = n - (t0 + i); // widths with i + w ≤ n
        const int wmax = room < (long long)zmax ? (int)room : zmax;
        for (int w = 1; w <= wmax; ++w) {
            s += sP[i + w - 1];
            hit = hit || (s >= sT[w - 1]);
        }
        if (hit) sflag[(int)((t0 + i) / C - c_first)] = 1;
    }
    __syncthreads();
    publish_flags(sflag, nblk_tile, c_first, nblk, row, bitmap, flagged, counters);
}

} // namespace pulscan
