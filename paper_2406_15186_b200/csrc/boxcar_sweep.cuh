// boxcar_sweep.cuh — kernel (b): the boxcar sweep over the float32 power spectrum.
//
// What must be found (§2.2.5; Alg. 4): for every start bin i and every width
// w ≤ zmax the sum S(i,w) = Σ_{j<w} P[i+j], and per candidate block the maxima.  A window can only become a candidate
// if S(i,w) ≥ T_w, the power at which width w reaches the σ threshold (L342-344: "compared with precomputed
// threshold values").  In noise that happens for ~1e-9 of all (i,w), so this kernel is a FILTER: it marks the
// candidate blocks that contain at least one window with S ≥ T_w·(1−ε) and kernel (c) then evaluates exactly those
// blocks in double precision.  Nothing a marked block could emit is lost and an unmarked block cannot emit.
//
// The paper's kernel (Alg. 4) does one shared-memory add per (bin, width) — issue-bound, ~2·zmax instructions per
// bin.  Here the tile (+ zmax halo) is staged in shared memory by one TMA bulk copy, turned into its prefix sum
// PP[i] = Σ_{j<i} P[j] once, and swept with COVER SUMS: P ≥ 0, so a window of width w is bounded above by the sum of
// the aligned g-bin groups that cover it, U(k0,m) = PP[(k0+m)·g] − PP[k0·g].  For a level (g, [wlo, whi]) a thread
// holds PP at 8 consecutive group starts in registers and slides over m: one FADD + half an FMNMX3 per cover sum,
// (n/g)·(whi/g+2) cover sums instead of n·(whi−wlo+1) window sums.  g grows like √w (chosen on the host so that a
// cover of pure noise passes with probability ≤ p_flag), which makes every level cost O(n).  Covers that pass go to a
// shared-memory work list and are refined afterwards by whole warps: their ≤ g² windows are summed from PP and
// compared with their own T'_w.
//
// Float safety.  PP is a float32 scan; every PP[i] carries at most ~36 roundings of magnitude
// ≤ 2⁻²⁴·PP[len], so a difference of two entries is off by < slack = kSlackUlps·2⁻²⁴·PP[len] from the exact sum of
// the float32 powers.  Every comparison adds the slack on the side that keeps the cover / window.
//
// Exhaustive mode (the cross-check) evaluates every (i, w) by the paper's recursion instead.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace pulscan {

constexpr int kMaxLevels = 8;
constexpr int kSweepThreads = 256;
constexpr int kSweepR = 8;                 // consecutive group starts per thread
constexpr int kScanPer = 20;               // floats per thread per scan pass: 80-byte lane stride is bank-conflict-free
constexpr int kScanPass = kScanPer * kSweepThreads;
constexpr int kWorkCap = 384;              // flagged (8 group starts × 4 cover lengths) cells per tile before giving up
constexpr int kMaxWarpTasks = 128;         // warp-tasks per tile (8 levels of at most tile/(256·g) each)
constexpr int kPadG = 16;                  // replicated entries after each decimated prefix array (window over-read)
constexpr float kSlackUlps = 96.f;         // ≥ 2·(19 + 5 + 7 + 3 + passes) + 1 roundings, see above

struct SweepLevel {
    int lg;        // log2 of the group size g
    int wlo, whi;  // widths this level answers for
    int m_lo;      // smallest number of groups a cover of a width-wlo window has
    int m_hi;      // largest number of groups a cover of a width-whi window has
    int m_start;   // m_lo rounded down to a multiple of 4 (16-byte alignment of the sliding window's vector loads)
    int nsteps;    // 4-wide steps over m: m_start + 4·nsteps > m_hi; ≤ 33; τ = +inf below m_lo and above m_hi
    int tau_off;   // offset of τ[m_start ..] in the τ table (4·nsteps entries)
    int pg_off;    // offset (floats) of this level's decimated prefix array PG[k] = PP[k·g] in shared memory
    int nk;        // group starts per tile = tile / g
    int wt_off;    // first warp-task of this level; a warp-task is 32 lanes × 8 group starts
    int nwt;       // warp-tasks of this level
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
    int npass;       // scan passes per tile = ceil(len / kScanPass)
    int z_floats;    // floats of ONE tile buffer: 4 + npass·kScanPass + 4 (Z[3] = PP[0], raw powers / PP from Z[4])
    int smem_floats; // two tile buffers + decimated arrays
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
// Prefix scan, in place.  Z is a tile buffer: on entry Z[4+i] = P[t0+i] for i < len and 0 for len ≤ i < len+kScanPer
// (beyond that: don't care); on exit Z[3+i] = PP[i] = Σ_{j<i} P[t0+j] for i ∈ [0, len] (Z[3] = 0 is set once per
// kernel).  In-place is safe because every read of a pass happens before the pass's barrier and every write after it,
// and a thread writes exactly the entries it has read.
// Each thread owns kScanPer = 20 consecutive entries (80-byte lane stride: conflict-free 16-byte accesses), so the
// multiples of g among them follow a fixed pattern and the decimated arrays PG_lg[k] = PP[k << lg], k ∈ [0, len >> lg],
// are written straight from the scan registers with compile-time register indices.  Entries past len >> lg (written by
// the thread that straddles len, ≤ 5 of them, inside the kPadG pad) equal PP[len] because of the zeros after len: a
// cover that reaches past the staged bins gains nothing; the other pad entries only ever meet τ = +inf and are zeroed
// once per kernel.  Also clears the tile's block flags (between its barriers).  Ends with a CTA barrier.
struct ScanSmem {
    alignas(16) float wtot[kSweepThreads / 32];
};

__device__ __forceinline__ float scan_sel5(const float (&x)[kScanPer], int q) {
    float v = x[19];
    v = (q == 3) ? x[15] : v;
    v = (q == 2) ? x[11] : v;
    v = (q == 1) ? x[7] : v;
    v = (q == 0) ? x[3] : v;
    return v;
}

__device__ __forceinline__ void scan_tile(const SweepParams& sp, float* Z, float* sG, ScanSmem& ss, unsigned char* sflag,
                                          int nblk_tile) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int len = sp.len;
    float carry = 0.f;
    if (tid < sp.narr) sG[sp.arr_off[tid]] = 0.f;
    for (int pass = 0; pass < sp.npass; ++pass) {
        const int i0 = pass * kScanPass + kScanPer * tid;
        const bool act = i0 < len;
        float4* zq = reinterpret_cast<float4*>(Z + 4) + (i0 >> 2);
        float x[kScanPer];
        if (act) {
#pragma unroll
            for (int q = 0; q < kScanPer / 4; ++q) {
                const float4 v = zq[q];
                x[4 * q] = v.x; x[4 * q + 1] = v.y; x[4 * q + 2] = v.z; x[4 * q + 3] = v.w;
            }
            // prefix inside each quad (5 independent chains), then the chain over the quad totals
#pragma unroll
            for (int q = 0; q < kScanPer / 4; ++q) {
                x[4 * q + 1] += x[4 * q]; x[4 * q + 2] += x[4 * q + 1]; x[4 * q + 3] += x[4 * q + 2];
            }
#pragma unroll
            for (int q = 1; q < kScanPer / 4; ++q) x[4 * q + 3] += x[4 * q - 1];
        } else {
#pragma unroll
            for (int j = 0; j < kScanPer; ++j) x[j] = 0.f;
        }
        float incl = x[kScanPer - 1];
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const float t = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += t;
        }
        float excl = __shfl_up_sync(0xffffffffu, incl, 1);
        if (lane == 0) excl = 0.f;
        if (lane == 31) ss.wtot[warp] = incl;
        __syncthreads();
        // every thread has left the previous tile's publish_flags: clear the block flags for this tile (ordered before
        // the first refinement by the barrier that ends the pass)
        if (pass == 0)
            for (int i = tid; i < nblk_tile; i += kSweepThreads) sflag[i] = 0;
        const float4 wa = *reinterpret_cast<const float4*>(ss.wtot), wb = *reinterpret_cast<const float4*>(ss.wtot + 4);
        const float wt[8] = {wa.x, wa.y, wa.z, wa.w, wb.x, wb.y, wb.z, wb.w};
        float wbase = 0.f, total = 0.f;
#pragma unroll
        for (int w = 0; w < kSweepThreads / 32; ++w) {
            if (w == warp) wbase = total;
            total += wt[w];
        }
        if (act) {
            const float off = carry + (wbase + excl);
#pragma unroll
            for (int q = kScanPer / 4 - 1; q >= 0; --q) {       // x[j] = PP[i0 + j + 1]
                const float oq = q ? off + x[4 * q - 1] : off;  // x[4q−1] is still the thread-local prefix here
                x[4 * q] += oq; x[4 * q + 1] += oq; x[4 * q + 2] += oq;
                x[4 * q + 3] += off;
            }
#pragma unroll
            for (int q = 0; q < kScanPer / 4; ++q) zq[q] = make_float4(x[4 * q], x[4 * q + 1], x[4 * q + 2], x[4 * q + 3]);
            const int u = (i0 >> 2) + 1;                        // candidates for lg ≥ 2: PP[4(u+q)] = x[4q+3], q = 0..4
            for (int a = 0; a < sp.narr; ++a) {
                const int lg = sp.arr_lg[a];
                float* dst = sG + sp.arr_off[a];
                if (lg == 2) {
#pragma unroll
                    for (int q = 0; q < 5; ++q) dst[u + q] = x[4 * q + 3];
                } else if (lg == 3) {
                    const bool odd = u & 1;                     // hits q = odd, odd+2 (and 4 when even)
                    float* d = dst + ((u + 1) >> 1);
                    d[0] = odd ? x[7] : x[3];
                    d[1] = odd ? x[15] : x[11];
                    if (!odd) d[2] = x[19];
                } else if (lg >= 4) {
                    const int sh = lg - 2, q0 = (-u) & ((1 << sh) - 1);
                    if (q0 < 5) dst[(u + q0) >> sh] = scan_sel5(x, q0);
                    if (lg == 4 && q0 == 0) dst[((u + 4) >> 2)] = x[19];
                } else if (lg == 1) {
#pragma unroll
                    for (int q = 0; q < kScanPer / 2; ++q) dst[(i0 >> 1) + 1 + q] = x[2 * q + 1];
                } else {
#pragma unroll
                    for (int j = 0; j < kScanPer; ++j)
                        if (i0 + j + 1 <= len + kPadG) dst[i0 + j + 1] = x[j];
                }
            }
        }
        carry += total;
        __syncthreads();
    }
}

// One 4-wide step over m for 8 group starts.  O is the rotation of the 12-entry window W (compile time, so that the
// window never moves between registers): W[(O + j) % 12] = PG[k0b + m + j], j = 0..11 after the load below.
template <int O>
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
        for (int r = 0; r < kSweepR; ++r) u[r] = W[(O + q + r) % 12] - A[r];
        const float m0 = fmaxf(fmaxf(u[0], u[1]), u[2]);
        const float m1 = fmaxf(fmaxf(u[3], u[4]), u[5]);
        const float m2 = fmaxf(fmaxf(u[6], u[7]), m0);
        hit = hit || (fmaxf(m1, m2) >= tq[q]);
    }
    return hit;
}

// All covers of one level for 8 consecutive group starts k0b..k0b+7: returns the bit mask of the 4-wide m steps in
// which some cover reached its threshold (slack already folded into A).
__device__ __forceinline__ unsigned sweep_task(const float* __restrict__ PG, int k0b, int m_start, int nsteps,
                                               const float* __restrict__ tau, float slack) {
    float A[kSweepR], W[12];
    {
        const float4 a0 = *reinterpret_cast<const float4*>(PG + k0b);
        const float4 a1 = *reinterpret_cast<const float4*>(PG + k0b + 4);
        A[0] = a0.x - slack; A[1] = a0.y - slack; A[2] = a0.z - slack; A[3] = a0.w - slack;
        A[4] = a1.x - slack; A[5] = a1.y - slack; A[6] = a1.z - slack; A[7] = a1.w - slack;
        const float* p = PG + k0b + m_start;
        const float4 w0 = *reinterpret_cast<const float4*>(p);
        const float4 w1 = *reinterpret_cast<const float4*>(p + 4);
        W[0] = w0.x; W[1] = w0.y; W[2] = w0.z; W[3] = w0.w; W[4] = w1.x; W[5] = w1.y; W[6] = w1.z; W[7] = w1.w;
        W[8] = W[9] = W[10] = W[11] = 0.f;
    }
    unsigned mask = 0;
    const float* p = PG + k0b + m_start + 8;
    for (int s = 0; s < nsteps; s += 3) {
        if (sweep_step<0>(A, W, p, tau)) mask |= 1u << s;
        if (s + 1 < nsteps && sweep_step<4>(A, W, p + 4, tau + 4)) mask |= 2u << s;
        if (s + 2 < nsteps && sweep_step<8>(A, W, p + 8, tau + 8)) mask |= 4u << s;
        p += 12; tau += 12;
    }
    return mask;
}

struct SweepCtx {
    const float* Z;         // PP region (PP[i] = Z[3+i])
    const float* Tp;        // shared: T'_w, w = 1..zmax (conservative float thresholds)
    unsigned char* sflag;   // shared: one byte per candidate block touched by the tile
    int t0, n;              // n_bins < 2^31 (pulscan_plan_create)
    int C;
    int rem;                // t0 − c_first·C: offset of the tile's first bin inside its candidate block
    float inv_C;
    float slack;
};

// Candidate block (relative to the tile's first one) that owns start bin t0 + i.  i < 2^24, so the float quotient is
// off by at most one and the two corrections make it exact.
__device__ __forceinline__ int rel_block(const SweepCtx& cx, int i) {
    const int x = cx.rem + i;
    int q = __float2int_rz(__int2float_rn(x) * cx.inv_C);
    q -= (q * cx.C > x);
    q += ((q + 1) * cx.C <= x);
    return q;
}

// One flagged cell (level L, group starts k0b..k0b+7, cover lengths m4..m4+3), one cover per lane: re-test it and sum
// the windows of every cover that passes, all 32 lanes sharing the ≤ g² (start, end) pairs.
__device__ __forceinline__ void refine_cell(const SweepCtx& cx, const SweepLevel& lv, const float* __restrict__ PG,
                                            const float* __restrict__ tau, int k0b, int step) {
    const int lane = threadIdx.x & 31;
    const int k0 = k0b + (lane & 7);
    const int m = lv.m_start + 4 * step + (lane >> 3);
    const float U = PG[k0 + m] - PG[k0];
    const int g = 1 << lv.lg;
    bool live = U + cx.slack >= tau[4 * step + (lane >> 3)];
    if (live && g <= cx.C) {   // nothing left to find if the (one or two) blocks owning the cover's start bins are marked
        const int b0 = k0 << lv.lg;
        live = !(cx.sflag[rel_block(cx, b0)] && cx.sflag[rel_block(cx, b0 + g - 1)]);
    }
    unsigned hits = __ballot_sync(0xffffffffu, live);
    while (hits) {
        const int src = __ffs(hits) - 1;
        hits &= hits - 1;
        const int kk = k0b + (src & 7), mm = lv.m_start + 4 * step + (src >> 3);
        const int i0 = kk << lv.lg, e0 = (kk + mm - 1) << lv.lg;
        for (int idx = lane; idx < g * g; idx += 32) {
            const int i = i0 + (idx >> lv.lg), e = e0 + (idx & (g - 1));
            const int w = e - i + 1;
            if (w < 1 || w < lv.wlo || w > lv.whi || cx.t0 + e >= cx.n) continue;
            const float S = cx.Z[3 + e + 1] - cx.Z[3 + i];
            if (S + cx.slack >= cx.Tp[w - 1]) cx.sflag[rel_block(cx, i)] = 1;
        }
        if (g <= cx.C) {       // later covers of this cell: drop those whose blocks have just been marked
            bool dead = false;
            if (hits >> lane & 1u) {
                const int b0 = k0 << lv.lg;
                dead = cx.sflag[rel_block(cx, b0)] && cx.sflag[rel_block(cx, b0 + g - 1)];
            }
            __syncwarp();
            hits &= ~__ballot_sync(0xffffffffu, dead);
        }
    }
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

// What one tile needs to know; written by thread 0 when it issues the tile's TMA copy, read by everybody two barriers later.
struct TileMeta {
    int row, t0;
    int c_first, nblk_tile;   // candidate blocks touched by the tile's start bins
    int first_pad;            // valid bins staged (the rest of the buffer up to len + kScanPer must read as zero)
    int pad_[3];
};

// A warp-task: the covers of one level for 32 × 8 consecutive group starts.  The list is the same for every tile, so it
// is built once per CTA; warp w runs tasks w, w + 8, … of every tile.
struct alignas(16) WarpTask {
    int pg_off, tau_off, m_start, nsteps;
    int level, kbase, nk, pad_;
};

struct SweepCtl {
    ScanSmem scan;
    alignas(8) uint64_t mbar[2];
    TileMeta meta[2];
    unsigned work_n;
    unsigned work[kWorkCap];
    WarpTask task[kMaxWarpTasks];
};

// The sweep proper, on a tile whose PP region and decimated arrays are ready.  Marks sflag[]; the caller publishes.
// Flagged cells go to a shared work list and are refined by all warps after a barrier (a warp refining its own cells
// on the spot was measured slower: the few warps with hits then hold everybody at the final barrier).
// counters[2] += work-list cells, counters[3] += tiles whose work list overflowed (all their blocks get marked).
// Ends with a CTA barrier after which nobody reads Z, sG or the work list any more.
__device__ __forceinline__ void sweep_covers(const SweepParams& sp, const float* __restrict__ sG,
                                             const float* __restrict__ sTau, SweepCtl& ctl, const SweepCtx& cx,
                                             int nblk_tile, unsigned* __restrict__ counters) {
    const int lane = threadIdx.x & 31;
    for (int q = threadIdx.x >> 5; q < sp.ntasks; q += kSweepThreads / 32) {
        const int4 ta = *reinterpret_cast<const int4*>(&ctl.task[q]);            // pg_off, tau_off, m_start, nsteps
        const int4 tb = *reinterpret_cast<const int4*>(&ctl.task[q].level);      // level, kbase, nk
        const int k0b = tb.y + lane * kSweepR;
        if (k0b < tb.z) {
            unsigned mask = sweep_task(sG + ta.x, k0b, ta.z, ta.w, sTau + ta.y, cx.slack);
            while (mask) {
                const int s = __ffs(mask) - 1;
                mask &= mask - 1;
                const unsigned pos = atomicAdd(&ctl.work_n, 1u);
                if (pos < (unsigned)kWorkCap) ctl.work[pos] = ((unsigned)q << 24) | ((unsigned)s << 16) | (unsigned)(k0b >> 3);
            }
        }
    }
    __syncthreads();
    const unsigned nwork = ctl.work_n;
    if (nwork > (unsigned)kWorkCap) {
        for (int i = threadIdx.x; i < nblk_tile; i += kSweepThreads) cx.sflag[i] = 1;
    } else {
        for (unsigned e = threadIdx.x >> 5; e < nwork; e += kSweepThreads / 32) {
            const unsigned w = ctl.work[e];
            const WarpTask& t = ctl.task[w >> 24];
            refine_cell(cx, sp.lv[t.level], sG + t.pg_off, sTau + t.tau_off, (int)(w & 0xFFFFu) << 3, (int)((w >> 16) & 0xFFu));
        }
    }
    if (threadIdx.x == 0 && nwork) {
        atomicAdd(counters + 2, nwork);
        if (nwork > (unsigned)kWorkCap) atomicAdd(counters + 3, 1u);
    }
    __syncthreads();
}

// Thread 0: describe tile `item` (= row·tiles_per_row + tile index) in `m` and start its TMA copy into Zbuf + 4.
// The copy is clipped to the row's allocation (pitchP), so it never touches the next spectrum (R11); P rows start
// 16-byte aligned and pitchP, tile and len are multiples of 4, so the copy always satisfies TMA's alignment rules.
__device__ __forceinline__ void sweep_issue_tile(const SweepParams& sp, long long item, const float* __restrict__ P,
                                                 long long pitchP, long long n, int tiles_per_row, int C, float* Zbuf,
                                                 uint64_t* mbar, TileMeta& m) {
    const int row = (int)(item / tiles_per_row);
    const int t0 = (int)(item - (long long)row * tiles_per_row) * sp.tile;          // n < 2^31
    const long long avail = pitchP - t0;
    const int ncopy = (int)(avail < (long long)sp.len ? avail : (long long)sp.len);
    const long long nv = n - t0;
    m.row = row; m.t0 = t0;
    m.first_pad = (int)(nv < (long long)sp.len ? nv : (long long)sp.len);
    m.c_first = t0 / C;
    const int last_start = (int)min((long long)t0 + sp.tile - 1, n - 1);
    m.nblk_tile = last_start / C - m.c_first + 1;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");    // the buffer's earlier generic accesses precede the copy
    const uint32_t bytes = (uint32_t)ncopy * 4u;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(mbar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(Zbuf + 4)),
                 "l"(P + (long long)row * pitchP + t0), "r"(bytes), "r"(smem_u32(mbar))
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

// Pruned sweep, persistent: gridDim.x CTAs (a multiple of the SM count) stride over the n_items = tiles_per_row · batch
// tiles; two tile buffers, so the TMA copy of a CTA's next tile is in flight while it scans and sweeps the current one.
// Dynamic shared memory: [2 × z_floats tile buffers][decimated arrays][ntau τ][zmax T'][SweepCtl][flag bytes].
__global__ void __launch_bounds__(kSweepThreads, 4)
boxcar_sweep_kernel(const __grid_constant__ SweepParams sp, const float* __restrict__ P, long long pitchP, long long n,
                    int tiles_per_row, long long n_items, int C, long long nblk, const float* __restrict__ tau_g,
                    const float* __restrict__ Tp_g, unsigned* __restrict__ bitmap, unsigned* __restrict__ flagged,
                    unsigned* __restrict__ counters) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* Zb0 = reinterpret_cast<float*>(smem_raw);
    float* sG = Zb0 + 2 * sp.z_floats;
    float* sTau = Zb0 + sp.smem_floats;
    float* sTp = sTau + ((sp.ntau + 3) & ~3);
    SweepCtl& ctl = *reinterpret_cast<SweepCtl*>(sTp + ((sp.zmax + 3) & ~3));
    unsigned char* sflag = reinterpret_cast<unsigned char*>(&ctl + 1);
    const int tid = threadIdx.x;
    const long long stride = gridDim.x;
    const float inv_C = 1.0f / (float)C;

    // ---- once per CTA: τ table, constants of the buffers, the first two copies
    for (int i = tid; i < sp.ntau; i += kSweepThreads) sTau[i] = tau_g[i];
    for (int i = tid; i < sp.zmax; i += kSweepThreads) sTp[i] = Tp_g[i];
    for (int i = tid; i < sp.smem_floats - 2 * sp.z_floats; i += kSweepThreads) sG[i] = 0.f;   // incl. the arrays' pads
    if (tid < 2) Zb0[tid * sp.z_floats + 3] = 0.f;                                             // PP[0]
    if (tid < 2 * kScanPer) Zb0[(tid / kScanPer) * sp.z_floats + 4 + sp.len + tid % kScanPer] = 0.f;   // zeros after len
    for (int q = tid; q < sp.ntasks; q += kSweepThreads) {
        int L = 0;
        while (L + 1 < sp.nlevels && q >= sp.lv[L + 1].wt_off) ++L;
        const SweepLevel& lv = sp.lv[L];
        ctl.task[q] = WarpTask{lv.pg_off, lv.tau_off, lv.m_start, lv.nsteps, L, (q - lv.wt_off) * 32 * kSweepR, lv.nk, 0};
    }
    if (tid == 0) {
        ctl.work_n = 0;
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&ctl.mbar[0])));
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&ctl.mbar[1])));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        const long long i0 = blockIdx.x;
        if (i0 < n_items) sweep_issue_tile(sp, i0, P, pitchP, n, tiles_per_row, C, Zb0, &ctl.mbar[0], ctl.meta[0]);
        if (i0 + stride < n_items)
            sweep_issue_tile(sp, i0 + stride, P, pitchP, n, tiles_per_row, C, Zb0 + sp.z_floats, &ctl.mbar[1], ctl.meta[1]);
    }
    __syncthreads();

    int it = 0;
    for (long long item = blockIdx.x; item < n_items; item += stride, ++it) {
        const int b = it & 1;
        float* Z = Zb0 + b * sp.z_floats;
        const TileMeta mt = ctl.meta[b];
        mbar_wait(&ctl.mbar[b], (uint32_t)(it >> 1) & 1u);
        if (mt.first_pad < sp.len) {                         // last tile of a row: nothing beyond the spectrum's end
            for (int i = mt.first_pad + tid; i < sp.len; i += kSweepThreads) Z[4 + i] = 0.f;
            __syncthreads();
        }
        scan_tile(sp, Z, sG, ctl.scan, sflag, mt.nblk_tile);
        const float pp_max = Z[3 + sp.len];
        SweepCtx cx{Z, sTp, sflag, mt.t0, (int)n, C, mt.t0 - mt.c_first * C, inv_C, kSlackUlps * 5.9604644775390625e-8f * pp_max};
        sweep_covers(sp, sG, sTau, ctl, cx, mt.nblk_tile, counters);
        if (tid == 0) {
            ctl.work_n = 0;
            const long long nxt = item + 2 * stride;
            if (nxt < n_items) sweep_issue_tile(sp, nxt, P, pitchP, n, tiles_per_row, C, Z, &ctl.mbar[b], ctl.meta[b]);
        } else if (tid >= 32 && tid < 32 + kScanPer) {
            Z[4 + sp.len + (tid - 32)] = 0.f;                // the scan has written PP garbage over the zeros after len
        }
        publish_flags(sflag, mt.nblk_tile, mt.c_first, nblk, mt.row, bitmap, flagged, counters);
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
