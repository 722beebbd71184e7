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
// bin.  Here the tile (+ zmax halo) is staged in shared memory by one TMA bulk copy and swept with COVER SUMS:
// P ≥ 0, so a window of width w is bounded above by the sum of the aligned g-bin groups that cover it.  For a level
// (g, [wlo, whi]) thread t accumulates U(k0,m) = Σ_{k<m} G_g[k0+k] for R consecutive group starts k0 in registers
// and compares with τ(m) = T'_{max(wlo, (m−2)g+2)} — (n/g)·(whi/g+2) additions instead of n·(whi−wlo+1).  g grows
// like √w (chosen on the host so that a noise cover passes with probability ≤ p_flag), which makes every level cost
// O(n).  A cover that passes is refined exactly (its ≤ g² windows summed and compared with their own T'_w).
//
// Exhaustive mode (the cross-check) evaluates every (i, w) by the paper's recursion instead.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace pulscan {

constexpr int kMaxLevels = 8;
constexpr int kSweepR = 8;      // consecutive group starts per thread (register sliding window)
constexpr int kSweepThreads = 256;
constexpr int kSweepPad = 2 * kSweepR; // zero entries after each group array (sliding-window over-read)

struct SweepLevel {
    int lg;        // log2 of the group size g
    int wlo, whi;  // widths this level answers for
    int m_lo;      // smallest number of groups a cover of a width-wlo window has
    int m_hi;      // largest number of groups a cover of a width-whi window has
    int tau_off;   // offset of τ[0..m_hi) in the τ table (τ[m−1] ↔ cover of m groups; +inf below m_lo)
    int g_off;     // offset (floats) of this level's group array in shared memory
    int task_off;  // first flattened task index of this level
    int ntasks;    // ceil(tile/g / R)
};

struct SweepParams {
    int nlevels;
    int lgmax;      // arrays for lg = 0..lgmax are built
    int tile;       // start bins per CTA
    int len;        // tile + halo, multiple of 64
    int ntasks;
    int ntau;
    int smem_floats; // data floats (group arrays incl. pads)
    int g_off[8];    // offsets of the group arrays for lg = 0..7
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

// U(k0,m) for R consecutive k0 = base..base+R−1 and m = 1..m_hi; returns max over (k0, m) of U − τ[m−1].
template <int R>
__device__ __forceinline__ float sweep_task(const float* __restrict__ G, int base, int m_hi,
                                            const float* __restrict__ tau) {
    float buf[R], U[R];
#pragma unroll
    for (int j = 0; j < R; ++j) { buf[j] = G[base + j]; U[j] = 0.f; }
    float flag = -INFINITY;
    for (int m0 = 0; m0 < m_hi; m0 += R) {
#pragma unroll
        for (int s = 0; s < R; ++s) {
            const int m = m0 + s;
            if (m < m_hi) {
#pragma unroll
                for (int r = 0; r < R; ++r) U[r] += buf[(r + s) % R];
                float mx = U[0];
#pragma unroll
                for (int r = 1; r < R; ++r) mx = fmaxf(mx, U[r]);
                flag = fmaxf(flag, mx - tau[m]);
                buf[s] = G[base + R + m];
            }
        }
    }
    return flag;
}

struct SweepCtx {
    const float* sP;
    const float* Tp;        // global: T'_w, w = 1..zmax (conservative float thresholds)
    unsigned char* sflag;   // shared: one byte per candidate block touched by the tile
    long long t0, n;
    int tile, C;
    long long c_first;      // first candidate block of the tile
};

// A cover of m+1 groups starting at group k0 passed its bound: sum its windows exactly (float32) and mark the
// candidate block of every start bin that owns a window with S ≥ T'_w.
__device__ __noinline__ void refine_cover(const SweepCtx& cx, const SweepLevel& lv, const float* __restrict__ G,
                                          int k0, int m) {
    const int g = 1 << lv.lg;
    const int i_lo = k0 * g;
    long long lim = cx.n - cx.t0;
    int i_hi = i_lo + g;
    if (i_hi > cx.tile) i_hi = cx.tile;
    if ((long long)i_hi > lim) i_hi = (int)lim;
    float inner = 0.f;
    for (int k = k0 + 1; k < k0 + m; ++k) inner += G[k];
    const int e_lo = (m == 0) ? i_lo : (k0 + m) * g; // first bin of the last group of the cover
    for (int i = i_lo; i < i_hi; ++i) {
        const int cb = (int)((cx.t0 + i) / cx.C - cx.c_first);
        if (cx.sflag[cb]) continue;
        float s = inner;
        if (m > 0)
            for (int j = i; j < i_lo + g; ++j) s += cx.sP[j];
        const int e_first = (m == 0) ? i : e_lo;
        for (int e = e_first; e < e_lo + g; ++e) { // window [i, e]
            s += cx.sP[e];
            const int w = e - i + 1;
            if (w < lv.wlo) continue;
            if (w > lv.whi || cx.t0 + e >= cx.n) break;
            if (s >= __ldg(cx.Tp + (w - 1))) { cx.sflag[cb] = 1; break; }
        }
    }
}

template <int R>
__device__ __noinline__ void refine_task(const SweepCtx& cx, const SweepLevel& lv, const float* __restrict__ G,
                                         int base, const float* __restrict__ tau) {
    const int g = 1 << lv.lg;
    for (int r = 0; r < R; ++r) {
        const int k0 = base + r;
        if (k0 * g >= cx.tile || cx.t0 + (long long)k0 * g >= cx.n) break;
        float U = 0.f;
        for (int m = 0; m < lv.m_hi; ++m) {
            U += G[k0 + m];
            if (U >= tau[m]) refine_cover(cx, lv, G, k0, m);
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

// Pruned sweep.  Grid: tiles_per_row · batch CTAs of kSweepThreads; dynamic shared memory:
//   [smem_floats group arrays][ntau τ][nblk_tile flag bytes][mbarrier].
__global__ void __launch_bounds__(kSweepThreads)
boxcar_sweep_kernel(const __grid_constant__ SweepParams sp, const float* __restrict__ P, long long pitchP, long long n,
                    int tiles_per_row, int C, long long nblk, const float* __restrict__ tau_g,
                    const float* __restrict__ Tp_g, unsigned* __restrict__ bitmap, unsigned* __restrict__ flagged,
                    unsigned* __restrict__ counters) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* sG = reinterpret_cast<float*>(smem_raw);
    float* sTau = sG + sp.smem_floats;
    uint64_t* mbar = reinterpret_cast<uint64_t*>(sTau + ((sp.ntau + 3) & ~3));
    unsigned char* sflag = reinterpret_cast<unsigned char*>(mbar + 2);

    const int tid = threadIdx.x;
    const long long row = blockIdx.x / tiles_per_row;
    const long long t0 = (long long)(blockIdx.x % tiles_per_row) * sp.tile;
    const long long c_first = t0 / C;
    long long last_start = t0 + sp.tile - 1;
    if (last_start > n - 1) last_start = n - 1;
    const int nblk_tile = (int)(last_start / C - c_first) + 1;

    for (int i = tid; i < sp.ntau; i += kSweepThreads) sTau[i] = tau_g[i];
    for (int i = tid; i < nblk_tile; i += kSweepThreads) sflag[i] = 0;
    load_tile(sG, P + row * pitchP, t0, n, pitchP, sp.len, mbar); // ends with __syncthreads()

    // group arrays: G_lg[k] = G_{lg−1}[2k] + G_{lg−1}[2k+1], plus kSweepPad zeros after each array
    for (int i = tid; i < kSweepPad; i += kSweepThreads) sG[sp.len + i] = 0.f;
    for (int lg = 1; lg <= sp.lgmax; ++lg) {
        const float* src = sG + sp.g_off[lg - 1];
        float* dst = sG + sp.g_off[lg];
        const int cnt = sp.len >> lg;
        for (int k = tid; k < cnt; k += kSweepThreads) {
            const float2 a = reinterpret_cast<const float2*>(src)[k];
            dst[k] = a.x + a.y;
        }
        for (int i = tid; i < kSweepPad; i += kSweepThreads) dst[cnt + i] = 0.f;
        __syncthreads();
    }
    if (sp.lgmax == 0) __syncthreads();

    SweepCtx cx{sG, Tp_g, sflag, t0, n, sp.tile, C, c_first};
    for (int task = tid; task < sp.ntasks; task += kSweepThreads) {
        int L = 0;
        while (L + 1 < sp.nlevels && task >= sp.lv[L + 1].task_off) ++L;
        const SweepLevel& lv = sp.lv[L];
        const int base = (task - lv.task_off) * kSweepR;
        const float* G = sG + lv.g_off;
        const float flag = sweep_task<kSweepR>(G, base, lv.m_hi, sTau + lv.tau_off);
        if (flag >= 0.f) refine_task<kSweepR>(cx, lv, G, base, sTau + lv.tau_off);
    }
    __syncthreads();
    publish_flags(sflag, nblk_tile, c_first, nblk, row, bitmap, flagged, counters);
}

// Exhaustive sweep (cross-check mode): thread per start bin, the paper's recursion S(i,w) = S(i,w−1) + P[i+w−1]
// over every width, compared with T'_w.  Same outputs as the pruned kernel.  Dynamic shared memory:
//   [len floats][zmax T'][nblk_tile flag bytes][mbarrier].
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
