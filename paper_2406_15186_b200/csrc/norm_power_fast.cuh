// norm_power_fast.cuh — kernel (a), fast path: full normalisation blocks of exactly B = EPT·NT bins.
//
// Same result as norm_power.cuh's general path (exact medians, Eq. 8), organised for throughput:
//  * both components move through the same phases together, so one CTA barrier serves two selects;
//  * each select is ONE histogram pass (256 value-linear buckets between known bounds, bucket index taken from the
//    mantissa of fma(v − lo, scale, 1.5·2²³): FADD, FFMA, shared-memory red.add) whose bucket indices are kept packed
//    four to a register, so the gather pass is one byte-compare per four values;
//  * warp 0 / warp 1 scan the re / im histogram (8 buckets per lane + one warp scan) and publish the bucket holding
//    rank k, plus the next non-empty bucket when rank k+1 (even length) lies beyond it;
//  * the few dozen members are ranked by counting, one thread per member;
//  * the MAD needs no min/max pass: |v − m| ≤ max(hi − a, b − lo).
// Nine CTA barriers per block instead of ~40.  Whenever a shortcut does not apply (degenerate range, a bucket with
// more than kFastListCap members, e.g. a block stretched by a strong outlier) the block id goes to a redo list and
// norm_power_redo_kernel runs it through the general path.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "norm_power.cuh"

namespace pulscan {

constexpr int kFastListCap = 128;
constexpr float kMagic = 12582912.0f;          // 1.5·2²³: adding it leaves round(t) in the low mantissa bits
constexpr unsigned kMagicBits = 0x4B400000u;   // low byte is zero, so (bits & 0xFF) is the bucket for t in [0, 255]

struct FastSmem {
    unsigned hist[2][2][kSelBuckets]; // [phase: median, MAD][component][bucket]
    float list[2][kFastListCap];
    unsigned list_n[2][2];            // [phase][component]
    float wmin[2][32], wmax[2][32];
    int sel[2], nb2[2];
    unsigned excl[2], cnt[2];
    unsigned res_key[2][2][2];        // [phase][component][rank k, rank k+1] as order-preserving keys
    int fail;
};

__device__ __forceinline__ void red_shared_inc(unsigned addr) {
    asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(addr) : "memory");
}

// Histogram pass for one component: bucket = round((v − lo)·scale) ∈ [0, 255]; packs the bucket bytes into idx[].
template <int EPT, bool SUB>
__device__ __forceinline__ void fast_hist(const float (&v)[EPT], float lo, float scale, unsigned hist_addr,
                                          unsigned (&idx)[(EPT + 3) / 4]) {
#pragma unroll
    for (int q = 0; q < (EPT + 3) / 4; ++q) idx[q] = 0;
#pragma unroll
    for (int r = 0; r < EPT; ++r) {
        const float t = SUB ? __fsub_rn(v[r], lo) : v[r];
        const unsigned bits = __float_as_uint(__fmaf_rn(t, scale, kMagic));
        red_shared_inc(hist_addr + ((bits & 0xFFu) << 2));   // masked: a NaN input cannot leave the histogram
        idx[r >> 2] = __byte_perm(idx[r >> 2], bits, (r & 3) == 0 ? 0x3214 : (r & 3) == 1 ? 0x3240 : (r & 3) == 2 ? 0x3410 : 0x4210);
    }
}

// One warp scans one component's 256-bucket histogram (8 buckets per lane) and publishes: the bucket holding rank kk,
// the number of values below it, the member count to gather, and the next non-empty bucket if rank kk+1 is needed
// and lies beyond the selected bucket.
__device__ __forceinline__ void fast_scan(const unsigned* __restrict__ hist, unsigned kk, bool need_next, FastSmem& sm,
                                          int c) {
    const int lane = threadIdx.x & 31;
    const uint4 h0 = reinterpret_cast<const uint4*>(hist)[2 * lane];
    const uint4 h1 = reinterpret_cast<const uint4*>(hist)[2 * lane + 1];
    const unsigned cnt[8] = {h0.x, h0.y, h0.z, h0.w, h1.x, h1.y, h1.z, h1.w};
    unsigned tot = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) tot += cnt[j];
    unsigned inc = tot;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, inc, off);
        if (lane >= off) inc += t;
    }
    const unsigned base = inc - tot;
    const unsigned owner_mask = __ballot_sync(0xffffffffu, base <= kk && kk < inc);
    const int owner = __ffs(owner_mask) - 1;      // exactly one lane (kk < total)
    int sel = 0;
    unsigned excl = 0, c_sel = 0;
    if (lane == owner) {
        unsigned run = base;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            if (run <= kk && kk < run + cnt[j]) { sel = 8 * lane + j; excl = run; c_sel = cnt[j]; }
            run += cnt[j];
        }
    }
    sel = __shfl_sync(0xffffffffu, sel, owner);
    excl = __shfl_sync(0xffffffffu, excl, owner);
    c_sel = __shfl_sync(0xffffffffu, c_sel, owner);
    int nb2 = sel;
    unsigned total = c_sel;
    if (need_next && kk + 1 >= excl + c_sel) {     // rank kk+1 is the smallest value of the next non-empty bucket
        int mine = 1 << 20;
        unsigned mine_c = 0;
#pragma unroll
        for (int j = 7; j >= 0; --j)
            if (8 * lane + j > sel && cnt[j] > 0) { mine = 8 * lane + j; mine_c = cnt[j]; }
        int best = mine;
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) best = min(best, __shfl_xor_sync(0xffffffffu, best, off));
        const unsigned who = __ballot_sync(0xffffffffu, mine == best && best < (1 << 20));
        if (who) {
            nb2 = best;
            total += __shfl_sync(0xffffffffu, mine_c, __ffs(who) - 1);
        } else {
            total = 0xFFFFFFFFu; // cannot happen for kk+1 < len; treated as a failure
        }
    }
    if (lane == 0) {
        sm.sel[c] = sel; sm.nb2[c] = nb2; sm.excl[c] = excl; sm.cnt[c] = total;
        if (total > (unsigned)kFastListCap) sm.fail = 1;
    }
}

__device__ __forceinline__ unsigned atom_shared_inc(unsigned addr) { // one ATOMS, no compiler-side warp aggregation
    unsigned old;
    asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(addr) : "memory");
    return old;
}

// Copy the values whose packed bucket byte equals `sel` (or `nb2`) to list[].  Per 4-value word one XOR and the
// zero-byte test (x − 0x01010101) & ~x & 0x80808080; only words with a hit (≈ 4 % of them) do more.
template <int EPT>
__device__ __forceinline__ void fast_gather(const float (&v)[EPT], const unsigned (&idx)[(EPT + 3) / 4], int sel, int nb2,
                                            float* list, unsigned list_n_addr) {
    const unsigned s4 = (unsigned)sel * 0x01010101u, n4 = (unsigned)nb2 * 0x01010101u;
    const bool two = nb2 != sel;
#pragma unroll
    for (int q = 0; q < (EPT + 3) / 4; ++q) {
        const unsigned x = idx[q] ^ s4;
        unsigned has = (x - 0x01010101u) & ~x & 0x80808080u;
        if (two) {
            const unsigned y = idx[q] ^ n4;
            has |= (y - 0x01010101u) & ~y & 0x80808080u;
        }
        while (has) {                                   // lowest flagged byte is always a true match
            const int j = (__ffs(has) - 1) >> 3;
            has &= has - 1;
            const unsigned byte = (idx[q] >> (8 * j)) & 0xFFu;
            if (byte != (unsigned)sel && byte != (unsigned)nb2) continue;   // borrow artefact above a true match
            float val = v[4 * q];
            if (4 * q + 1 < EPT && j == 1) val = v[4 * q + 1];
            if (4 * q + 2 < EPT && j == 2) val = v[4 * q + 2];
            if (4 * q + 3 < EPT && j == 3) val = v[4 * q + 3];
            const unsigned slot = atom_shared_inc(list_n_addr);
            if (slot < (unsigned)kFastListCap) list[slot] = val;
        }
    }
}

// Threads [0, NT/2) rank the members of component 0, threads [NT/2, NT) those of component 1 (NT/2 ≥ kFastListCap).
// The value of rank r is max{x : #{y < x} ≤ r}; each member counts the members below it and the qualifying ones
// race with atomicMax on the order-preserving key of the float.  res_key[c][0..1] must be 0 on entry.
__device__ __forceinline__ void fast_rank(FastSmem& sm, int c, int t, unsigned kk, int phase) {
    const unsigned cnt = sm.cnt[c];
    if ((unsigned)t < cnt) {
        const float x = sm.list[c][t];
        unsigned below = 0;
        for (unsigned j = 0; j < cnt; ++j) below += (sm.list[c][j] < x) ? 1u : 0u;
        const unsigned target = kk - sm.excl[c];
        const unsigned key = float_key(x);
        if (below <= target) atomicMax(&sm.res_key[phase][c][0], key);
        if (below <= target + 1) atomicMax(&sm.res_key[phase][c][1], key);
    }
}

__device__ __forceinline__ float key_float(unsigned k) {
    return __uint_as_float(k ^ ((k >> 31) ? 0x80000000u : 0xFFFFFFFFu));
}

template <int EPT, int NT>
__global__ void __launch_bounds__(NT)
norm_power_fast_kernel(const float2* __restrict__ spectra, long long pitch_in, int blocks_per_row,
                       float* __restrict__ P, long long pitchP, unsigned* __restrict__ redo,
                       unsigned* __restrict__ redo_count) {
    static_assert(NT >= 2 * kFastListCap && NT % 64 == 0, "rank phase maps one thread per member per component");
    constexpr int B = EPT * NT;
    constexpr int NQ = (EPT + 3) / 4;
    constexpr bool kEven = (B & 1) == 0;
    constexpr unsigned kRank = (unsigned)((B - 1) >> 1);
    __shared__ __align__(16) FastSmem sm;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long row = blockIdx.x / blocks_per_row;
    const long long lo_bin = (long long)(blockIdx.x % blocks_per_row) * B;
    const float2* src = spectra + row * pitch_in + lo_bin;

    float v[2][EPT];
    unsigned idx[2][NQ];
    float vmin[2] = {INFINITY, INFINITY}, vmax[2] = {-INFINITY, -INFINITY};
#pragma unroll
    for (int r = 0; r < EPT; ++r) {
        const float2 z = __ldg(src + tid + r * NT);
        v[0][r] = z.x; v[1][r] = z.y;
    }
#pragma unroll
    for (int r = 0; r < EPT; ++r) {
        vmin[0] = fminf(vmin[0], v[0][r]); vmax[0] = fmaxf(vmax[0], v[0][r]);
        vmin[1] = fminf(vmin[1], v[1][r]); vmax[1] = fmaxf(vmax[1], v[1][r]);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            vmin[c] = fminf(vmin[c], __shfl_xor_sync(0xffffffffu, vmin[c], off));
            vmax[c] = fmaxf(vmax[c], __shfl_xor_sync(0xffffffffu, vmax[c], off));
        }
    }
    // zero the four histograms and the counters; publish the warp extrema
    for (int i = tid; i < 4 * kSelBuckets; i += NT) (&sm.hist[0][0][0])[i] = 0;
    if (tid < 4) (&sm.list_n[0][0])[tid] = 0;
    if (tid < 8) (&sm.res_key[0][0][0])[tid] = 0;
    if (tid == 0) sm.fail = 0;
    if (lane == 0) {
        sm.wmin[0][warp] = vmin[0]; sm.wmax[0][warp] = vmax[0];
        sm.wmin[1][warp] = vmin[1]; sm.wmax[1][warp] = vmax[1];
    }
    __syncthreads();                                                                     // S1
    float lo[2], hi[2], scale[2];
    bool bad = false;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        float a = sm.wmin[c][0], b = sm.wmax[c][0];
#pragma unroll
        for (int w = 1; w < NT / 32; ++w) { a = fminf(a, sm.wmin[c][w]); b = fmaxf(b, sm.wmax[c][w]); }
        lo[c] = a; hi[c] = b;
        const float width = b - a;
        scale[c] = 255.0f / width;
        bad = bad || !(width > 0.f) || !isfinite(width) || !isfinite(scale[c]);
    }
    float inv[2] = {0.f, 0.f};
    if (!bad) {
        // ---------------- median of each component
#pragma unroll
        for (int c = 0; c < 2; ++c) fast_hist<EPT, true>(v[c], lo[c], scale[c], smem_addr(&sm.hist[0][c][0]), idx[c]);
        __syncthreads();                                                                 // S2
        if (warp < 2) fast_scan(&sm.hist[0][warp][0], kRank, kEven, sm, warp);
        __syncthreads();                                                                 // S3
        bad = sm.fail != 0;
    }
    if (!bad) {
#pragma unroll
        for (int c = 0; c < 2; ++c) fast_gather<EPT>(v[c], idx[c], sm.sel[c], sm.nb2[c], sm.list[c], smem_addr(&sm.list_n[0][c]));
        __syncthreads();                                                                 // S4
        fast_rank(sm, tid >= NT / 2, tid & (NT / 2 - 1), kRank, 0);
        __syncthreads();                                                                 // S5
        // ---------------- |v − median| and its median (the MAD)
        float dscale[2];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const float a = key_float(sm.res_key[0][c][0]), b = kEven ? key_float(sm.res_key[0][c][1]) : a;
            const float h = 0.5f * __fsub_rn(b, a);
#pragma unroll
            for (int r = 0; r < EPT; ++r) v[c][r] = fabsf(__fsub_rn(__fsub_rn(v[c][r], a), h));
            const float dmax = fmaxf(hi[c] - a, b - lo[c]) * 1.000001f;   // ≥ every |v − m|
            dscale[c] = 255.0f / dmax;
            bad = bad || !(dmax > 0.f) || !isfinite(dmax) || !isfinite(dscale[c]);
        }
        if (!bad) {
#pragma unroll
            for (int c = 0; c < 2; ++c) fast_hist<EPT, false>(v[c], 0.f, dscale[c], smem_addr(&sm.hist[1][c][0]), idx[c]);
        }
        __syncthreads();                                                                 // S6
        if (!bad && warp < 2) fast_scan(&sm.hist[1][warp][0], kRank, kEven, sm, warp);
        __syncthreads();                                                                 // S7
        bad = bad || sm.fail != 0;
    }
    if (!bad) {
#pragma unroll
        for (int c = 0; c < 2; ++c) fast_gather<EPT>(v[c], idx[c], sm.sel[c], sm.nb2[c], sm.list[c], smem_addr(&sm.list_n[1][c]));
        __syncthreads();                                                                 // S8
        fast_rank(sm, tid >= NT / 2, tid & (NT / 2 - 1), kRank, 1);
        __syncthreads();                                                                 // S9
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const float a = key_float(sm.res_key[1][c][0]), b = kEven ? key_float(sm.res_key[1][c][1]) : a;
            const double s = kKappa * (0.5 * ((double)a + (double)b));
            inv[c] = (s > 0.0 && isfinite(s)) ? (float)(0.70710678118654752440 / s) : 0.f;
        }
        float* dst = P + row * pitchP + lo_bin;
#pragma unroll
        for (int r = 0; r < EPT; ++r) {
            const float x = v[0][r] * inv[0], y = v[1][r] * inv[1];
            dst[tid + r * NT] = fmaf(x, x, y * y);
        }
    } else if (tid == 0) {
        redo[atomicAdd(redo_count, 1u)] = blockIdx.x;   // the general path will do this block
    }
}

} // namespace pulscan
