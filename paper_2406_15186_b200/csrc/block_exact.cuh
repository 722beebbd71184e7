// block_exact.cuh — kernel (c): exact evaluation of the candidate blocks marked by the sweep, significance,
// threshold and compaction.
//
// For a marked block c of spectrum b this is PAPER.md's definition written out in double precision:
//   S(i,w) for every start bin i of the block and every width w ≤ zmax with i + w ≤ n   (L169-199; R11, R12)
//   M(c,w) = max_i S(i,w), I(c,w) = lowest arg-max                                      (Alg. 4; R14)
//   ln p(c,w) = ln Q(w, M) + ln n_trials, clamped to ≤ 0                                 (L154-158 Eq. 9; R15)
//   w* = width with the smallest ln p (largest σ), smallest w on ties                   (R13)
//   emit (b, I, w*, M, σ) iff ln p ≤ ln sf(σ_threshold)                                  (L342-344, L361; R17)
// S(i,w) = pre[i+w] − pre[i] from a double-precision prefix sum of the block's powers (+ zmax halo) held in shared
// memory; one thread owns one width and walks the block's start bins, so maxima need no cross-thread reduction.
// Only widths whose maximum reaches T_w·(1−1e-9) have their ln Q evaluated: the others cannot be emitted, and if one
// of them were the arg-min of ln p nothing would be emitted for the block at all.
// Records are appended with one atomicAdd per block (at most one record per block: contention is negligible).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/pulscan.h"
#include "power_source.cuh"
#include "significance.cuh"

namespace pulscan {

constexpr int kExactThreads = 512;

struct ExactSmemHdr {
    double part[kExactThreads];   // per-thread chunk sums for the prefix scan
    double best_lnp[kExactThreads / 32];
    int best_w[kExactThreads / 32];
    int best_i[kExactThreads / 32];
    double best_s[kExactThreads / 32];
};

// Append one record (20-byte or, for the harmonic search, 24-byte); records beyond `capacity` are counted, not written.
__device__ __forceinline__ void emit_candidate(long long row, int32_t bin, int w, double S, double lnp, int numharm,
                                               pulscan_candidate* __restrict__ out, pulscan_hcandidate* __restrict__ out_h,
                                               unsigned* __restrict__ out_count, unsigned capacity) {
    const float sigma = (float)sigma_from_lnp(lnp);
    const unsigned slot = atomicAdd(out_count, 1u);
    if (slot >= capacity) return;
    if (out_h) {
        pulscan_hcandidate r;
        r.spectrum = (int32_t)row; r.bin = bin; r.width = w; r.numharm = numharm;
        r.power = (float)S; r.sigma = sigma;
        out_h[slot] = r;
    } else {
        pulscan_candidate r;
        r.spectrum = (int32_t)row; r.bin = bin; r.width = w;
        r.power = (float)S; r.sigma = sigma;
        out[slot] = r;
    }
}

__global__ void __launch_bounds__(kExactThreads)
block_exact_kernel(const PowerSource src_pw, long long n, int zmax, int C, long long nblk,
                   const double* __restrict__ T_g, double ln_trials, double lnp_thr, int r_block, int shape_mult, int signif_mode, int numharm,
                   pulscan_hcandidate* __restrict__ out_h, int per_width, unsigned capacity,
                   const unsigned* __restrict__ flagged, const unsigned* __restrict__ counters,
                   pulscan_candidate* __restrict__ out, unsigned* __restrict__ out_count) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    ExactSmemHdr& hdr = *reinterpret_cast<ExactSmemHdr*>(smem_raw);
    double* pre = reinterpret_cast<double*>(smem_raw + sizeof(ExactSmemHdr)); // [L + 1]
    const int tid = threadIdx.x;
    const unsigned nflag = counters[0];

    for (unsigned e = blockIdx.x; e < nflag; e += gridDim.x) {
        const unsigned gid = flagged[e];
        const long long row = gid / nblk;
        const long long c = gid % nblk;
        const long long lo = c * C;
        long long hi = lo + C;
        if (hi > n) hi = n;
        const int nstart = (int)(hi - lo);
        long long end = hi + zmax - 1;              // last bin any window of the block can touch, exclusive: hi−1+zmax
        if (end > n) end = n;
        const int L = (int)(end - lo);
        PowerSource::Row src(src_pw, row);

        // double-precision exclusive prefix sum: pre[j] = Σ_{t<j} P[lo+t]
        const int chunk = (L + kExactThreads - 1) / kExactThreads;
        const int a = tid * chunk;
        const int b = min(a + chunk, L);
        double s = 0.0;
        for (int j = a; j < b; ++j) s += (double)src(lo + j);
        hdr.part[tid] = s;
        __syncthreads();
        if (tid < 32) { // scan of the 512 chunk sums by one warp, 16 each
            double run = 0.0;
            double loc[kExactThreads / 32];
#pragma unroll
            for (int q = 0; q < kExactThreads / 32; ++q) { loc[q] = run; run += hdr.part[tid * (kExactThreads / 32) + q]; }
            double inc = run;
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                double t = __shfl_up_sync(0xffffffffu, inc, off);
                if (tid >= off) inc += t;
            }
            const double base = inc - run;
#pragma unroll
            for (int q = 0; q < kExactThreads / 32; ++q) hdr.part[tid * (kExactThreads / 32) + q] = base + loc[q];
        }
        __syncthreads();
        {
            double run = hdr.part[tid];
            for (int j = a; j < b; ++j) { pre[j] = run; run += (double)src(lo + j); }
            if (b == L && a < L) pre[L] = run;
            if (L == 0 && tid == 0) pre[0] = 0.0;
        }
        __syncthreads();

        // one width per thread: maximum over the block's start bins, then ln p where it can matter
        double my_lnp = INFINITY, my_s = 0.0;
        int my_w = 0, my_i = 0;
        for (int w = tid + 1; w <= zmax; w += kExactThreads) {
            const int imax = min(nstart, L - w + 1);   // starts i with i + w ≤ L
            double best = -1.0;
            int arg = -1;
            for (int i = 0; i < imax; ++i) {
                const double v = pre[i + w] - pre[i];
                if (v > best) { best = v; arg = i; }
            }
            if (arg >= 0 && best >= T_g[w - 1] * (1.0 - 1e-9)) {
                // harmonic-summed spectra: χ² with H(H+1)·w d.o.f. (L220); signif_mode 1: Alg. 3's polynomial instead of the tail
                double lnp = lnp_of(signif_mode, w * shape_mult, best) + ln_trials;
                if (lnp > 0.0) lnp = 0.0;
                if (per_width) {   // the paper's GPU output: one candidate per (block, searched width) above the threshold (Alg. 4)
                    if (lnp <= lnp_thr)
                        emit_candidate(row, r_block ? (int32_t)lo : (int32_t)(lo + arg), w, best, lnp, numharm, out, out_h, out_count, capacity);
                } else if (lnp < my_lnp) { my_lnp = lnp; my_w = w; my_i = arg; my_s = best; } // ascending w: ties keep the smaller
            }
        }
        // block arg-min over (ln p, w)
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            const double ol = __shfl_xor_sync(0xffffffffu, my_lnp, off);
            const int ow = __shfl_xor_sync(0xffffffffu, my_w, off);
            const int oi = __shfl_xor_sync(0xffffffffu, my_i, off);
            const double os = __shfl_xor_sync(0xffffffffu, my_s, off);
            if (ol < my_lnp || (ol == my_lnp && ow != 0 && (my_w == 0 || ow < my_w))) { my_lnp = ol; my_w = ow; my_i = oi; my_s = os; }
        }
        if ((tid & 31) == 0) {
            hdr.best_lnp[tid >> 5] = my_lnp; hdr.best_w[tid >> 5] = my_w; hdr.best_i[tid >> 5] = my_i; hdr.best_s[tid >> 5] = my_s;
        }
        __syncthreads();
        if (tid == 0) {
            for (int q = 1; q < kExactThreads / 32; ++q) {
                const double ol = hdr.best_lnp[q];
                const int ow = hdr.best_w[q];
                if (ol < my_lnp || (ol == my_lnp && ow != 0 && (my_w == 0 || ow < my_w))) {
                    my_lnp = ol; my_w = ow; my_i = hdr.best_i[q]; my_s = hdr.best_s[q];
                }
            }
            if (my_w > 0 && my_lnp <= lnp_thr)   // R-Block: block index × block width (L222-226)
                emit_candidate(row, r_block ? (int32_t)lo : (int32_t)(lo + my_i), my_w, my_s, my_lnp, numharm, out, out_h, out_count, capacity);
        }
        __syncthreads();
    }
}

} // namespace pulscan
