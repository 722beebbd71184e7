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

// Threads per CTA / resident CTAs per SM.  Two CTAs of 512 threads let one block's barrier-separated set-up (prefix build, ln p
// of the passing widths) overlap another block's window sums.  Measured on a B200, kernel (c) ms at cfg 2 / 3 / 4 / 5:
// 1024 x 1: 0.058 / 0.065 / 0.209 / 0.061; 512 x 2: 0.055 / 0.062 / 0.196 / 0.057; 512 x 1: 0.053 / 0.061 / 0.215 / 0.055;
// 256 x 4: 0.053 / 0.061 / 0.243 / 0.055.
#ifndef PULSCAN_EXACT_THREADS
#define PULSCAN_EXACT_THREADS 512
#endif
#ifndef PULSCAN_EXACT_MIN_CTAS
#define PULSCAN_EXACT_MIN_CTAS 2
#endif
constexpr int kExactThreads = PULSCAN_EXACT_THREADS;

struct alignas(16) ExactSmemHdr {   // the prefix array behind it is read with 16-byte loads
    double part[kExactThreads];   // per-thread chunk sums for the prefix scan
    double list_s[kExactThreads]; // widths of the current step whose maximum reaches T_w: (maximum, width, arg-max)
    int list_w[kExactThreads];
    int list_i[kExactThreads];
    unsigned nlist[2];
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

// Partial result of one part of a block (see `parts` below): the best width among the rounds that part evaluated.
struct alignas(8) ExactPartial {
    double lnp, s;
    int w, i;
};

// lg_split: the start bins of a block are cut into 2^lg_split chunks handled by adjacent lanes, so that zmax·2^lg_split
// (width, chunk) pairs keep all kExactThreads threads busy when zmax is small and balance the rounds when it is large (host choice).
// parts > 1 (large zmax): the rounds of widths of one block are dealt to `parts` CTAs (each rebuilds the block's prefix sum),
// their partial arg-minima meet in `partial` and the CTA that arrives last (`done` counter) reduces and emits — a few
// hundred marked blocks then occupy the whole GPU instead of one CTA each.  Only the first `split_slots` marked blocks are
// split (the size of `partial` / `done`); the rest is evaluated by one CTA per block.
// seg < C (long candidate blocks, e.g. the paper's R-Block width 32768, L224): the block's start bins are walked in segments of
// `seg` bins, each with its own prefix sum (+ zmax halo) in shared memory; the running maximum and arg-max of every width are
// carried from segment to segment in shared memory behind the prefix array (a width always belongs to the same thread), a
// later segment replaces them on `>` only (R14: the lowest bin wins ties), and ln p is evaluated after the last segment.
__global__ void __launch_bounds__(kExactThreads, PULSCAN_EXACT_MIN_CTAS)
block_exact_kernel(const PowerSource src_pw, long long n, int zmax, int C, long long nblk,
                   const double* __restrict__ T_g, double ln_trials, double lnp_thr, int r_block, int shape_mult, int signif_mode, int numharm,
                   pulscan_hcandidate* __restrict__ out_h, int per_width, unsigned capacity, int lg_split, int parts, int seg,
                   unsigned split_slots, ExactPartial* __restrict__ partial, unsigned* __restrict__ done,
                   const unsigned* __restrict__ flagged, const unsigned* __restrict__ counters,
                   pulscan_candidate* __restrict__ out, unsigned* __restrict__ out_count) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    ExactSmemHdr& hdr = *reinterpret_cast<ExactSmemHdr*>(smem_raw);
    double* pre = reinterpret_cast<double*>(smem_raw + sizeof(ExactSmemHdr)); // [L + 1], L ≤ min(C, seg) + zmax − 1
    const int Cs = min(C, seg);                                                 // start bins per segment
    double* carry_s = pre + ((Cs + zmax + 2) & ~1);                             // [zmax + 1], only when seg < C
    int* carry_i = reinterpret_cast<int*>(carry_s + zmax + 1);                  // [zmax + 1]
    const int tid = threadIdx.x, lane = tid & 31;
    const unsigned nflag = counters[0];
    if (tid == 0) { hdr.nlist[0] = 0; hdr.nlist[1] = 0; }
    __syncthreads();
    const int nsplit = 1 << lg_split, piece = tid & (nsplit - 1), w_per_round = kExactThreads >> lg_split;
    // start bins per chunk: even (16-byte loads of pairs of doubles), and ≡ 2 (mod 4) when there are several chunks, so that
    // the chunks' 16-byte loads of a warp (lanes of a chunk 32 bytes apart) interleave on the banks: 4 wavefronts per 512 bytes
    int cs = (Cs + nsplit - 1) >> lg_split;
    if (nsplit >= 2) cs += (2 - cs) & 3;

    const unsigned n_split = parts > 1 ? min(nflag, split_slots) : 0u;
    const unsigned n_items = n_split * (unsigned)parts + (nflag - n_split);
    for (unsigned item = blockIdx.x; item < n_items; item += gridDim.x) {
        const bool split = item < n_split * (unsigned)parts;
        const unsigned e = split ? item / (unsigned)parts : n_split + (item - n_split * (unsigned)parts);
        const int part = split ? (int)(item % (unsigned)parts) : 0, nparts = split ? parts : 1;
        const unsigned gid = flagged[e];
        const long long row = gid / nblk;
        const long long c = gid % nblk;
        const long long lo = c * C;
        long long hi = lo + C;
        if (hi > n) hi = n;
        const int nstart_all = (int)(hi - lo);
        const int nseg = (nstart_all + Cs - 1) / Cs;
        double my_lnp = INFINITY, my_s = 0.0;
        int my_w = 0, my_i = 0;
        for (int sg = 0; sg < nseg; ++sg) {
        const bool last_seg = sg == nseg - 1;
        const int seg_off = sg * Cs;                // first start bin of this segment, relative to the block
        const long long slo = lo + seg_off;
        const int nstart = min(Cs, nstart_all - seg_off);
        long long end = slo + nstart + zmax - 1;    // last bin any window of the segment can touch, exclusive
        if (end > n) end = n;
        const int L = (int)(end - slo);
        if (tid == 0) { hdr.nlist[0] = 0; hdr.nlist[1] = 0; }   // (barriers of the prefix build separate this from the first use)

        // double-precision prefix sum pre[j] = Σ_{t<j} P[lo+t]: coalesced loads (or rebuilds, power_source.cuh) into
        // pre[j+1], each thread then scans its own chunk in place and the chunk totals are scanned by one warp
        {
            PowerSource::Row src(src_pw, row);
            for (int j = tid; j < L; j += kExactThreads) pre[j + 1] = (double)src(slo + j);
            if (tid == 0) pre[0] = 0.0;
        }
        __syncthreads();
        const int chunk = (L + kExactThreads - 1) / kExactThreads;
        const int a = min(tid * chunk, L), b = min(a + chunk, L);
        {
            double run = 0.0;
            for (int j = a; j < b; ++j) { run += pre[j + 1]; pre[j + 1] = run; }
            hdr.part[tid] = run;
        }
        __syncthreads();
        if (tid < 32) { // exclusive scan of the kExactThreads chunk sums by one warp, kExactThreads/32 each
            double run = 0.0;
            for (int q = 0; q < kExactThreads / 32; ++q) { const double v = hdr.part[tid * (kExactThreads / 32) + q]; hdr.part[tid * (kExactThreads / 32) + q] = run; run += v; }
            double inc = run;
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                const double t = __shfl_up_sync(0xffffffffu, inc, off);
                if (tid >= off) inc += t;
            }
            const double base = inc - run;
            for (int q = 0; q < kExactThreads / 32; ++q) hdr.part[tid * (kExactThreads / 32) + q] += base;
        }
        __syncthreads();
        {
            const double base = hdr.part[tid];
            for (int j = a; j < b; ++j) pre[j + 1] += base;
        }
        __syncthreads();

        // (four consecutive widths, chunk of start bins) per thread.  A 4 × 4 register tile — starts i..i+3, widths W4..W4+3 —
        // needs pre[i..i+3] and pre[i+W4 .. i+W4+6]: 6 shared-memory loads for 16 window sums instead of 32 (the kernel is
        // bound by the rate of LDS instructions).  Per width the maximum and its lowest arg-max (strict >, ascending starts:
        // R14), combined over the chunks of a width by shuffles (adjacent lanes, the lower chunk holds the lower bins).
        int rnd = 0;                                        // which of the two list counters this round uses
        const int nquads = zmax / 4 + 1;                    // width quads {4q, …, 4q+3}; width 0 does not exist
        for (int q0 = part * w_per_round; q0 < nquads; q0 += nparts * w_per_round) {
            const int W4 = 4 * (q0 + (tid >> lg_split));
            double best[4] = {-1.0, -1.0, -1.0, -1.0};
            int arg[4] = {-1, -1, -1, -1};
            if (W4 <= zmax) {
                const int lo_i = piece * cs, hi_i = lo_i + cs;
                const int full_end = min(hi_i, min(nstart, L - (W4 + 3) + 1));   // all four widths exist for starts below this
                int i = lo_i;
                for (; i + 4 <= full_end; i += 4) {
                    const double2 p01 = *reinterpret_cast<const double2*>(pre + i), p23 = *reinterpret_cast<const double2*>(pre + i + 2);
                    const double* pj = pre + i + W4;
                    const double2 j01 = *reinterpret_cast<const double2*>(pj), j23 = *reinterpret_cast<const double2*>(pj + 2),
                                  j45 = *reinterpret_cast<const double2*>(pj + 4);
                    const double pi[4] = {p01.x, p01.y, p23.x, p23.y};
                    const double jv[7] = {j01.x, j01.y, j23.x, j23.y, j45.x, j45.y, pj[6]};
#pragma unroll
                    for (int a4 = 0; a4 < 4; ++a4)
#pragma unroll
                        for (int b4 = 0; b4 < 4; ++b4) {
                            const double v = jv[a4 + b4] - pi[a4];
                            if (v > best[b4]) { best[b4] = v; arg[b4] = i + a4; }
                        }
                }
#pragma unroll
                for (int b4 = 0; b4 < 4; ++b4) {            // the starts that only some of the four widths have
                    const int w = W4 + b4;
                    const int i1 = min(hi_i, min(nstart, L - w + 1));
                    for (int t = i; t < i1; ++t) {
                        const double v = pre[t + w] - pre[t];
                        if (v > best[b4]) { best[b4] = v; arg[b4] = t; }
                    }
                    if (w < 1 || w > zmax) { best[b4] = -1.0; arg[b4] = -1; }
                }
            }
#pragma unroll
            for (int b4 = 0; b4 < 4; ++b4, rnd ^= 1) {         // one of the thread's four widths per step (the list holds 1024)
                for (int off = 1; off < nsplit; off <<= 1) {   // lanes piece, piece^off: the lower piece holds the lower bins
                    const double ob = __shfl_xor_sync(0xffffffffu, best[b4], off);
                    const int oa = __shfl_xor_sync(0xffffffffu, arg[b4], off);
                    const bool other_lower = (piece & off) != 0;
                    if (ob > best[b4] || (ob == best[b4] && other_lower && oa >= 0)) { best[b4] = ob; arg[b4] = oa; }
                }
                // The widths whose maximum reaches T_w are collected and their ln p evaluated by all threads: the series of
                // ln Q is a serial loop of up to w terms, and only one lane in 2^lg_split holds a width after the reduction.
                const int w = W4 + b4;
                if (nseg > 1) {                                // long block: merge with the segments before, hand on to the next
                    if (piece == 0 && w >= 1 && w <= zmax) {
                        if (arg[b4] >= 0) arg[b4] += seg_off;  // relative to the block from here on
                        if (sg > 0) {
                            const double cb = carry_s[w];
                            if (!(best[b4] > cb)) { best[b4] = cb; arg[b4] = carry_i[w]; }
                        }
                        if (!last_seg) { carry_s[w] = best[b4]; carry_i[w] = arg[b4]; }
                    }
                    if (!last_seg) continue;                   // (uniform over the CTA) ln p after the last segment only
                }
                if (piece == 0 && arg[b4] >= 0 && best[b4] >= T_g[w - 1] * (1.0 - 1e-9)) {
                    const unsigned slot = atomicAdd(&hdr.nlist[rnd], 1u);
                    hdr.list_s[slot] = best[b4]; hdr.list_w[slot] = w; hdr.list_i[slot] = arg[b4];
                }
                __syncthreads();
                const int nl = (int)hdr.nlist[rnd];
                if (tid == 0) hdr.nlist[rnd ^ 1] = 0;
                for (int idx = tid; idx < nl; idx += kExactThreads) {
                    const int lw = hdr.list_w[idx], li = hdr.list_i[idx];
                    const double ls = hdr.list_s[idx];
                    // harmonic-summed spectra: χ² with H(H+1)·w d.o.f. (L220); signif_mode 1: Alg. 3's polynomial instead of the tail
                    double lnp = lnp_of(signif_mode, lw * shape_mult, ls) + ln_trials;
                    if (lnp > 0.0) lnp = 0.0;
                    if (per_width) {   // the paper's GPU output: one candidate per (block, searched width) above the threshold (Alg. 4)
                        if (lnp <= lnp_thr)
                            emit_candidate(row, r_block ? (int32_t)lo : (int32_t)(lo + li), lw, ls, lnp, numharm, out, out_h, out_count, capacity);
                    } else if (lnp < my_lnp || (lnp == my_lnp && lw < my_w)) { my_lnp = lnp; my_w = lw; my_i = li; my_s = ls; }   // ties keep the smaller width
                }
                __syncthreads();
            }
        }
        __syncthreads();                                    // the next segment overwrites the prefix array
        }   // segments
        // block arg-min over (ln p, w)
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            const double ol = __shfl_xor_sync(0xffffffffu, my_lnp, off);
            const int ow = __shfl_xor_sync(0xffffffffu, my_w, off);
            const int oi = __shfl_xor_sync(0xffffffffu, my_i, off);
            const double os = __shfl_xor_sync(0xffffffffu, my_s, off);
            if (ol < my_lnp || (ol == my_lnp && ow != 0 && (my_w == 0 || ow < my_w))) { my_lnp = ol; my_w = ow; my_i = oi; my_s = os; }
        }
        if (lane == 0) {
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
            if (nparts > 1 && !per_width) {      // meet the other parts of this block; the last one to arrive finishes the job
                ExactPartial* slot = partial + (size_t)e * parts;
                slot[part] = ExactPartial{my_lnp, my_s, my_w, my_i};
                __threadfence();
                if (atomicAdd(done + e, 1u) != (unsigned)(parts - 1)) my_w = 0;
                else {
                    __threadfence();
                    for (int q = 0; q < parts; ++q) {
                        if (q == part) continue;
                        const double ol = __ldcg(&slot[q].lnp);
                        const int ow = __ldcg(&slot[q].w);
                        if (ol < my_lnp || (ol == my_lnp && ow != 0 && (my_w == 0 || ow < my_w))) {
                            my_lnp = ol; my_w = ow; my_i = __ldcg(&slot[q].i); my_s = __ldcg(&slot[q].s);
                        }
                    }
                }
            }
            if (my_w > 0 && my_lnp <= lnp_thr)   // R-Block: block index × block width (L222-226)
                emit_candidate(row, r_block ? (int32_t)lo : (int32_t)(lo + my_i), my_w, my_s, my_lnp, numharm, out, out_h, out_count, capacity);
        }
        __syncthreads();
    }
}

} // namespace pulscan
