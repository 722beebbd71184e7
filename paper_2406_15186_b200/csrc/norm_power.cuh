// norm_power.cuh — kernel (a): per-block, per-component exact median/MAD normalisation fused with the power.
//
// PAPER.md:L140-150 (§2.2.3, Eq. 8): each component (re, im) of each block is normalised independently as
// (v − median)/(κ·MAD); then P = |X'|² (halved here so that noise has mean 1, R2).  The paper's CPU code
// finds the medians with Quickselect (L230) and its GPU code approximates them by median-of-medians (Alg. 1);
// this kernel is exact and built for the SM: one CTA per normalisation block, the block's values live in registers
// (EPT per thread per component, loaded once with coalesced 8-byte loads), and each order statistic is found by a
// histogram select: 256 value-linear buckets between the block's min and max (one shared-memory atomic per value),
// a CTA scan to find the bucket holding rank k, then an exact rank count among that bucket's few dozen members.
// A bucket that is still too full is re-bucketed over its own [min, max] until it fits; ranges that float32 cannot
// bucket linearly fall back to the order-preserving integer key of the float.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace pulscan {

constexpr int kSelBuckets = 256;
constexpr int kSelListCap = 1024;
constexpr double kKappa = 1.4826022185056018; // 1/Φ⁻¹(3/4), PAPER.md:L142 (Alg. 1 L648 prints 1.4826)

struct SelectSmem {
    unsigned hist[kSelBuckets];
    float list[kSelListCap];
    float red_a[32];
    float red_b[32];
    unsigned warp_tot[8];
    int sel_bucket;
    unsigned sel_excl;
    unsigned sel_count;
    unsigned list_n;
    float out_k;
    float out_next;
};

__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ unsigned float_key(float v) {
    unsigned b = __float_as_uint(v);
    return b ^ ((b >> 31) ? 0xFFFFFFFFu : 0x80000000u);
}

// ---------------------------------------------------------------------------------------------------------------
// What kernel (a) leaves behind for the rest of the search.  Either (or both) of:
//   P  float32 [batch][pitchP]: the normalised power of every bin (pulscan_normalise_power, the exhaustive sweep, the
//      full-resolution sweep of very low thresholds, the harmonic sum);
//   G  float32 [batch][pitchG]: G[k] = (P[4k] + P[4k+1]) + (P[4k+2] + P[4k+3]), the sums of aligned groups of four bins
//      (zeros beyond n_bins) — all the streaming sweep needs, a quarter of the bytes — together with
//   stats float32 [batch][nb][8]: per normalisation block (a, inv, k) of the real and of the imaginary parts, from which
//      any bin's power is rebuilt bit-identically by norm_power_value() wherever a flagged span needs it.
struct NormOut {
    float* P;            // may be null
    long long pitchP;
    float* G;            // may be null; needs B % 4 == 0
    long long pitchG;
    float* stats;        // null iff G is null
};

// The normalised power of one bin.  x' = ((v − a) − h)·inv is evaluated as fma(v − a, inv, k), k = −h·inv, and
// P = fma(x', x', y'·y'); every kernel that produces or rebuilds a power goes through this function.
__device__ __forceinline__ float norm_power_value(float2 z, float a0, float i0, float k0, float a1, float i1, float k1) {
    const float x = __fmaf_rn(__fsub_rn(z.x, a0), i0, k0), y = __fmaf_rn(__fsub_rn(z.y, a1), i1, k1);
    return __fmaf_rn(x, x, __fmul_rn(y, y));
}

// Quad sums of four rounds of powers: p0..p3 belong to bins lane_bin + (r0 + q)·NT, q = 0..3, where the four lanes
// 4j..4j+3 of a warp hold four consecutive bins of an aligned group.  A transposing butterfly (3 shuffles for 4 sums)
// leaves in lane 4j + q the sum of round r0 + q, always added as (p[0] + p[1]) + (p[2] + p[3]) up to commutation.
__device__ __forceinline__ float quad_sums4(float p0, float p1, float p2, float p3) {
    const int q = threadIdx.x & 3;
    float a = (q & 1) ? p1 : p0;
    const float b = (q & 1) ? p0 : p1;
    a += __shfl_xor_sync(0xffffffffu, b, 1);
    float c = (q & 1) ? p3 : p2;
    const float d = (q & 1) ? p2 : p3;
    c += __shfl_xor_sync(0xffffffffu, d, 1);
    float e = (q & 2) ? c : a;
    const float f = (q & 2) ? a : c;
    e += __shfl_xor_sync(0xffffffffu, f, 2);
    return e;
}

// One round only (block lengths that are not a multiple of 4·NT): every lane of a group ends up with the group's sum.
__device__ __forceinline__ float quad_sum1(float p) {
    p += __shfl_xor_sync(0xffffffffu, p, 1);
    p += __shfl_xor_sync(0xffffffffu, p, 2);
    return p;
}

// Monotone non-decreasing map of a value in [lo, hi] to a bucket in [0, 255].  Explicit round-to-nearest
// intrinsics: the histogram pass and the gather pass must compute the same bucket, so no FMA contraction.
struct BucketMap {
    float lo, scale;
    unsigned klo, shift;
    bool use_keys;
    __device__ __forceinline__ int operator()(float v) const {
        if (use_keys) return (int)((float_key(v) - klo) >> shift);
        int b = __float2int_rz(__fmul_rn(__fsub_rn(v, lo), scale));
        return min(b, kSelBuckets - 1);
    }
};

template <int NT>
__device__ __forceinline__ void block_minmax(float& mn, float& mx, SelectSmem& sm) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, off));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, off));
    }
    if ((threadIdx.x & 31) == 0) {
        sm.red_a[threadIdx.x >> 5] = mn;
        sm.red_b[threadIdx.x >> 5] = mx;
    }
    __syncthreads();
    mn = sm.red_a[0];
    mx = sm.red_b[0];
#pragma unroll
    for (int i = 1; i < NT / 32; ++i) {
        mn = fminf(mn, sm.red_a[i]);
        mx = fmaxf(mx, sm.red_b[i]);
    }
    __syncthreads();
}

// k-th smallest (0-based) of the CTA's `len` values v[r] ↔ element tid + r·NT, and, if need_next, the (k+1)-th.
template <int EPT, int NT>
__device__ void block_select(const float (&v)[EPT], int len, int k, bool need_next, SelectSmem& sm, float& out_k,
                             float& out_next) {
    const int tid = threadIdx.x;
    float mn = INFINITY, mx = -INFINITY;
#pragma unroll
    for (int r = 0; r < EPT; ++r)
        if (tid + r * NT < len) { mn = fminf(mn, v[r]); mx = fmaxf(mx, v[r]); }
    block_minmax<NT>(mn, mx, sm);
    float lo = mn, hi = mx;
    unsigned below = 0, in_range = (unsigned)len;
    bool first = true, has_next = false;
    float vk = lo, vnext = lo;
    for (int iter = 0;; ++iter) {
        const unsigned kk = (unsigned)k - below; // rank inside [lo, hi]
        if (lo == hi) {
            vk = lo; vnext = lo; has_next = (kk + 1 < in_range);
            break;
        }
        BucketMap bm;
        const float width = hi - lo;
        bm.lo = lo;
        bm.scale = (float)kSelBuckets / width;
        bm.use_keys = iter >= 3 || !isfinite(width) || !isfinite(bm.scale);
        bm.klo = float_key(lo);
        const unsigned krange = float_key(hi) - bm.klo;
        bm.shift = (krange < (unsigned)kSelBuckets) ? 0u : (unsigned)(32 - __clz(krange) - 8);
        if (tid < kSelBuckets) sm.hist[tid] = 0;
        if (tid == 0) sm.list_n = 0;
        __syncthreads();
#pragma unroll
        for (int r = 0; r < EPT; ++r) {
            const float x = v[r];
            if (tid + r * NT < len && (first || (x >= lo && x <= hi))) atomicAdd(&sm.hist[bm(x)], 1u);
        }
        __syncthreads();
        // CTA scan over the 256 buckets: find the bucket whose cumulative count passes kk
        if (tid < kSelBuckets) {
            unsigned inc = sm.hist[tid];
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                unsigned t = __shfl_up_sync(0xffffffffu, inc, off);
                if ((tid & 31) >= off) inc += t;
            }
            // The warp total is published by lane 0 (not lane 31): nvcc 12.9 reuses the lane-0 address base + (tid >> 3)
            // of block_minmax for any sm.x[tid >> 5] store, which is misaligned for other lanes.
            const unsigned wtot = __shfl_sync(0xffffffffu, inc, 31);
            if ((tid & 31) == 0) sm.warp_tot[tid >> 5] = wtot;
            sm.hist[tid] = inc; // inclusive within the warp; warp bases are added after the barrier
        }
        __syncthreads();
        if (tid < kSelBuckets) {
            unsigned base = 0;
            for (int w = 0; w < (tid >> 5); ++w) base += sm.warp_tot[w];
            const unsigned inc = sm.hist[tid] + base;
            const unsigned prev = (tid & 31) ? sm.hist[tid - 1] + base : base;
            if (prev <= kk && kk < inc) {
                sm.sel_bucket = tid;
                sm.sel_excl = prev;
                sm.sel_count = inc - prev;
            }
        }
        __syncthreads();
        const int bsel = sm.sel_bucket;
        const unsigned excl = sm.sel_excl, cnt = sm.sel_count;
        if (cnt <= (unsigned)kSelListCap) {
#pragma unroll
            for (int r = 0; r < EPT; ++r) {
                const float x = v[r];
                if (tid + r * NT < len && (first || (x >= lo && x <= hi)) && bm(x) == bsel)
                    sm.list[atomicAdd(&sm.list_n, 1u)] = x;
            }
            __syncthreads();
            const unsigned target = kk - excl;
            for (unsigned t = tid; t < cnt; t += NT) {
                const float x = sm.list[t];
                unsigned rank = 0;
                for (unsigned j = 0; j < cnt; ++j) {
                    const float y = sm.list[j];
                    rank += (y < x || (y == x && j < t)) ? 1u : 0u;
                }
                if (rank == target) sm.out_k = x;
                if (rank == target + 1) sm.out_next = x;
            }
            __syncthreads();
            vk = sm.out_k;
            has_next = (target + 1 < cnt);
            vnext = has_next ? sm.out_next : vk;
            break;
        }
        // too many members: narrow the range to the selected bucket's own [min, max] and go again
        mn = INFINITY; mx = -INFINITY;
#pragma unroll
        for (int r = 0; r < EPT; ++r) {
            const float x = v[r];
            if (tid + r * NT < len && (first || (x >= lo && x <= hi)) && bm(x) == bsel) {
                mn = fminf(mn, x); mx = fmaxf(mx, x);
            }
        }
        block_minmax<NT>(mn, mx, sm);
        lo = mn; hi = mx; below += excl; in_range = cnt; first = false;
    }
    if (need_next && !has_next) { // rank k is the largest of its bucket: the next order statistic lies above
        mn = INFINITY; mx = -INFINITY;
#pragma unroll
        for (int r = 0; r < EPT; ++r)
            if (tid + r * NT < len && v[r] > vk) mn = fminf(mn, v[r]);
        block_minmax<NT>(mn, mx, sm);
        vnext = mn;
    }
    __syncthreads();
    out_k = vk;
    out_next = vnext;
}

// The two central order statistics a ≤ b of the CTA's values (a = b for odd len): the median is (a + b)/2 (R4).
template <int EPT, int NT>
__device__ __forceinline__ void block_median_pair(const float (&v)[EPT], int len, SelectSmem& sm, float& a, float& b) {
    const bool even = (len & 1) == 0;
    block_select<EPT, NT>(v, len, (len - 1) >> 1, even, sm, a, b);
    if (!even) b = a;
}

// One component of one block: v ← |v − median(v)| in place; returns 1/(√2·κ·MAD) (0 if κ·MAD is 0 or not finite,
// R7), the √2 folding the ½ of P = (re'² + im'²)/2 into the scale, and the median as a + h (a = lower central value,
// h = half the gap to the upper one).
// The median (a + b)/2 is never rounded to float32: v − (a+b)/2 is formed as (v − a) − (b − a)/2, whose rounding
// errors are relative to the deviation itself, so a spectrum riding on a large offset loses nothing.
template <int EPT, int NT>
__device__ __forceinline__ float normalise_component(float (&v)[EPT], int len, SelectSmem& sm, float& a_out, float& h_out) {
    float a, b;
    block_median_pair<EPT, NT>(v, len, sm, a, b);
    const float h = 0.5f * __fsub_rn(b, a);
    a_out = a; h_out = h;
#pragma unroll
    for (int r = 0; r < EPT; ++r) v[r] = fabsf(__fsub_rn(__fsub_rn(v[r], a), h));
    block_median_pair<EPT, NT>(v, len, sm, a, b);
    const double s = kKappa * (0.5 * ((double)a + (double)b));
    return (s > 0.0 && isfinite(s)) ? (float)(0.70710678118654752440 / s) : 0.f;
}

// One normalisation block by the general path: len values at src → powers at dst.  The normalised component
// ((v − a) − h)·inv is evaluated as fma(v − a, inv, −h·inv) from the re-read input (the registers hold |v − m| by
// then); norm_power_v2.cuh uses the same expression, so both paths produce identical bits.
// Write one block's outputs from its statistics: len bins at src → P and/or (G, stats).  Bin tid + r·NT belongs to thread
// tid; lo is the block's first bin in its row (a multiple of 4 when G is written), `blk` its index in [batch][nb].
template <int EPT, int NT>
__device__ __forceinline__ void norm_block_write(const float2* __restrict__ src, int len, long long row, long long lo, long long blk,
                                                 const NormOut& out, float a0, float i0, float k0, float a1, float i1, float k1) {
    const int tid = threadIdx.x;
    if (out.P) {
        float* dst = out.P + row * out.pitchP + lo;
#pragma unroll
        for (int r = 0; r < EPT; ++r) {
            const int idx = tid + r * NT;
            if (idx < len) dst[idx] = norm_power_value(__ldg(src + idx), a0, i0, k0, a1, i1, k1);
        }
    }
    if (out.G) {
        float* g = out.G + row * out.pitchG + (lo >> 2);
        auto pw = [&](int r) {
            const int idx = tid + r * NT;
            return idx < len ? norm_power_value(__ldg(src + idx), a0, i0, k0, a1, i1, k1) : 0.f;
        };
        if constexpr (EPT % 4 == 0) {
#pragma unroll
            for (int r0 = 0; r0 < EPT; r0 += 4) {
                const float e = quad_sums4(pw(r0), pw(r0 + 1), pw(r0 + 2), pw(r0 + 3));
                const int r = r0 + (tid & 3);
                if ((tid & ~3) + r * NT < len) g[(tid >> 2) + r * (NT / 4)] = e;   // the group's first bin exists
            }
        } else {
#pragma unroll
            for (int r = 0; r < EPT; ++r) {
                const float e = quad_sum1(pw(r));
                if ((tid & 3) == 0 && tid + r * NT < len) g[(tid >> 2) + r * (NT / 4)] = e;
            }
        }
        if (tid == 0) {
            float* st = out.stats + blk * 8;
            st[0] = a0; st[1] = i0; st[2] = k0; st[3] = a1; st[4] = i1; st[5] = k1;
        }
    }
}

// One normalisation block by the general path: len values at src → outputs.  The statistics are found on
// register-resident values; the outputs are then computed from the re-read input (the registers hold |v − m| by then)
// through norm_power_value(), as in norm_power_v2.cuh, so both paths produce identical bits.
template <int EPT, int NT>
__device__ __forceinline__ void norm_block_general(const float2* __restrict__ src, int len, long long row, long long lo,
                                                   long long blk, const NormOut& out, SelectSmem& sm) {
    const int tid = threadIdx.x;
    float re[EPT], im[EPT];
#pragma unroll
    for (int r = 0; r < EPT; ++r) {
        const int idx = tid + r * NT;
        float2 z = make_float2(0.f, 0.f);
        if (idx < len) z = __ldg(src + idx);
        re[r] = z.x;
        im[r] = z.y;
    }
    float a_re, h_re, a_im, h_im;
    const float inv_re = normalise_component<EPT, NT>(re, len, sm, a_re, h_re);
    const float inv_im = normalise_component<EPT, NT>(im, len, sm, a_im, h_im);
    norm_block_write<EPT, NT>(src, len, row, lo, blk, out, a_re, inv_re, -h_re * inv_re, a_im, inv_im, -h_im * inv_im);
}

// General kernel: one CTA per normalisation block.  Grid: blocks_per_row · batch CTAs; block j = first_block +
// (blockIdx.x mod blocks_per_row) of spectrum blockIdx.x / blocks_per_row.  Block j covers bins [jB, (j+1)B), the
// last block of a row extends to n (R6).  Output: P[row·pitchP + bin] = ((re−m_re)/s_re)²/2 + ((im−m_im)/s_im)²/2,
// s = κ·MAD; s = 0 or not finite → 0 (R7).  Handles any block length up to EPT·NT.
template <int EPT, int NT>
__global__ void __launch_bounds__(NT)
norm_power_kernel(const float2* __restrict__ spectra, long long pitch_in, long long n, int B, int nb, int first_block,
                  int blocks_per_row, NormOut out) {
    __shared__ SelectSmem sm;
    const long long row = blockIdx.x / blocks_per_row;
    const int j = first_block + (int)(blockIdx.x % blocks_per_row);
    const long long lo = (long long)j * B;
    const long long hi = (j == nb - 1) ? n : lo + B;
    norm_block_general<EPT, NT>(spectra + row * pitch_in + lo, (int)(hi - lo), row, lo, row * nb + j, out, sm);
}

// Redo kernel: the blocks the fast kernel declined (redo[e] = row·blocks_per_row + j, all of length B), by the general
// path.  A fixed small grid loops over the list, whose length is only known on the device.
template <int EPT, int NT>
__global__ void __launch_bounds__(NT)
norm_power_redo_kernel(const float2* __restrict__ spectra, long long pitch_in, int B, int nb, int blocks_per_row,
                       NormOut out, const unsigned* __restrict__ redo, const unsigned* __restrict__ redo_count) {
    __shared__ SelectSmem sm;
    const unsigned cnt = *redo_count;
    for (unsigned e = blockIdx.x; e < cnt; e += gridDim.x) {
        const unsigned id = redo[e];
        const long long row = id / (unsigned)blocks_per_row;
        const long long j = id % (unsigned)blocks_per_row;
        const long long lo = j * B;
        norm_block_general<EPT, NT>(spectra + row * pitch_in + lo, B, row, lo, row * nb + j, out, sm);
        __syncthreads();
    }
}

} // namespace pulscan
