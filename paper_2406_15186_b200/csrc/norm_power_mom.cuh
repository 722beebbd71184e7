// norm_power_mom.cuh — kernel (a), fast mode: the paper's own GPU normalisation, Algorithm 1 "Median of Medians
// Normalisation" (§2.5 "threads recursively find the median of 4 non-overlapping elements").
//
// It is an APPROXIMATION of the median and of the MAD (the exact kernel is norm_power_v2.cuh): for every chunk of B bins
// and each component,
//     local_median(a,b,c,d) = (a+b+c+d − min − max)/2                                                    (L627-631)
//     for strides ← count/4, count/16, …: s[i] ← local_median(s[i], s[i+stride], s[i+2·stride], s[i+3·stride])  (L636-642)
//     median ← median_of_medians(chunk); MAD ← median_of_medians(|chunk − median|); scale_factor ← 1.4826   (L643-649)
// with the readings R5 (absolute value) and R30 (B = 4^k or 2·4^k, a last level of two values returns their mean; the
// n mod B bins after the last chunk use the last chunk's median and MAD).  P = (re'² + im'²)/2 as in the exact path (R2).
//
// Mapping.  Element i of a level lives in thread i mod NT, slot i div NT, so as long as a thread holds a multiple of 4
// values the four members of a group (i, i+stride, i+2·stride, i+3·stride with stride = NT·k/4) are its own slots
// r, r+k/4, r+2k/4, r+3k/4: the first one to three levels need no communication and run while the loads stream in.  The
// remaining ≤ 2·NT values go through shared memory, one CTA barrier per level.  The block is read three times (median,
// MAD, output), the second and third time out of L1/L2; there is no histogram and no atomic.
// The median of four is evaluated as m2 + (m3 − m2)/2 from the two middle values (a min/max network) and everything is
// taken relative to the chunk's first bin, so rounding errors scale with the spread of the chunk, not with its offset.
#pragma once
#include <cuda_runtime.h>

namespace pulscan {

constexpr double kMomScale = 1.4826;   // Alg. 1 L648 prints this 5-digit constant

__device__ __forceinline__ float mom_med4(float a, float b, float c, float d) {
    const float lo1 = fminf(a, b), hi1 = fmaxf(a, b), lo2 = fminf(c, d), hi2 = fmaxf(c, d);
    const float m2 = fmaxf(lo1, lo2), m3 = fminf(hi1, hi2);         // the two middle values, in either order
    return __fmaf_rn(0.5f, __fsub_rn(m3, m2), m2);
}

// Levels a thread can do on its own K values (slots r ↔ element tid + r·NT): K → K/4 while K is a multiple of 4.
template <int K>
__device__ __forceinline__ void mom_local_levels(float (&v)[K], int& k_out) {
    if constexpr (K % 4 == 0) {
        float w[K / 4];
#pragma unroll
        for (int r = 0; r < K / 4; ++r) w[r] = mom_med4(v[r], v[r + K / 4], v[r + 2 * (K / 4)], v[r + 3 * (K / 4)]);
        mom_local_levels<K / 4>(w, k_out);
#pragma unroll
        for (int r = 0; r < K / 4; ++r) v[r] = w[r];
    } else {
        k_out = K;
    }
}

constexpr int mom_local_result(int k) {
    while (k % 4 == 0) k /= 4;
    return k;
}

// CTA part of the reduction: `count` values per component in sm[c][0..count), element order as in Alg. 1.  Returns the
// result of both components to every thread.  Starts and ends with a barrier.
template <int NT>
__device__ __forceinline__ float2 mom_cta_levels(float (*sm)[2 * NT], int count) {
    const int tid = threadIdx.x;
    while (count >= 4) {
        const int stride = count >> 2;
        __syncthreads();
        float r0 = 0.f, r1 = 0.f;
        const bool mine = tid < stride;                                   // stride ≤ NT/2
        if (mine) {
            r0 = mom_med4(sm[0][tid], sm[0][tid + stride], sm[0][tid + 2 * stride], sm[0][tid + 3 * stride]);
            r1 = mom_med4(sm[1][tid], sm[1][tid + stride], sm[1][tid + 2 * stride], sm[1][tid + 3 * stride]);
        }
        __syncthreads();                                                  // everybody has read before anybody overwrites
        if (mine) { sm[0][tid] = r0; sm[1][tid] = r1; }
        count = stride;
    }
    __syncthreads();
    float2 out;
    if (count == 2) out = make_float2(0.5f * (sm[0][0] + sm[0][1]), 0.5f * (sm[1][0] + sm[1][1]));
    else out = make_float2(sm[0][0], sm[1][0]);
    __syncthreads();
    return out;
}

// Grid: nb · batch CTAs; CTA x handles chunk (x mod nb) of spectrum x / nb: statistics from bins [jB, (j+1)B), output for
// [jB, (j+1)B) — to n for the last chunk of the row (R30).  B = EPT · NT, EPT a multiple of 4.
template <int EPT, int NT>
__global__ void __launch_bounds__(NT)
norm_power_mom_kernel(const float2* __restrict__ spectra, long long pitch_in, long long n, int nb, float* __restrict__ P,
                      long long pitchP) {
    static_assert(EPT % 4 == 0, "the first level of Alg. 1 is done on a thread's own values");
    constexpr int B = EPT * NT;
    constexpr int K1 = EPT / 4;                          // values per thread after the streaming first level
    constexpr int KL = mom_local_result(K1);           // … after the thread-local levels (1 or 2)
    static_assert(KL <= 2, "shared-memory stage sized for two values per thread");
    __shared__ float sm[2][2 * NT];
    const int tid = threadIdx.x;
    const long long row = blockIdx.x / nb;
    const int j = (int)(blockIdx.x - row * nb);
    const long long lo = (long long)j * B;
    const long long hi = (j == nb - 1) ? n : lo + B;
    const float2* src = spectra + row * pitch_in + lo;
    const float2 pv = __ldg(src);                        // everything is taken relative to the chunk's first bin

    float2 centre = make_float2(0.f, 0.f);               // median − pv, per component
    float2 mad = make_float2(0.f, 0.f);
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {               // 0: median of u = v − pv; 1: median of |u − centre|
        float a[K1], b[K1];
#pragma unroll
        for (int r = 0; r < K1; ++r) {
            float x[4], y[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float2 z = __ldg(src + tid + (r + q * K1) * NT);
                x[q] = __fsub_rn(z.x, pv.x); y[q] = __fsub_rn(z.y, pv.y);
                if (pass) { x[q] = fabsf(__fsub_rn(x[q], centre.x)); y[q] = fabsf(__fsub_rn(y[q], centre.y)); }
            }
            a[r] = mom_med4(x[0], x[1], x[2], x[3]);
            b[r] = mom_med4(y[0], y[1], y[2], y[3]);
        }
        int kl;
        mom_local_levels<K1>(a, kl);
        mom_local_levels<K1>(b, kl);
#pragma unroll
        for (int r = 0; r < KL; ++r) { sm[0][tid + r * NT] = a[r]; sm[1][tid + r * NT] = b[r]; }
        const float2 res = mom_cta_levels<NT>(sm, KL * NT);
        if (pass == 0) centre = res; else mad = res;
    }
    // x' = (u − centre)/(1.4826·MAD); the ½ of P = (re'² + im'²)/2 is folded into the scale; MAD = 0 or not finite → 0 (R7)
    const double sx = kMomScale * (double)mad.x, sy = kMomScale * (double)mad.y;
    const float ix = (sx > 0.0 && isfinite(sx)) ? (float)(0.70710678118654752440 / sx) : 0.f;
    const float iy = (sy > 0.0 && isfinite(sy)) ? (float)(0.70710678118654752440 / sy) : 0.f;
    float* dst = P + row * pitchP + lo;
    const int len = (int)(hi - lo);
    for (int i = tid; i < len; i += NT) {
        const float2 z = __ldg(src + i);
        const float x = __fsub_rn(__fsub_rn(z.x, pv.x), centre.x) * ix, y = __fsub_rn(__fsub_rn(z.y, pv.y), centre.y) * iy;
        dst[i] = __fmaf_rn(x, x, y * y);
    }
}

} // namespace pulscan
