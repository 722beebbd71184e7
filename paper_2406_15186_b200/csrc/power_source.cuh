// power_source.cuh — where the rare-path kernels (sweep_refine_kernel, block_exact_kernel) read a bin's normalised power.
//
// The streaming path no longer keeps the float32 power spectrum in HBM: kernel (a) leaves the sums of aligned groups of four
// bins and, per normalisation block, the six numbers (a, inv, k per component) that define the normalisation
// (norm_power.cuh, NormOut).  A flagged span is then rebuilt from the input spectrum with the very function kernel (a) used,
// norm_power_value(), so the rebuilt powers are bit-identical to the ones that went into the group sums.
// Plans that do keep a per-bin array (exhaustive mode, full-resolution sweep, harmonic-summed spectra Y_H, Alg. 1
// normalisation) read that array instead.
#pragma once
#include <cuda_runtime.h>

#include "norm_power.cuh"

namespace pulscan {

struct PowerSource {
    const float* P;          // per-bin array [batch][pitchP], or null: rebuild from the spectrum
    long long pitchP;
    const float2* spectra;   // complex64 [batch][pitch]
    long long pitch;
    const float* stats;      // [batch][nb][8]: a_re, inv_re, k_re, a_im, inv_im, k_im, -, -
    int B, nb;               // normalisation block and blocks per row (the last block absorbs the remainder, R6)

    // Loader for the bins of one row.  It holds the statistics of two consecutive normalisation blocks, [lo, mid) and
    // [mid, hi): a flagged span is a few hundred bins, so after the first bin no division and no further look-up is needed;
    // a bin outside [lo, hi) reloads (spans longer than a normalisation block).
    struct Row {
        const PowerSource& s;
        long long row;
        long long lo = 0, mid = 0, hi = 0;       // hi = 0: nothing loaded yet
        float4 ua = {0.f, 0.f, 0.f, 0.f}, ub = {0.f, 0.f, 0.f, 0.f};   // (a_re, inv_re, k_re, a_im) of the two blocks
        float2 wa = {0.f, 0.f}, wb = {0.f, 0.f};                         // (inv_im, k_im)
        __device__ __forceinline__ Row(const PowerSource& src, long long r) : s(src), row(r) {}
        __device__ __forceinline__ void prepare(long long bin) {
            int j = (int)(bin / s.B);
            if (j >= s.nb) j = s.nb - 1;
            lo = (long long)j * s.B;
            const float* st = s.stats + (row * s.nb + j) * 8;
            ua = __ldg(reinterpret_cast<const float4*>(st));
            wa = __ldg(reinterpret_cast<const float2*>(st + 4));
            if (j + 1 < s.nb) {
                mid = lo + s.B;
                hi = (j + 2 < s.nb) ? mid + s.B : 0x7fffffffffffffffLL;   // the last block extends to the end of the row (R6)
                ub = __ldg(reinterpret_cast<const float4*>(st + 8));
                wb = __ldg(reinterpret_cast<const float2*>(st + 12));
            } else {
                mid = hi = 0x7fffffffffffffffLL;
                ub = ua; wb = wa;
            }
        }
        __device__ __forceinline__ float operator()(long long bin) {
            if (s.P) return __ldg(s.P + row * s.pitchP + bin);
            if (bin < lo || bin >= hi) prepare(bin);
            const bool t = bin >= mid;
            return norm_power_value(__ldg(s.spectra + row * s.pitch + bin), t ? ub.x : ua.x, t ? ub.y : ua.y, t ? ub.z : ua.z,
                                    t ? ub.w : ua.w, t ? wb.x : wa.x, t ? wb.y : wa.y);
        }
    };
};

} // namespace pulscan
