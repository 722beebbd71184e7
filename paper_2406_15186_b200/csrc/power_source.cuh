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

    // Loader for bins lo … of one row; remembers the statistics of the normalisation block it is in.
    struct Row {
        const PowerSource& s;
        long long row;
        int cur = -1;
        float a0 = 0.f, i0 = 0.f, k0 = 0.f, a1 = 0.f, i1 = 0.f, k1 = 0.f;
        __device__ __forceinline__ Row(const PowerSource& src, long long r) : s(src), row(r) {}
        __device__ __forceinline__ float operator()(long long bin) {
            if (s.P) return __ldg(s.P + row * s.pitchP + bin);
            int j = (int)(bin / s.B);
            if (j >= s.nb) j = s.nb - 1;
            if (j != cur) {
                const float4 u = __ldg(reinterpret_cast<const float4*>(s.stats + (row * s.nb + j) * 8));
                const float2 w = __ldg(reinterpret_cast<const float2*>(s.stats + (row * s.nb + j) * 8 + 4));
                a0 = u.x; i0 = u.y; k0 = u.z; a1 = u.w; i1 = w.x; k1 = w.y;
                cur = j;
            }
            return norm_power_value(__ldg(s.spectra + row * s.pitch + bin), a0, i0, k0, a1, i1, k1);
        }
    };
};

} // namespace pulscan
