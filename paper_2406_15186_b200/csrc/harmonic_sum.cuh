// harmonic_sum.cuh — harmonic sum by decimation (§2.3; Table 4 "DecimateHarmonics" L576).
//
// "Summing adjacent non-overlapping pairs, triples, quartets, etc. of frequency magnitudes to produce a magnitude spectra
// decimated by factors of 2, 3, 4": D_h(r) = Σ_{j<h} P[h·r + j].  "We then sum the overlapping sections of each decimated
// spectra (aligned so the 0th bin of each spectrum is summed) and discard the non-overlapping parts":
//     Y_H(r) = Σ_{h=1..H} D_h(r),   r ∈ [0, floor(n/H))            (reading R29: complete groups only)
// which in noise is χ² with H(H+1) degrees of freedom, i.e. a Gamma variate of shape H(H+1)/2 in the mean-1 units of P.
#pragma once
#include <cuda_runtime.h>

namespace pulscan {

constexpr int kHarmThreads = 256;

// One pass for all H = 2..HMAX: thread r forms Y_2(r), then adds D_3(r) for Y_3(r), then D_4(r) for Y_4(r), in the order
// h = 1, 2, …; j = 0, 1, … (the running sum of Y_H is a prefix of Y_{H+1}'s).  P is read 1 + 2 + 3 + 4 times per thread
// instead of once per (H, h, j); the reads of a warp for a given h are h contiguous floats per thread.
struct HarmonicOut {
    float* Y[3];          // Y_2, Y_3, Y_4
    long long pitch[3];
    long long nH[3];      // floor(n / H)
};

template <int HMAX>
__global__ void __launch_bounds__(kHarmThreads)
harmonic_sum_kernel(const float* __restrict__ P, long long pitchP, HarmonicOut out, long long total) {
    const long long n2 = out.nH[0];
    for (long long idx = (long long)blockIdx.x * kHarmThreads + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * kHarmThreads) {
        const long long row = idx / n2, r = idx - row * n2;
        const float* src = P + row * pitchP;
        float y = __ldg(src + r);
        const float2 d2 = __ldg(reinterpret_cast<const float2*>(src + 2 * r));        // rows are 16-byte aligned
        y += d2.x; y += d2.y;
        out.Y[0][row * out.pitch[0] + r] = y;
        if (HMAX >= 3 && r < out.nH[1]) {
            y += __ldg(src + 3 * r); y += __ldg(src + 3 * r + 1); y += __ldg(src + 3 * r + 2);
            out.Y[1][row * out.pitch[1] + r] = y;
            if (HMAX >= 4 && r < out.nH[2]) {
                const float4 d4 = __ldg(reinterpret_cast<const float4*>(src + 4 * r));
                y += d4.x; y += d4.y; y += d4.z; y += d4.w;
                out.Y[2][row * out.pitch[2] + r] = y;
            }
        }
    }
}

} // namespace pulscan
