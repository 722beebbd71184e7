// harmonic_sum.cuh — harmonic sum by decimation (§2.3; Table 4 "DecimateHarmonics" L576).
//
// "Summing adjacent non-overlapping pairs, triples, quartets, etc. of frequency magnitudes to produce a magnitude spectra
// decimated by factors of 2, 3, 4": D_h(r) = Σ_{j<h} P[h·r + j].  "We then sum the overlapping sections of each decimated
// spectra (aligned so the 0th bin of each spectrum is summed) and discard the non-overlapping parts":
//     Y_H(r) = Σ_{h=1..H} D_h(r),   r ∈ [0, floor(n/H))            (reading R29: complete groups only)
// which in noise is χ² with H(H+1) degrees of freedom, i.e. a Gamma variate of shape H(H+1)/2 in the mean-1 units of P.
// One thread per output bin; the H(H+1)/2 reads per output are contiguous runs of h floats starting at h·r, so a warp's
// reads for a given (h, j) are strided by h floats and hit each 128-byte line at most h times from L1.
#pragma once
#include <cuda_runtime.h>

namespace pulscan {

constexpr int kHarmThreads = 256;

template <int H>
__global__ void __launch_bounds__(kHarmThreads)
harmonic_sum_kernel(const float* __restrict__ P, long long pitchP, float* __restrict__ Y, long long pitchY, long long nH,
                    long long total) {
    for (long long idx = (long long)blockIdx.x * kHarmThreads + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * kHarmThreads) {
        const long long row = idx / nH, r = idx - row * nH;
        const float* src = P + row * pitchP;
        float y = 0.f;
#pragma unroll
        for (int h = 1; h <= H; ++h)
#pragma unroll
            for (int j = 0; j < h; ++j) y += __ldg(src + h * r + j);
        Y[row * pitchY + r] = y;
    }
}

} // namespace pulscan
