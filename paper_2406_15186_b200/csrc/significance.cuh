// significance.cuh — χ² tail and Gaussian-equivalent σ in double precision, host + device.
//
// PAPER.md:L154-158 (Eq. 9): a width-w boxcar of normalised powers is χ² with 2w degrees of freedom; in mean-1 power
// units (R2) the statistic is 2S, so p = Q(w, S) = e^{-S} Σ_{k<w} S^k/k!, a finite sum for integer w.
// L114/L158: p → Gaussian-equivalent σ through the normal survival function (one-sided, R16).
// Everything stays in the log domain: strong injections reach ln p ≈ −1200, far below double underflow of p itself.
#pragma once
#include <cmath>
#include <cuda_runtime.h>

namespace pulscan {

// ln Q(w, S).  The sum is normalised at its largest term (index ks = min(w−1, ⌊S⌋)); every term is positive.
// On the hot path only S ≥ T_w > w−1 occurs, where ks = w−1 and the terms fall geometrically: the loop stops once
// a term no longer changes the sum.
__host__ __device__ inline double ln_q(int w, double S) {
    if (!(S > 0.0)) return 0.0;
    int ks = (S >= (double)(w - 1)) ? (w - 1) : (int)floor(S);
    double sum = 1.0, t = 1.0;
    const double inv_s = 1.0 / S;
    for (int k = ks; k >= 1; --k) {
        t *= (double)k * inv_s;
        sum += t;
        if (t < 1e-18 * sum) break;
    }
    t = 1.0;
    for (int k = ks + 1; k <= w - 1; ++k) {
        t *= S / (double)k;
        sum += t;
        if (t < 1e-18 * sum) break;
    }
    return -S + (double)ks * log(S) - lgamma((double)ks + 1.0) + log(sum);
}

// ln sf(x) = ln(½ erfc(x/√2)); asymptotic expansion where erfc would underflow.
__host__ __device__ inline double ln_sf(double x) {
    const double kInvSqrt2 = 0.70710678118654752440;
    const double kHalfLn2Pi = 0.91893853320467274178;
    if (x < 0.0) return log1p(-0.5 * erfc(-x * kInvSqrt2));
    if (x < 25.0) return log(0.5 * erfc(x * kInvSqrt2));
    double r = 1.0 / (x * x), term = 1.0, sum = 1.0;
    for (int k = 1; k < 40; ++k) {
        double next = -term * (double)(2 * k - 1) * r;
        if (fabs(next) >= fabs(term) || fabs(next) < 1e-18) break;
        term = next;
        sum += term;
    }
    return -0.5 * x * x - log(x) - kHalfLn2Pi + log(sum);
}

// σ with ln sf(σ) = lnp (lnp < 0).  Newton on the log-survival function, safeguarded by a bracket.
__host__ __device__ inline double sigma_from_lnp(double lnp) {
    const double kHalfLn2Pi = 0.91893853320467274178;
    if (!(lnp < 0.0)) return -INFINITY;
    double lo = -40.0, hi = 1.0;
    if (ln_sf(lo) < lnp) return lo;
    while (ln_sf(hi) > lnp) { lo = hi; hi *= 2.0; }
    double x = 0.5 * (lo + hi);
    if (lnp < -3.0) { // tail start: −x²/2 − ln x − ½ln 2π ≈ lnp
        double g = sqrt(-2.0 * (lnp + kHalfLn2Pi));
        g = sqrt(fmax(1e-6, -2.0 * (lnp + kHalfLn2Pi + log(g))));
        if (g > lo && g < hi) x = g;
    }
    for (int it = 0; it < 100; ++it) {
        double f = ln_sf(x) - lnp;      // decreasing in x
        if (f > 0.0) lo = x; else hi = x;
        // d/dx ln sf(x) = −φ(x)/sf(x)
        double dlog = -exp(-0.5 * x * x - kHalfLn2Pi - (f + lnp));
        double xn = x - f / dlog;
        if (!(xn > lo && xn < hi)) xn = 0.5 * (lo + hi);
        if (fabs(xn - x) <= 1e-15 * fmax(1.0, fabs(x))) { x = xn; break; }
        x = xn;
    }
    return x;
}

// Host only: the power T at which ln Q(w, T) = lnp_target (bisection; ln Q is strictly decreasing in S).
inline double power_threshold(int w, double lnp_target) {
    double lo = 0.0, hi = (double)w + 16.0;
    while (ln_q(w, hi) > lnp_target) hi *= 2.0;
    for (int it = 0; it < 200 && hi - lo > 1e-14 * hi; ++it) {
        double mid = 0.5 * (lo + hi);
        if (ln_q(w, mid) > lnp_target) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

} // namespace pulscan
