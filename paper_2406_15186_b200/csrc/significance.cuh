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
    // terms ks−1 … 0: t_{j+1} = t_j · k/S with k = ks, ks−1, …; the ratio is carried as a double (no conversion per term) and
    // the stopping test runs every fourth term
    double kd = (double)ks;
    int k = ks;
    for (; k >= 4; k -= 4) {
        t *= kd * inv_s; sum += t; kd -= 1.0;
        t *= kd * inv_s; sum += t; kd -= 1.0;
        t *= kd * inv_s; sum += t; kd -= 1.0;
        t *= kd * inv_s; sum += t; kd -= 1.0;
        if (t < 1e-18 * sum) { k = 0; break; }
    }
    for (; k >= 1; --k) { t *= kd * inv_s; sum += t; kd -= 1.0; }
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

// Algorithm 3 (§2.6 Eq. 10-12): the paper's GPU approximation of ln p, a degree-16 polynomial
// in x = 1500·dof/pow fitted by regression, in the paper's units (pow = |X'|² summed over the window = 2S, dof = its χ²
// degrees of freedom = 2·shape; R31).  Horner form in double: the printed coefficients span 1e-46 … 1e2 and x
// reaches 1575 (the branch dof ≥ 1.05·pow cuts it off there), so neither the coefficients nor the powers of x fit float32.
// alg3_poly is the polynomial branch alone: pow·f(1500·dof/pow)/1500.
__host__ __device__ inline double alg3_poly(double pw, double dof) {
    const double x = 1500.0 * dof / pw;
    double f = -4.4604059e-46;
    f = f * x + 9.4927863e-42;
    f = f * x - 9.1470451e-38;
    f = f * x + 5.2810851e-34;
    f = f * x - 2.0376166e-30;
    f = f * x + 5.5480334e-27;
    f = f * x - 1.0973877e-23;
    f = f * x + 1.5991804e-20;
    f = f * x - 1.7231488e-17;
    f = f * x + 1.3660070e-14;
    f = f * x - 7.8617952e-12;
    f = f * x + 3.2136336e-9;
    f = f * x - 9.0466418e-7;
    f = f * x + 0.00016945948;
    f = f * x - 0.021494231;
    f = f * x + 2.9515954;
    f = f * x - 755.24091;
    return pw * f / 1500.0;
}
__host__ __device__ inline double power_to_logp(double pw, double dof) {
    if (dof >= pw * 1.05) return 0.0;
    return alg3_poly(pw, dof);
}

// ln p of a sum S of Gamma shape `shape` (mean-1 units): mode 0 the exact χ² tail, mode 1 Alg. 3.
__host__ __device__ inline double lnp_of(int signif_mode, int shape, double S) {
    return signif_mode ? power_to_logp(2.0 * S, 2.0 * (double)shape) : ln_q(shape, S);
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

// Host only: a lower bound of the smallest power S at which Alg. 3 reports ln p ≤ lnp_target for Gamma shape `shape`.  The
// polynomial is not monotone in S (for x ≳ 1100, i.e. S ≲ 1.36·shape, the printed coefficients do not determine it, and at the
// branch point x = 1575 it is already below −20 for shapes ≳ 110), so the first crossing is looked for from the branch point
// S = shape/1.05 upwards: a coarse grid, and inside every grid interval where a crossing cannot be excluded — the lower of its
// end values minus the largest change between neighbouring grid points is not above the target, a Lipschitz bound with a
// factor 2 in hand — a bisection that keeps excluding halves the same way (slopes by central differences) down to 1e-9
// relative.  What is returned is the lower end of the first interval that could not be excluded: never above the first
// crossing, so no window the oracle's Alg. 3 would report is dropped by the power pre-threshold.  The scan evaluates the
// polynomial branch itself from a hair below the branch point, where power_to_logp still returns 0.
inline double alg3_first_crossing(double sh, double target, double a, double b, double ga, double gb, double la, double lb, int depth) {
    // la, lb: |slope| estimates at the ends.  Nothing at or below the target inside [a, b]?
    if (fmin(ga, gb) - (b - a) * fmax(la, lb) > target) return -1.0;
    if (ga <= target || depth >= 48 || b - a <= 1e-9 * b) return a;
    const double m = 0.5 * (a + b), h = 1e-7 * m;
    const double gm = alg3_poly(2.0 * m, 2.0 * sh);
    const double lm = fabs(alg3_poly(2.0 * (m + h), 2.0 * sh) - alg3_poly(2.0 * (m - h), 2.0 * sh)) / (2.0 * h);
    const double r = alg3_first_crossing(sh, target, a, m, ga, gm, la, lm, depth + 1);
    return r >= 0.0 ? r : alg3_first_crossing(sh, target, m, b, gm, gb, lm, lb, depth + 1);
}
inline double power_threshold_poly(int shape, double lnp_target) {
    const double sh = (double)shape;
    const double s0 = sh / 1.05 * (1.0 - 1e-12);
    const double hi = 4.0 * power_threshold(shape, lnp_target) + 64.0;
    const double step = 0.01 + 0.01 * std::sqrt(sh);
    auto g = [&](double S) { return alg3_poly(2.0 * S, 2.0 * sh); };
    // sliding window over the grid: g at S − step, S, S + step, S + 2·step; the interval tested is [S, S + step]
    double gm1 = g(s0), g0 = gm1, g1 = g(s0 + step), g2 = g(s0 + 2.0 * step);
    for (double S = s0; S <= hi; S += step) {
        const double d = fmax(fabs(g0 - gm1), fmax(fabs(g1 - g0), fabs(g2 - g1)));   // largest change per step nearby
        if (fmin(g0, g1) - d <= lnp_target) {
            const double l = d / step;
            const double r = alg3_first_crossing(sh, lnp_target, S, S + step, g0, g1, l, l, 0);
            if (r >= 0.0) return r;
        }
        gm1 = g0; g0 = g1; g1 = g2; g2 = g(S + 3.0 * step);
    }
    return hi;
}

} // namespace pulscan
