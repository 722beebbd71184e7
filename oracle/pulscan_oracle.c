/*
 * pulscan_oracle.c — CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, double-precision restatement of what the Pulscan boxcar-search hot path computes
 * (White et al., arXiv 2406.15186; citations are "PAPER.md:L<line>").  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no source, header, table or
 * helper with the CUDA path under paper_2406_15186_b200/csrc/ and neither side includes the other.
 *
 * Every step follows the paper's definition in the paper's order; there is no blocking, pruning, fusion or
 * reordering.  Readings of passages where the paper is silent or garbled are the R-numbers of DESIGN.md §3.
 *
 * Parity pins (tests/test_oracle_*.py): numpy.median / scipy MAD / Φ⁻¹(¾); brute-force and closed-form
 * boxcar sums; mpmath 50-digit χ² tails and normal quantiles (tests/golden/significance_pins.txt);
 * scipy.special.gammaincc / chi2.sf / norm.isf; Exp(1) statistics of normalised noise; injection recovery;
 * the searched-width sets against the paper's printed list (L411) and Alg. 4's remainder rule; the harmonic sum against a
 * ramp's closed form, a numpy reshape route and the χ² degrees of freedom the paper states (KS test); Alg. 1 against a
 * numpy.median route and a hand example; the sampled / harmonic / per-width searches against a scipy route; Alg. 3 against
 * the listing's printed numbers (f(0), the dof >= 1.05·pow branch), an exact rational evaluation of the printed polynomial,
 * and — as the approximation it is — its error against orc_ln_q over (dof, power).
 * Parity unpinned: the paper's Bonferroni trial count (R15) — a plan parameter, default 1; the paper's own candidate lists
 * and the J1227-4853 values of Table 3 (data absent).
 *
 * Precision: float32 inputs are widened to double once; everything else is double.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* κ = 1/Φ⁻¹(3/4): PAPER.md:L142 ("scaled by the factor 1/φ⁻¹(3/4)"); Eq. 8 L147 prints 3/2 (garble, R3);
 * Alg. 1 L648 prints the 5-digit rounding 1.4826. */
#define ORC_KAPPA 1.4826022185056018

typedef struct {
    int32_t spectrum; /* index in the batch                                   */
    int32_t bin;      /* first bin of the window (R10)                        */
    int32_t width;    /* boxcar width w in [1, zmax] (R9)                     */
    int32_t numharm;  /* harmonics summed, H (1 for the plain search); §2.3       */
    double power;     /* S(bin, width), mean-1 units (R2)                     */
    double sigma;     /* Gaussian-equivalent significance (R16)               */
    double lnp;       /* ln of the (Bonferroni-adjusted) p-value              */
} orc_candidate;

static int cmp_double(const void* a, const void* b) {
    double x = *(const double*)a, y = *(const double*)b;
    return (x > y) - (x < y);
}

/* Median of n values: middle order statistic, or the mean of the two middle ones for even n (R4;
 * Alg. 1's local_median).  Sorts a scratch copy (library primitive: qsort). */
double orc_median(const double* v, int64_t n, double* scratch) {
    memcpy(scratch, v, (size_t)n * sizeof(double));
    qsort(scratch, (size_t)n, sizeof(double), cmp_double);
    if (n & 1) return scratch[n / 2];
    return 0.5 * (scratch[n / 2 - 1] + scratch[n / 2]);
}

/* Normalise one real sequence of one block in place: (v − median)/(κ·MAD)  (Eq. 8).
 * MAD = median(|v − median|) (R5).  If κ·MAD is 0 or not finite the block is set to 0 (R7).
 * Returns the median; *scale_out receives κ·MAD. */
double orc_normalise_block(double* v, int64_t n, double* scratch, double* dev, double* scale_out) {
    double med = orc_median(v, n, scratch);
    for (int64_t k = 0; k < n; ++k) dev[k] = fabs(v[k] - med);
    double mad = orc_median(dev, n, scratch);
    double s = ORC_KAPPA * mad;
    if (scale_out) *scale_out = s;
    if (!(s > 0.0) || !isfinite(s)) {
        for (int64_t k = 0; k < n; ++k) v[k] = 0.0;
    } else {
        for (int64_t k = 0; k < n; ++k) v[k] = (v[k] - med) / s;
    }
    return med;
}

/* Steps 1-3: blockwise per-component normalisation, then power.
 * spec: n interleaved (re, im) float32 pairs.  norm_block = B.  Blocks are [jB, (j+1)B) and the last block
 * extends to n (R6).  Real and imaginary parts are normalised independently, then
 * P = (re'^2 + im'^2)/2 (PAPER.md:L150 |X'|^2, halved so that noise has mean 1: R2). */
void orc_normalise_power(const float* spec, int64_t n, int64_t B, double* P) {
    int64_t nb = n / B;
    if (nb < 1) nb = 1;
#pragma omp parallel
    {
        int64_t maxlen = n - (nb - 1) * B; /* the last block is the longest: B + (n mod B), or n if nb = 1 */
        double* re = (double*)malloc((size_t)maxlen * sizeof(double));
        double* im = (double*)malloc((size_t)maxlen * sizeof(double));
        double* scratch = (double*)malloc((size_t)maxlen * sizeof(double));
        double* dev = (double*)malloc((size_t)maxlen * sizeof(double));
#pragma omp for schedule(dynamic, 4)
        for (int64_t j = 0; j < nb; ++j) {
            int64_t lo = j * B;
            int64_t hi = (j == nb - 1) ? n : (j + 1) * B;
            int64_t len = hi - lo;
            for (int64_t k = 0; k < len; ++k) {
                re[k] = (double)spec[2 * (lo + k)];
                im[k] = (double)spec[2 * (lo + k) + 1];
            }
            orc_normalise_block(re, len, scratch, dev, NULL);
            orc_normalise_block(im, len, scratch, dev, NULL);
            for (int64_t k = 0; k < len; ++k) P[lo + k] = 0.5 * (re[k] * re[k] + im[k] * im[k]);
        }
        free(re); free(im); free(scratch); free(dev);
    }
}

/* Step 4 on its own, for tiny inputs: every boxcar sum by the paper's recursion
 * Y_k = Y_{k-1}[:end-1] + X[k:end], i.e. S(i,w) = S(i,w-1) + P[i+w-1].
 * out is [zmax][n] row-major, out[(w-1)*n + i] = S(i,w) for i + w <= n, NaN where the window does not
 * exist (output length n-w+1, R11). */
void orc_boxcar_sums(const double* P, int64_t n, int32_t zmax, double* out) {
    for (int64_t i = 0; i < n; ++i) out[i] = P[i];
    for (int32_t w = 2; w <= zmax; ++w) {
        double* cur = out + (int64_t)(w - 1) * n;
        const double* prev = out + (int64_t)(w - 2) * n;
        for (int64_t i = 0; i < n; ++i) cur[i] = (i + w <= n) ? prev[i] + P[i + w - 1] : NAN;
    }
}

/* Steps 4-5 for one candidate block c = [cC, min((c+1)C, n)) (R12: a window belongs to the block of its first
 * bin): running sums by the recursion, per-width maximum M(c,w) and lowest arg-max I(c,w) (R14).
 * M[w-1] = -1 and I[w-1] = -1 when no window of width w starts in the block (R11).  sums: scratch of C doubles. */
void orc_block_maxima(const double* P, int64_t n, int32_t zmax, int64_t C, int64_t c, double* sums, double* M,
                      int64_t* I) {
    int64_t lo = c * C, hi = lo + C;
    if (hi > n) hi = n;
    for (int64_t i = lo; i < hi; ++i) sums[i - lo] = 0.0;
    for (int32_t w = 1; w <= zmax; ++w) {
        double best = -1.0;
        int64_t arg = -1;
        for (int64_t i = lo; i < hi && i + w <= n; ++i) {
            sums[i - lo] += P[i + w - 1]; /* S(i,w) = S(i,w-1) + P[i+w-1] */
            if (sums[i - lo] > best) { best = sums[i - lo]; arg = i; }
        }
        M[w - 1] = best;
        I[w - 1] = arg;
    }
}

/* ln Q(w,S), Q(w,S) = e^{-S} Σ_{k=0}^{w-1} S^k/k!: the survival function of a χ² variable with 2w degrees of
 * freedom evaluated at 2S (Eq. 9; a width-w boxcar is the sum of w χ²(2) powers, and in mean-1
 * units the χ² statistic is 2S, R2).  Evaluated term by term, normalised at the largest term so that nothing
 * overflows and every term is positive (no cancellation). */
double orc_ln_q(int32_t w, double S) {
    if (!(S > 0.0)) return 0.0;
    int32_t ks = (S >= (double)(w - 1)) ? (w - 1) : (int32_t)floor(S); /* index of the largest term */
    double sum = 1.0, t = 1.0;
    for (int32_t k = ks; k >= 1; --k) { t *= (double)k / S; sum += t; }           /* terms ks-1 … 0 */
    t = 1.0;
    for (int32_t k = ks + 1; k <= w - 1; ++k) { t *= S / (double)k; sum += t; }   /* terms ks+1 … w-1 */
    return -S + (double)ks * log(S) - lgamma((double)ks + 1.0) + log(sum);
}

/* ln of the one-sided normal survival function, ln(½ erfc(x/√2))  (R16). */
double orc_ln_sf(double x) {
    if (x < 0.0) return log1p(-0.5 * erfc(-x / M_SQRT2));
    if (x < 30.0) return log(0.5 * erfc(x / M_SQRT2));
    /* erfc underflows near x = 38: asymptotic series sf(x) = φ(x)/x · Σ (-1)^k (2k-1)!!/x^{2k} */
    double x2 = x * x, term = 1.0, sum = 1.0;
    for (int k = 1; k < 200; ++k) {
        double next = -term * (double)(2 * k - 1) / x2;
        if (fabs(next) >= fabs(term) || fabs(next) < 1e-18) break;
        term = next;
        sum += term;
    }
    return -0.5 * x2 - log(x) - 0.5 * log(2.0 * M_PI) + log(sum);
}

/* Gaussian-equivalent σ of a p-value given as ln p: the x with ln sf(x) = ln p (R16).  Plain bisection. */
double orc_sigma_from_lnp(double lnp) {
    if (!(lnp < 0.0)) return -INFINITY;
    double lo = -40.0, hi = 1.0;
    if (orc_ln_sf(lo) < lnp) return lo;
    while (orc_ln_sf(hi) > lnp) hi *= 2.0;
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (orc_ln_sf(mid) > lnp) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

/* ---- Algorithm 3 (§2.6, Eq. 10-12): the paper's GPU significance, an APPROXIMATION of ln p
 * obtained "by linear regression": Device function power_to_logp(pow, dof):
 *     if dof >= pow × 1.05 then logp ← 0.0
 *     else x ← 1500 × dof/pow;  f(x) ← A_2·x^16 + A_3·x^15 + … + A_17·x + A_18;  logp ← pow × f(x)/1500
 * with the 17 coefficients printed in the listing (A_1 = 1500).  Followed term by term in the printed order, in double.
 * Reading R31: `pow` and `dof` are in the paper's own units, |X'|² summed over the window and its χ² degrees of freedom
 * (Eq. 9: 2(z+1); L220: H(H+1)(z+1)), i.e. pow = 2S and dof = 2·shape in the mean-1 units of this file (R2): the
 * listing's own branch "dof >= 1.05·pow → 0" says pow has mean dof, and f(0)/1500 = −0.5035 ≈ −½ is the χ² tail's
 * exponent −pow/2.  The paper's logarithm is natural (Table 3: GPU ln p = −171.34 beside σ = 18.8). */
double orc_power_to_logp(double pow_, double dof) {
    if (dof >= pow_ * 1.05) return 0.0;
    double x = 1500.0 * dof / pow_;
    double f = -4.4604059e-46 * pow(x, 16) + 9.4927863e-42 * pow(x, 15)
             - 9.1470451e-38 * pow(x, 14) + 5.2810851e-34 * pow(x, 13)
             - 2.0376166e-30 * pow(x, 12) + 5.5480334e-27 * pow(x, 11)
             - 1.0973877e-23 * pow(x, 10) + 1.5991804e-20 * pow(x, 9)
             - 1.7231488e-17 * pow(x, 8) + 1.3660070e-14 * pow(x, 7)
             - 7.8617952e-12 * pow(x, 6) + 3.2136336e-9 * pow(x, 5)
             - 9.0466418e-7 * pow(x, 4) + 0.00016945948 * pow(x, 3)
             - 0.021494231 * pow(x, 2) + 2.9515954 * x - 755.24091;
    return pow_ * f / 1500.0;
}

/* ---- Algorithm 1: the paper's GPU normalisation, an APPROXIMATE median ("median of medians",
 * L232 "threads recursively find the median of 4 non-overlapping elements").  Followed step by step:
 *   local_median(a,b,c,d) = (a+b+c+d − min − max)/2                                             (L627-631)
 *   for strides ← count/4, count/16, …, 1:  sdata[i] ← local_median(sdata[i], sdata[i+stride], sdata[i+2·stride],
 *                                                                    sdata[i+3·stride]),  i < stride        (L636-642)
 * Reading R30: the count must be 4^k or 2·4^k; a last level of two values returns their mean (the median of two).
 * The input is overwritten. */
static double orc_local_median(double a, double b, double c, double d) {
    double mn = fmin(fmin(fmin(a, b), c), d);
    double mx = fmax(fmax(fmax(a, b), c), d);
    return (a + b + c + d - mn - mx) / 2.0;
}

double orc_median_of_medians(double* sdata, int64_t count) {
    while (count >= 4) {
        int64_t stride = count / 4;
        for (int64_t i = 0; i < stride; ++i)
            sdata[i] = orc_local_median(sdata[i], sdata[i + stride], sdata[i + 2 * stride], sdata[i + 3 * stride]);
        count = stride;
    }
    if (count == 2) return 0.5 * (sdata[0] + sdata[1]);
    return sdata[0];
}

/* Alg. 1's Procedure (L643-649) for every chunk of B bins, per component (L140): median ← median_of_medians(chunk);
 * MAD ← median_of_medians(|chunk − median|) (the listing omits the absolute value, R5); scale_factor ← 1.4826 (the
 * 5-digit constant the listing prints); normalised ← (chunk − median)/(scale_factor·MAD); then P = |X'|²/2 (R2).
 * Reading R30: chunk j is bins [jB, (j+1)B); the n mod B bins after the last chunk are normalised with the last chunk's
 * median and MAD (Alg. 1 reduces exactly one chunk of 4·blockDim values); MAD = 0 → 0 (R7).  Needs n ≥ B. */
void orc_normalise_power_mom(const float* spec, int64_t n, int64_t B, double* P) {
    int64_t nb = n / B;
    double* buf = (double*)malloc((size_t)B * sizeof(double));
    for (int64_t j = 0; j < nb; ++j) {
        int64_t lo = j * B;
        int64_t hi = (j == nb - 1) ? n : (j + 1) * B;
        double med[2], scale[2];
        for (int comp = 0; comp < 2; ++comp) {
            for (int64_t k = 0; k < B; ++k) buf[k] = (double)spec[2 * (lo + k) + comp];
            med[comp] = orc_median_of_medians(buf, B);
            for (int64_t k = 0; k < B; ++k) buf[k] = fabs((double)spec[2 * (lo + k) + comp] - med[comp]);
            scale[comp] = 1.4826 * orc_median_of_medians(buf, B);
        }
        for (int64_t k = lo; k < hi; ++k) {
            double x = (scale[0] > 0.0 && isfinite(scale[0])) ? ((double)spec[2 * k] - med[0]) / scale[0] : 0.0;
            double y = (scale[1] > 0.0 && isfinite(scale[1])) ? ((double)spec[2 * k + 1] - med[1]) / scale[1] : 0.0;
            P[k] = 0.5 * (x * x + y * y);
        }
    }
    free(buf);
}

/* Power S at which a width-w boxcar reaches ln p = lnp_target (used only to check threshold tables). */
double orc_power_threshold(int32_t w, double lnp_target) {
    double lo = 0.0, hi = (double)w + 10.0;
    while (orc_ln_q(w, hi) > lnp_target) hi *= 2.0;
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (orc_ln_q(w, mid) > lnp_target) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

/* The whole path for a batch (steps 1-8).  spectra: [batch][pitch] complex64 as interleaved float32, n bins used
 * per row.  Returns the number of candidates found; at most cap are written, ordered by (spectrum, bin) (R19).
 *   per block c, per width w: ln p(c,w) = ln Q(w, M(c,w));  ln p_adj = min(0, ln p + ln n_trials)        (R15)
 *   w* = the width with the smallest ln p_adj (= the largest σ, σ being a decreasing function of ln p);
 *        the smallest such w on exact ties                                                            (R13)
 *   emit (b, I(c,w*), w*, M(c,w*), σ) iff ln p_adj <= ln sf(sigma_threshold)  (σ >= threshold)          (R17)
 */
int64_t orc_search_sampled(const float* spectra, int64_t batch, int64_t n, int64_t pitch, int32_t zmax, int64_t B,
                           int64_t C, double sigma_threshold, double n_trials, int32_t z_step, int32_t log_sampling,
                           orc_candidate* out, int64_t cap);
int64_t orc_search_ex(const float* spectra, int64_t batch, int64_t n, int64_t pitch, int32_t zmax, int64_t B, int64_t C,
                      double sigma_threshold, double n_trials, int32_t z_step, int32_t log_sampling, int32_t r_block,
                      orc_candidate* out, int64_t cap);

int64_t orc_search(const float* spectra, int64_t batch, int64_t n, int64_t pitch, int32_t zmax, int64_t B,
                   int64_t C, double sigma_threshold, double n_trials, orc_candidate* out, int64_t cap) {
    return orc_search_sampled(spectra, batch, n, pitch, zmax, B, C, sigma_threshold, n_trials, 1, 0, out, cap);
}

/* Which boxcar widths are SEARCHED for candidates (all are computed): "the user can select the step size
 * to determine which boxcar filtered spectra are searched"; Alg. 4 L693-695 searches drift z (from 0) when
 * remainder(z / z_step) = 0, "this condition on z can be replaced with a check for if the current z is a power of 2
 * for logarithmic sampling"; L411 "only search logarithmically spaced (i.e. z = 1, 2, 4, 8, ... z-max) boxcar filter
 * widths".  The width is w = z + 1 (R9).  Reading R28: z = 0 (the unfiltered spectrum) is searched in both modes, as
 * Alg. 4's loop starts at z = 0 and remainder(0 / z_step) = 0. */
int32_t orc_width_searched(int32_t w, int32_t z_step, int32_t log_sampling) {
    int32_t z = w - 1;
    if (log_sampling) return z == 0 || (z & (z - 1)) == 0;
    return z % z_step == 0;
}

/* orc_search restricted to the searched widths: the reduction over widths (R13) runs over those only. */
int64_t orc_search_sampled(const float* spectra, int64_t batch, int64_t n, int64_t pitch, int32_t zmax, int64_t B,
                           int64_t C, double sigma_threshold, double n_trials, int32_t z_step, int32_t log_sampling,
                           orc_candidate* out, int64_t cap) {
    return orc_search_ex(spectra, batch, n, pitch, zmax, B, C, sigma_threshold, n_trials, z_step, log_sampling, 0, out, cap);
}

/* ... and, with r_block != 0, "Pulscan R-Block" (§2.4): "simply saving the block index (an approximate
 * frequency location) of candidates rather than the exact r-bin they came from".  The record's bin is then the first bin
 * of the candidate block, block index × block width (Table 3: R-Block r = 360448 = 11 × 32768 against the exact
 * 364318); width, power and significance are unchanged. */
int64_t orc_search_ex(const float* spectra, int64_t batch, int64_t n, int64_t pitch, int32_t zmax, int64_t B, int64_t C,
                      double sigma_threshold, double n_trials, int32_t z_step, int32_t log_sampling, int32_t r_block,
                      orc_candidate* out, int64_t cap) {
    int64_t nblk = (n + C - 1) / C;
    double ln_trials = log(n_trials);
    double lnp_thr = orc_ln_sf(sigma_threshold);
    double* P = (double*)malloc((size_t)n * sizeof(double));
    orc_candidate* blockbest = (orc_candidate*)malloc((size_t)nblk * sizeof(orc_candidate));
    int64_t found = 0;
    for (int64_t b = 0; b < batch; ++b) {
        orc_normalise_power(spectra + 2 * b * pitch, n, B, P);
#pragma omp parallel
        {
            double* sums = (double*)malloc((size_t)C * sizeof(double));
            double* M = (double*)malloc((size_t)zmax * sizeof(double));
            int64_t* I = (int64_t*)malloc((size_t)zmax * sizeof(int64_t));
#pragma omp for schedule(dynamic, 16)
            for (int64_t c = 0; c < nblk; ++c) {
                orc_block_maxima(P, n, zmax, C, c, sums, M, I);
                double best_lnp = INFINITY;
                int32_t best_w = 0;
                for (int32_t w = 1; w <= zmax; ++w) {
                    if (I[w - 1] < 0) continue; /* no window of this width starts in the block */
                    if (!orc_width_searched(w, z_step, log_sampling)) continue;
                    double lnp = orc_ln_q(w, M[w - 1]) + ln_trials;
                    if (lnp > 0.0) lnp = 0.0;
                    if (lnp < best_lnp) { best_lnp = lnp; best_w = w; } /* strict: smallest w on ties */
                }
                orc_candidate r;
                memset(&r, 0, sizeof r);
                r.spectrum = -1;
                if (best_w > 0 && best_lnp <= lnp_thr) {
                    r.spectrum = (int32_t)b;
                    r.bin = r_block ? (int32_t)(c * C) : (int32_t)I[best_w - 1];
                    r.width = best_w;
                    r.numharm = 1;
                    r.power = M[best_w - 1];
                    r.lnp = best_lnp;
                    r.sigma = orc_sigma_from_lnp(best_lnp);
                }
                blockbest[c] = r;
            }
            free(sums); free(M); free(I);
        }
        for (int64_t c = 0; c < nblk; ++c) { /* blocks in order: the list comes out sorted by (spectrum, bin) */
            if (blockbest[c].spectrum < 0) continue;
            if (found < cap) out[found] = blockbest[c];
            ++found;
        }
    }
    free(P); free(blockbest);
    return found;
}

/* Harmonic sum by decimation (§2.3).  "Summing adjacent non-overlapping pairs, triples, quartets,
 * etc. of frequency magnitudes to produce a magnitude spectra decimated by factors of 2, 3, 4": D_h(r) = Σ_{j<h} P[h·r + j].
 * "We then sum the overlapping sections of each decimated spectra (aligned so the 0th bin of each spectrum is summed) and
 * discard the non-overlapping parts": Y_H(r) = Σ_{h=1}^{H} D_h(r) for r in [0, floor(n/H)), which in noise is χ² with
 * Σ 2h = H(H+1) degrees of freedom (L214-216) — in the mean-1 units used here (R2) a Gamma variate of shape H(H+1)/2.
 * Reading R29: only complete groups count, so Y_H has floor(n/H) bins.  Returns that length; Y must hold it. */
int64_t orc_harmonic_sum(const double* P, int64_t n, int32_t H, double* Y) {
    int64_t nH = n / H;
    for (int64_t r = 0; r < nH; ++r) {
        double y = 0.0;
        for (int32_t h = 1; h <= H; ++h)
            for (int32_t j = 0; j < h; ++j) y += P[(int64_t)h * r + j];
        Y[r] = y;
    }
    return nH;
}

/* The search with harmonic summing: for H = 1..numharm the summed spectrum Y_H is boxcar-filtered "as previously
 * described", the output being χ² with H(H+1)(z+1) degrees of freedom (L220): ln p = ln Q(w·H(H+1)/2, S) in mean-1
 * units.  Candidate blocks, widths (zmax, sampling), the reduction over widths (R13), the threshold and R-Block are as in
 * orc_search_ex, applied to each Y_H on its own (bins are those of Y_H, i.e. of the fundamental); a width needs
 * w < floor(n/H) to exist.  Records carry numharm = H and come out ordered by (H, spectrum, bin).  Normalisation happens
 * once, on the full-resolution spectrum, before the decimation (Table 4's kernel order L571-578). */
int64_t orc_search_general(const float* spectra, int64_t batch, int64_t n, int64_t pitch, int32_t zmax, int64_t B,
                           int64_t C, double sigma_threshold, double n_trials, int32_t z_step, int32_t log_sampling,
                           int32_t r_block, int32_t numharm, int32_t norm_mode, orc_candidate* out, int64_t cap);

int64_t orc_search_harmonics(const float* spectra, int64_t batch, int64_t n, int64_t pitch, int32_t zmax, int64_t B,
                             int64_t C, double sigma_threshold, double n_trials, int32_t z_step, int32_t log_sampling,
                             int32_t r_block, int32_t numharm, orc_candidate* out, int64_t cap) {
    return orc_search_general(spectra, batch, n, pitch, zmax, B, C, sigma_threshold, n_trials, z_step, log_sampling, r_block,
                              numharm, 0, out, cap);
}

/* … and with norm_mode = 1 the normalisation is the paper's GPU one (Alg. 1, orc_normalise_power_mom) instead of the exact
 * median/MAD; everything after the power spectrum is unchanged. */
int64_t orc_search_opts(const float* spectra, int64_t batch, int64_t n, int64_t pitch, int32_t zmax, int64_t B,
                        int64_t C, double sigma_threshold, double n_trials, int32_t z_step, int32_t log_sampling,
                        int32_t r_block, int32_t numharm, int32_t norm_mode, int32_t per_width, orc_candidate* out, int64_t cap);

int64_t orc_search_general(const float* spectra, int64_t batch, int64_t n, int64_t pitch, int32_t zmax, int64_t B,
                           int64_t C, double sigma_threshold, double n_trials, int32_t z_step, int32_t log_sampling,
                           int32_t r_block, int32_t numharm, int32_t norm_mode, orc_candidate* out, int64_t cap) {
    return orc_search_opts(spectra, batch, n, pitch, zmax, B, C, sigma_threshold, n_trials, z_step, log_sampling, r_block,
                           numharm, norm_mode, 0, out, cap);
}

/* … and with per_width != 0 the paper's GPU output: instead of the best width per block (R13), one record per
 * (block, searched width) whose maximum reaches the threshold (Alg. 4: thread 0 "writes out [the] local candidate"
 * of every searched z; L322 "highest sigma candidate" is picked afterwards).  Ordered by (H, spectrum, block, width). */
int64_t orc_search_all(const float* spectra, int64_t batch, int64_t n, int64_t pitch, int32_t zmax, int64_t B,
                       int64_t C, double sigma_threshold, double n_trials, int32_t z_step, int32_t log_sampling,
                       int32_t r_block, int32_t numharm, int32_t norm_mode, int32_t per_width, int32_t signif_mode,
                       orc_candidate* out, int64_t cap);

int64_t orc_search_opts(const float* spectra, int64_t batch, int64_t n, int64_t pitch, int32_t zmax, int64_t B,
                        int64_t C, double sigma_threshold, double n_trials, int32_t z_step, int32_t log_sampling,
                        int32_t r_block, int32_t numharm, int32_t norm_mode, int32_t per_width, orc_candidate* out, int64_t cap) {
    return orc_search_all(spectra, batch, n, pitch, zmax, B, C, sigma_threshold, n_trials, z_step, log_sampling, r_block,
                          numharm, norm_mode, per_width, 0, out, cap);
}

/* ln p of a width-w maximum S of the spectrum summed over H harmonics (shape = w·H(H+1)/2 in mean-1 units):
 * signif_mode 0: the exact χ² tail (Eq. 9); 1: the paper's GPU approximation, Alg. 3, called with the paper's units
 * pow = 2S, dof = 2·shape (R31). */
static double orc_lnp_of(int32_t signif_mode, int32_t shape, double S) {
    if (signif_mode) return orc_power_to_logp(2.0 * S, 2.0 * (double)shape);
    return orc_ln_q(shape, S);
}

/* … and with signif_mode = 1 every ln p comes from Alg. 3's polynomial instead of the exact tail (the paper's GPU-native
 * configuration: Alg. 1 + Alg. 3 + log-spaced widths + harmonic sum, L544, Fig. 10); the reduction over widths, the
 * threshold (ln p <= ln sf(σ_thr): "compared with precomputed threshold values", L342-344) and σ = Φ_sf⁻¹(e^{ln p}) then
 * use that value.  Nothing else changes. */
int64_t orc_search_all(const float* spectra, int64_t batch, int64_t n, int64_t pitch, int32_t zmax, int64_t B,
                       int64_t C, double sigma_threshold, double n_trials, int32_t z_step, int32_t log_sampling,
                       int32_t r_block, int32_t numharm, int32_t norm_mode, int32_t per_width, int32_t signif_mode,
                       orc_candidate* out, int64_t cap) {
    double ln_trials = log(n_trials);
    double lnp_thr = orc_ln_sf(sigma_threshold);
    double* P = (double*)malloc((size_t)n * sizeof(double));
    double* Y = (double*)malloc((size_t)n * sizeof(double));
    int64_t found = 0;
    for (int32_t H = 1; H <= numharm; ++H) {
        int32_t kappa = H * (H + 1) / 2;
        for (int64_t b = 0; b < batch; ++b) {
            if (norm_mode) orc_normalise_power_mom(spectra + 2 * b * pitch, n, B, P);
            else orc_normalise_power(spectra + 2 * b * pitch, n, B, P);
            int64_t nH = orc_harmonic_sum(P, n, H, Y);
            int64_t nblk = (nH + C - 1) / C;
            orc_candidate* blockbest = (orc_candidate*)malloc((size_t)nblk * sizeof(orc_candidate));
#pragma omp parallel
            {
                double* sums = (double*)malloc((size_t)C * sizeof(double));
                double* M = (double*)malloc((size_t)zmax * sizeof(double));
                int64_t* I = (int64_t*)malloc((size_t)zmax * sizeof(int64_t));
#pragma omp for schedule(dynamic, 16)
                for (int64_t c = 0; c < nblk; ++c) {
                    orc_block_maxima(Y, nH, zmax, C, c, sums, M, I);
                    double best_lnp = INFINITY;
                    int32_t best_w = 0;
                    for (int32_t w = 1; w <= zmax; ++w) {
                        if (I[w - 1] < 0) continue;
                        if (!orc_width_searched(w, z_step, log_sampling)) continue;
                        double lnp = orc_lnp_of(signif_mode, w * kappa, M[w - 1]) + ln_trials;
                        if (lnp > 0.0) lnp = 0.0;
                        if (lnp < best_lnp) { best_lnp = lnp; best_w = w; }
                    }
                    orc_candidate r;
                    memset(&r, 0, sizeof r);
                    r.spectrum = -1;
                    if (best_w > 0 && best_lnp <= lnp_thr) {
                        r.spectrum = (int32_t)b;
                        r.bin = r_block ? (int32_t)(c * C) : (int32_t)I[best_w - 1];
                        r.width = best_w;
                        r.numharm = H;
                        r.power = M[best_w - 1];
                        r.lnp = best_lnp;
                        r.sigma = orc_sigma_from_lnp(best_lnp);
                    }
                    blockbest[c] = r;
                }
                free(sums); free(M); free(I);
            }
            for (int64_t c = 0; c < nblk && !per_width; ++c) {
                if (blockbest[c].spectrum < 0) continue;
                if (found < cap) out[found] = blockbest[c];
                ++found;
            }
            free(blockbest);
            if (per_width) { /* plain serial loop: every (block, searched width) above the threshold */
                double* sums = (double*)malloc((size_t)C * sizeof(double));
                double* M = (double*)malloc((size_t)zmax * sizeof(double));
                int64_t* I = (int64_t*)malloc((size_t)zmax * sizeof(int64_t));
                for (int64_t c = 0; c < nblk; ++c) {
                    orc_block_maxima(Y, nH, zmax, C, c, sums, M, I);
                    for (int32_t w = 1; w <= zmax; ++w) {
                        if (I[w - 1] < 0 || !orc_width_searched(w, z_step, log_sampling)) continue;
                        double lnp = orc_lnp_of(signif_mode, w * kappa, M[w - 1]) + ln_trials;
                        if (lnp > 0.0) lnp = 0.0;
                        if (lnp > lnp_thr) continue;
                        orc_candidate r;
                        memset(&r, 0, sizeof r);
                        r.spectrum = (int32_t)b;
                        r.bin = r_block ? (int32_t)(c * C) : (int32_t)I[w - 1];
                        r.width = w; r.numharm = H; r.power = M[w - 1]; r.lnp = lnp;
                        r.sigma = orc_sigma_from_lnp(lnp);
                        if (found < cap) out[found] = r;
                        ++found;
                    }
                }
                free(sums); free(M); free(I);
            }
        }
    }
    free(P); free(Y);
    return found;
}

int orc_num_threads(void) {
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        n = __builtin_omp_get_num_threads();
    }
#endif
    return n;
}

double orc_kappa(void) { return ORC_KAPPA; }
