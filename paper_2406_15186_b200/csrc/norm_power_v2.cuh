// norm_power_v2.cuh — kernel (a), single-histogram path: full normalisation blocks of exactly B = EPT·NT bins.
//
// Same result as norm_power.cuh's general path (exact medians, Eq. 8).  What is different:
//  * the block (B complex64 = 8·B bytes) is staged in shared memory by ONE TMA bulk copy and every pass re-reads it
//    with conflict-free LDS.64, so the values never occupy registers;
//  * ONE histogram pass per component serves the median AND the MAD.  The 2048 value-linear buckets span
//    mean ± 2·sd of a 128-bin sample (warp 0 computes it while the others zero the histograms);
//    bucket = RN(2047·sat(v·scale + off)), taken from the mantissa of fma(t, 2047·2⁻²², 2.0f), whose bit pattern
//    0x40000000 | idx turns into the histogram byte offset with one shift (the 0x4 falls off the top);
//  * the median's bucket jm comes from a two-level scan (16-bucket chunk sums by all threads, then one warp per
//    component).  The two central values lie in buckets jm and jm+e, so the median m lies in the (half-integer)
//    bucket c2/2, c2 = 2·jm + e.  The MAD is the median of |v − m|: with t = |2·bucket − c2| the "shell" of a bucket,
//    the first shell t1 with #{t ≤ t1} > rank brackets it, and shells t1−2 … t1+2 contain it: the same histogram,
//    folded about c2/2, locates the MAD;
//  * membership of a value in (median net ∪ MAD shells) is ONE test on the bucket indices kept packed two per
//    register and read as fp16 pairs (bucket indices ≤ 2047 sit in fp16's denormal + first binade, where the
//    encoding is linear, so HFMA2/HADD2 do exact integer arithmetic on them):
//        z = ||4·(idx − ⌊c2/2⌋)| − K| − K,   member ⇔ |z| ≤ HW   (2t ∈ [0, HW] ∪ [2K − HW, 2K + HW])
//    five half2 instructions per two values; the hits (≈ 30 of 4096) are re-read, classified exactly (median net or MAD
//    shells) and appended to the list of their class, the re-reads of both components in flight together;
//  * one warp per component ranks the ≤ 64 median-net members and the ≤ 64 shell members exactly, and VERIFIES that
//    no value outside the shells can lie between the two central deviations (bucket boundaries mapped back to values
//    in double, with a margin).  Anything unusual (degenerate sample, lists too long, verification failed) sends the
//    block id to the redo list and norm_power_redo_kernel runs it through the general path.
// Six CTA barriers per block.
#pragma once
#include <cstdint>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include "norm_power.cuh"

#ifndef PULSCAN_V2_SAMPLE_AHEAD
#define PULSCAN_V2_SAMPLE_AHEAD 0
#endif
#ifndef PULSCAN_NORM_OCC128_SMALL
#define PULSCAN_NORM_OCC128_SMALL 10   /* EPT <= 16 fits 48 registers without spills: cfg 5 kernel (a) 8.85 -> 8.61 ms */
#endif
#ifndef PULSCAN_NORM_OCC128
#define PULSCAN_NORM_OCC128 8
#endif

namespace pulscan {

constexpr int kV2NB = 2048;            // buckets per component
constexpr int kV2KPT = 16;             // buckets per chunk
constexpr int kV2NCH = kV2NB / kV2KPT; // chunks per component (128)
constexpr int kV2ListCap = 128;        // gathered members per component
constexpr int kV2ClsCap = 64;          // median-net / shell members per component (2 per lane)
#ifndef PULSCAN_V2_RANGE
#define PULSCAN_V2_RANGE 2.0f   /* measured at cfg 3: 2.5 → 3.25 ms, 2.0 → 3.20 ms, 1.75 → 3.16 ms but 127 blocks redone, 1.5 → 48 k redone */
#endif
constexpr float kV2Range = PULSCAN_V2_RANGE;       // histogram spans mean ± kV2Range·sd of the sample
constexpr float kV2IdxScale = 2047.0f * 2.384185791015625e-07f;  // 2047·2⁻²²

struct alignas(16) V2Ctl {
    unsigned long long mbar;
    unsigned cls_n[2][2];             // members gathered so far: [component][0: median net, 1: shells]
    int fail;                         // 0 = ok; 1 degenerate geometry, 2 search window, 3 list capacity, 4 verification, 5 sample
    float scale[2], off[2];           // bucket map of each component
    int c2[2];                        // 2·jm + e: twice the (half-integer) bucket of the median
    int t0[2], tE[2], tm[2];          // shells [t0, tE] of t = |2·bucket − c2| hold the MAD; median net t ≤ tm
    unsigned hc2[2], hK[2], hHW[2];   // membership-test constants as fp16 pairs (−4·⌊c2/2⌋, K, HW' in bucket units of 2⁻²⁴)
    unsigned n_in[2], excl_med[2];    // values strictly inside the shells; values below the median net
    unsigned n_med[2], n_shl[2];      // values in the median net / in the shells (what the gather must deliver)
    float a[2], h[2], inv[2];         // median = a + h (a = lower central value, h = half the gap); 1/(√2·κ·MAD)
    alignas(16) unsigned chunk_tot[2][kV2NCH];
    alignas(16) unsigned CE[2][kV2NCH + 4];   // exclusive prefix of chunk_tot; CE[NCH] = B
    float cls[2][2][kV2ClsCap + 4];   // [component][0: median net, 1: shells (values, then deviations)], +inf padded to a multiple of 4
};

__device__ __forceinline__ unsigned v2_smem(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void v2_red_inc(unsigned addr) {
    asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(addr) : "memory");
}

// Bucket of one value: bits = 0x40000000 | idx, idx = RN(2047·sat(v·scale + off)) ∈ [0, 2047].  Monotone in v.
__device__ __forceinline__ unsigned v2_bucket_bits(float v, float scale, float off) {
    const float t = __saturatef(__fmaf_rn(v, scale, off));
    return __float_as_uint(__fmaf_rn(t, kV2IdxScale, 2.0f));
}

// One warp: location and spread of the block from 128 of its bins (four runs of 32 consecutive bins) → the bucket
// map (scale, off) of both components in ctl; ctl.fail = 5 if the sample is degenerate.
template <int B>
__device__ __forceinline__ void v2_estimate(const float2* __restrict__ sdat, V2Ctl& ctl) {
    const int lane = threadIdx.x & 31;
    const float2 pv = sdat[0];
    float q[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float2 s = sdat[k * (B / 4) + lane];
        const float r = s.x - pv.x, i = s.y - pv.y;
        q[0] += r; q[1] = __fmaf_rn(r, r, q[1]); q[2] += i; q[3] = __fmaf_rn(i, i, q[3]);
    }
    // transposing butterfly: 4 sums over 32 lanes with 2 + 1 + 3 shuffles; lanes 8k … 8k+7 end up with quantity k
    const bool up = lane & 16;
    const float k0 = up ? q[2] : q[0], k1 = up ? q[3] : q[1], g0 = up ? q[0] : q[2], g1 = up ? q[1] : q[3];
    const float a0 = k0 + __shfl_xor_sync(0xffffffffu, g0, 16);
    const float a1 = k1 + __shfl_xor_sync(0xffffffffu, g1, 16);
    const bool up8 = lane & 8;
    float x = (up8 ? a1 : a0) + __shfl_xor_sync(0xffffffffu, up8 ? a0 : a1, 8);
    x += __shfl_xor_sync(0xffffffffu, x, 4);
    x += __shfl_xor_sync(0xffffffffu, x, 2);
    x += __shfl_xor_sync(0xffffffffu, x, 1);
    const float s1 = __shfl_sync(0xffffffffu, x, lane & 16);          // Σ of my component (lanes < 16: re; ≥ 16: im)
    const float s2 = __shfl_sync(0xffffffffu, x, (lane & 16) + 8);    // Σ of squares
    const float mean = s1 * (1.f / 128.f);
    const float var = __fmaf_rn(-mean, mean, s2 * (1.f / 128.f));
    const float sc = rsqrtf(var) * (1.f / (2.f * kV2Range));
    const float centre = (up ? pv.y : pv.x) + mean;
    const float of = __fmaf_rn(-centre, sc, 0.5f);
    const bool ok = (var > 0.f) && isfinite(sc) && isfinite(of) && fabsf(of) <= 64.f;
    if ((lane & 15) == 0) {
        ctl.scale[lane >> 4] = sc; ctl.off[lane >> 4] = of;
        if (!ok) ctl.fail = 5;
    }
}

// #values in buckets [0, p), p ∈ [0, NB], from the chunk prefix CE and the fine counts L; p may differ per lane.
__device__ __forceinline__ unsigned v2_count_below(const unsigned* __restrict__ L, const unsigned* __restrict__ CE, int p) {
    const int ch = p >> 4, rem = p & 15;
    unsigned a = CE[ch];
    const unsigned* q = L + (ch << 4);
#pragma unroll
    for (int j = 0; j < kV2KPT - 1; ++j)
        if (j < rem) a += q[j];
    return a;
}

__device__ __forceinline__ unsigned v2_incl_scan(unsigned x) {
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += t;
    }
    return x;
}

// One warp, one component: from the chunk totals and the fine histogram L, find the median bucket jm, the bucket
// jm+e of the next central value, the shells that contain the MAD, and publish the membership-test constants.
// kk = (B−1)/2 is the 0-based rank of the lower central value; even B also needs rank kk+1.
template <int B>
__device__ __forceinline__ void v2_locate(V2Ctl& ctl, const unsigned* __restrict__ L, int c) {
    constexpr unsigned kk = (unsigned)((B - 1) >> 1);
    constexpr bool kEven = (B & 1) == 0;
    const int lane = threadIdx.x & 31;
    unsigned* CE = ctl.CE[c];
    // ---- exclusive prefix over the 128 chunk totals, 4 per lane
    const uint4 ct = reinterpret_cast<const uint4*>(ctl.chunk_tot[c])[lane];
    const unsigned p1 = ct.x, p2 = p1 + ct.y, p3 = p2 + ct.z, sum = p3 + ct.w;
    const unsigned incl = v2_incl_scan(sum);
    const unsigned base = incl - sum;
    reinterpret_cast<uint4*>(CE)[lane] = make_uint4(base, base + p1, base + p2, base + p3);
    if (lane == 31) CE[kV2NCH] = incl;
    __syncwarp();
    // ---- chunk holding rank kk = number of chunks that end at or below kk
    const unsigned nle = (base + p1 <= kk) + (base + p2 <= kk) + (base + p3 <= kk) + (incl <= kk);
    const int cj = (int)__reduce_add_sync(0xffffffffu, nle);
    if (cj >= kV2NCH) { if (lane == 0) ctl.fail = 1; return; }       // histogram does not hold B values: cannot happen
    // ---- fine view: the 32 buckets from the start of that chunk
    const int fb = cj << 4;
    const unsigned cnt = (fb + lane < kV2NB) ? L[fb + lane] : 0u;
    const unsigned finc = v2_incl_scan(cnt);
    const unsigned eb = CE[cj];
    const unsigned below = __ballot_sync(0xffffffffu, eb + finc <= kk);   // a prefix of the lanes
    const int jl = __popc(below);                                       // < 16: rank kk lies in chunk cj
    const int jm = fb + jl;
    const unsigned top_jm = eb + __shfl_sync(0xffffffffu, finc, jl);    // values in buckets ≤ jm
    int e = 0;
    if (kEven && kk + 1 >= top_jm) {                                    // rank kk+1 is in the next non-empty bucket
        const unsigned later = __ballot_sync(0xffffffffu, cnt > 0 && lane > jl);
        if (!later) { if (lane == 0) ctl.fail = 2; return; }
        e = __ffs(later) - 1 - jl;
    }
    // ---- shells.  With σ ≥ 0, G(σ) = #{buckets in [jm + e0 − σ, jm + e1 + σ]} = #{t ≤ 2σ + (e & 1)}.
    // Coarse: whole chunks around chunk cj bracket G from both sides and give the first window of 32 candidates.
    const int e0 = e >> 1, e1 = e - e0, c2 = 2 * jm + e;
    const unsigned gc = CE[min(kV2NCH, cj + 1 + lane)] - CE[max(0, cj - lane)];
    const unsigned coarse = __ballot_sync(0xffffffffu, gc >= kk + 1);
    if (!coarse) { if (lane == 0) ctl.fail = 2; return; }
    const int lstar = __ffs(coarse) - 1;
    const int ws = max(0, kV2KPT * (lstar - 1) - e1 + 1);
    int sg1 = -1, sg2 = -1;
    for (int it = 0; it < 4 && sg2 < 0; ++it) {
        const int w0 = ws + 32 * it;
        // upper ends jm+e1+w0+1+lane: exclusive scan from a uniform start; lower ends jm+e0−w0−lane: scan downwards
        const int H0 = min(jm + e1 + w0 + 1, kV2NB), L0 = max(jm + e0 - w0, 0);
        // #values in buckets [L0, H0): two chunk prefixes and one warp sum of the two partial chunks (modulo 2³², like g below)
        const unsigned partH = lane < (H0 & 15) ? L[(H0 & ~15) + lane] : 0u, partL = lane < (L0 & 15) ? L[(L0 & ~15) + lane] : 0u;
        const unsigned a0 = CE[H0 >> 4] - CE[L0 >> 4] + __reduce_add_sync(0xffffffffu, partH - partL);
        const unsigned xh = (H0 + lane < kV2NB) ? L[H0 + lane] : 0u;
        const unsigned xl = (lane >= 1 && L0 - lane >= 0) ? L[L0 - lane] : 0u;
        // G at σ = w0 + lane: a0 + (xh of the lanes below) + (xl up to this lane) = a0 + scan(xh + xl) − xh: one scan
        const unsigned g = a0 + v2_incl_scan(xh + xl) - xh;
        const unsigned f1 = __ballot_sync(0xffffffffu, g >= kk + 1);
        const unsigned f2 = kEven ? __ballot_sync(0xffffffffu, g >= kk + 2) : f1;
        if (sg1 < 0 && f1) sg1 = w0 + __ffs(f1) - 1;
        if (f2) sg2 = w0 + __ffs(f2) - 1;
    }
    if (sg1 < 0 || sg2 < 0) { if (lane == 0) ctl.fail = 2; return; }
    // The two central deviations lie in ((t1/2 − 1)·h, (t2/2 + 1)·h]: shells t1−2 … t2+2 hold them (h = bucket width).
    const int par = e & 1;
    const int t0 = 2 * sg1 + par - 2, tE = 2 * sg2 + par + 2;
    const int K = (t0 + tE) >> 1;
    const int HW = max(tE - t0, 2 * e);
    const int t0n = K - (HW >> 1), tEn = K + (HW >> 1), tm = HW >> 1;   // the nets the test really selects
    // The test runs on 4·(idx − ⌊c2/2⌋), every term a multiple of 4 and therefore exact in fp16 up to 8188; for odd c2
    // it sees t ± 1 and its half-width is widened by one shell (the extra members are dropped by v2_resolve).
    const int HWt = HW + 2 * par;
    const bool okgeo = t0 >= 0 && t0n > tm + 2 && K + HWt < 1900;
    // six counts, one per lane: buckets with t ≤ T are [⌈(c2−T)/2⌉, ⌊(c2+T)/2⌋]
    int p = 0;
    if (lane == 0) p = (c2 + (t0n - 1)) / 2 + 1;         // n_in  = A(p0) − A(p1), T = t0n − 1 ≥ 0
    if (lane == 1) p = (c2 - (t0n - 1) + 1) / 2;
    if (lane == 2) p = (c2 + tEn) / 2 + 1;               // upto  = A(p2) − A(p3)
    if (lane == 3) p = (c2 - tEn + 1) / 2;
    if (lane == 4) p = (c2 + tm) / 2 + 1;                // n_med = A(p4) − A(p5)
    if (lane == 5) p = (c2 - tm + 1) / 2;
    p = min(max(p, 0), kV2NB);                           // c2 − T may be negative: ⌈·/2⌉ of a negative is clamped anyway
    const unsigned A = v2_count_below(L, CE, p);
    const unsigned n_in = __shfl_sync(0xffffffffu, A, 0) - __shfl_sync(0xffffffffu, A, 1);
    const unsigned upto = __shfl_sync(0xffffffffu, A, 2) - __shfl_sync(0xffffffffu, A, 3);
    const unsigned excl_med = __shfl_sync(0xffffffffu, A, 5);
    const unsigned n_med = __shfl_sync(0xffffffffu, A, 4) - excl_med;
    const bool okcnt = n_med <= (unsigned)kV2ClsCap && upto - n_in <= (unsigned)kV2ClsCap &&
                       n_med + (upto - n_in) <= (unsigned)kV2ListCap;
    if (lane == 0) {
        if (!okgeo) ctl.fail = 1;
        else if (!okcnt) ctl.fail = 3;
        ctl.c2[c] = c2; ctl.t0[c] = t0n; ctl.tE[c] = tEn; ctl.tm[c] = tm;
        constexpr float kUnit = 5.9604644775390625e-08f;                 // 2⁻²⁴ = one bucket in fp16 bits
        const __half2 h0 = __float2half2_rn(-4.0f * (float)(c2 >> 1) * kUnit), h1 = __float2half2_rn((float)K * kUnit),
                      h2 = __float2half2_rn((float)HWt * kUnit);
        ctl.hc2[c] = *reinterpret_cast<const unsigned*>(&h0);
        ctl.hK[c] = *reinterpret_cast<const unsigned*>(&h1);
        ctl.hHW[c] = *reinterpret_cast<const unsigned*>(&h2);
        ctl.n_in[c] = n_in; ctl.excl_med[c] = excl_med; ctl.n_med[c] = n_med; ctl.n_shl[c] = upto - n_in;
    }
}

__device__ __forceinline__ float v2_key_float(unsigned k) {
    return __uint_as_float(k ^ ((k >> 31) ? 0x80000000u : 0xFFFFFFFFu));
}

// Values of 0-based ranks t and t+1 among arr[0..n), one warp, n ≤ 64; arr is padded with +inf to a multiple of 4.
// The value of rank r is max{x : #{y < x} ≤ r}, so ties need no ordering.
__device__ __forceinline__ void v2_rank_pair(const float* __restrict__ arr, int n, int t, float& vt, float& vt1) {
    const int lane = threadIdx.x & 31;
    const float y0 = lane < n ? arr[lane] : INFINITY;
    int lt0 = 0;
    unsigned ka = 0, kb = 0;                                            // order-preserving keys; 0 = none
    if (n <= 32) {
        for (int j = 0; j < n; j += 4) {
            const float4 x = *reinterpret_cast<const float4*>(arr + j);
            lt0 += (x.x < y0) + (x.y < y0) + (x.z < y0) + (x.w < y0);
        }
    } else {
        const float y1 = lane + 32 < n ? arr[lane + 32] : INFINITY;
        int lt1 = 0;
        for (int j = 0; j < n; j += 4) {
            const float4 x = *reinterpret_cast<const float4*>(arr + j);
            lt0 += (x.x < y0) + (x.y < y0) + (x.z < y0) + (x.w < y0);
            lt1 += (x.x < y1) + (x.y < y1) + (x.z < y1) + (x.w < y1);
        }
        if (lane + 32 < n) {
            const unsigned k1 = float_key(y1);
            if (lt1 <= t) ka = k1;
            if (lt1 <= t + 1) kb = k1;
        }
    }
    if (lane < n) {
        const unsigned k0 = float_key(y0);
        if (lt0 <= t) ka = max(ka, k0);
        if (lt0 <= t + 1) kb = max(kb, k0);
    }
    vt = v2_key_float(__reduce_max_sync(0xffffffffu, ka));
    vt1 = v2_key_float(__reduce_max_sync(0xffffffffu, kb));
}

// One warp, one component: rank the gathered members of the median net and of the shells exactly, verify that the
// shells really hold the MAD, publish a, h, inv.
template <int B>
__device__ __forceinline__ void v2_resolve(V2Ctl& ctl, int c) {
    constexpr int kk = (B - 1) >> 1;
    constexpr bool kEven = (B & 1) == 0;
    const int lane = threadIdx.x & 31;
    float* med = ctl.cls[c][0];
    float* shl = ctl.cls[c][1];
    const int nm = (int)ctl.cls_n[c][0], ns = (int)ctl.cls_n[c][1];   // the gather has split the members already
    const float scale = ctl.scale[c], off = ctl.off[c];
    const int c2 = ctl.c2[c], t0 = ctl.t0[c], tE = ctl.tE[c];
    const int tmr = kk - (int)ctl.excl_med[c], tsr = kk - (int)ctl.n_in[c];
    if (nm != (int)ctl.n_med[c] || ns != (int)ctl.n_shl[c] ||      // the gather must deliver exactly what the histogram counted
        tmr < 0 || tsr < 0 || tmr + (kEven ? 1 : 0) >= nm || tsr + (kEven ? 1 : 0) >= ns) {
        if (lane == 0) ctl.fail = 3;
        return;
    }
    if (lane < 4) { med[nm + lane] = INFINITY; shl[ns + lane] = INFINITY; }
    __syncwarp();
    float a, b;
    v2_rank_pair(med, nm, tmr, a, b);
    if (!kEven) b = a;
    const float h = 0.5f * __fsub_rn(b, a);
    // deviations of the shell members, same arithmetic as the general path
    if (lane < ns) shl[lane] = fabsf(__fsub_rn(__fsub_rn(shl[lane], a), h));
    if (lane + 32 < ns) shl[lane + 32] = fabsf(__fsub_rn(__fsub_rn(shl[lane + 32], a), h));
    __syncwarp();
    float da, db;
    v2_rank_pair(shl, ns, tsr, da, db);
    if (!kEven) db = da;
    // ---- verification.  vb(k) = value at the boundary between buckets k−1 and k.  Every value whose bucket lies
    // strictly inside the shells deviates by at most din, every value beyond them by at least dout; the margin of
    // 0.05 bucket covers the float rounding of the map and of its inverse (|off| ≤ 64).
    const double m = (double)a + (double)h;
    const double rs = (double)(1.0f / scale);
    const double eps = 0.05 * rs * (1.0 / 2047.0);
    auto vb = [&](int k) { return (((double)k - 0.5) * (1.0 / 2047.0) - (double)off) * rs; };
    const int jl_in = (c2 - t0) / 2 + 1;              // lowest bucket inside on the low side (t < t0 ⇔ 2j − c2 > −t0)
    const int jh_in = (c2 + t0 + 1) / 2 - 1;          // highest bucket inside on the high side
    const int jl_out = (c2 - tE + 1) / 2 - 1;         // highest bucket beyond the shells on the low side (may be < 0)
    const int jh_out = (c2 + tE) / 2 + 1;             // lowest bucket beyond the shells on the high side (may be ≥ NB)
    const bool bounded = c2 - t0 >= 0 && jl_in >= 1 && jh_in + 1 <= kV2NB - 1;   // else a clamped end bucket would be "inside"
    double din = 0.0, dout = INFINITY;
    if (bounded) din = fmax(m - vb(jl_in), vb(jh_in + 1) - m) + eps;
    if (c2 - tE + 1 >= 0 && jl_out >= 0) dout = fmin(dout, m - vb(jl_out + 1) - eps);
    if (jh_out <= kV2NB - 1) dout = fmin(dout, vb(jh_out) - m - eps);
    const bool verified = bounded && (double)da >= din && (double)db <= dout;
    const double s = kKappa * (0.5 * ((double)da + (double)db));
    if (lane == 0) {
        if (!verified) ctl.fail = 4;
        ctl.a[c] = a; ctl.h[c] = h;
        ctl.inv[c] = (s > 0.0 && isfinite(s)) ? (float)(0.70710678118654752440 / s) : 0.f;
    }
}

// Stage `bytes` (multiple of 16) global → shared with one TMA bulk copy; thread 0 only.  The mbarrier must have been
// initialised (and fenced) by the same thread.
__device__ __forceinline__ void v2_tma_issue(void* smem_dst, const void* gmem_src, uint32_t bytes, unsigned long long* mbar) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(v2_smem(mbar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     v2_smem(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(v2_smem(mbar))
                 : "memory");
}

__device__ __forceinline__ void v2_mbar_wait(unsigned long long* mbar, unsigned parity) {
    unsigned done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(v2_smem(mbar)), "r"(parity)
            : "memory");
    }
}

// Which instantiations use the L2 look-ahead (see the kernel): measured on a B200 it pays for short blocks only, where the
// first touch of a block is a larger share of its time (cfg 5, B = 2048: 8.25 -> 7.61 ms with a look-ahead of 592 CTAs;
// cfg 3, B = 4096: 3.18 -> 3.25 ms; cfg 4, B = 8192: 0.905 -> 0.96 ms), so it is compiled out of the others.
template <int EPT, int NT, bool STAGED>
constexpr bool kV2L2Ahead() { return !STAGED && EPT * NT <= 2048; }

// Dynamic shared memory of norm_power_v2_kernel<EPT, NT>: [stage: 8·B + 16 bytes][hist: 2·NB·4][V2Ctl].
template <int EPT, int NT, bool STAGED>
constexpr size_t v2_smem_bytes() {
    return (STAGED ? (size_t)EPT * NT * 8 + 16 : 0) + (size_t)2 * kV2NB * 4 + sizeof(V2Ctl);
}

// Grid: blocks_per_row · batch CTAs; CTA x handles block (x mod blocks_per_row) of spectrum x / blocks_per_row, bins
// [j·B, (j+1)·B).  `lim_lo`/`lim_hi` bound the input allocation: the TMA copy is 16-byte granular and is only used when
// its rounded range stays inside; otherwise the CTA stages the block with ordinary loads.
// STAGED = false: nothing is staged; the histogram pass, the (rare) gather hits and the output pass read the block from
// global memory (the second and third time out of L1/L2, where a block read microseconds earlier still is), which
// leaves 19 KB of shared memory per CTA so that more blocks are in flight per SM to cover the warp-serial phases.
// KEEPIDX = false: the bucket indices are not kept in registers between the histogram pass and the gather; the gather re-reads
// the block (L2, partly L1) and recomputes them.  More instructions and one more read pass, but the kernel fits 40 registers
// and the SM holds 11-12 blocks instead of 8: the kernel is bound by the latency of its phases, not by their issue slots.
#ifndef PULSCAN_NORM_OCC128_NOIDX
#define PULSCAN_NORM_OCC128_NOIDX 11
#endif
template <int EPT, int NT, bool STAGED, bool KEEPIDX>
constexpr int v2_min_ctas() {
    if (STAGED) return (EPT * NT <= 4096) ? 4 : 2;
    if (!KEEPIDX) return NT == 128 ? PULSCAN_NORM_OCC128_NOIDX : 6;
    return NT == 128 ? (EPT <= 16 ? PULSCAN_NORM_OCC128_SMALL : PULSCAN_NORM_OCC128) : (EPT * NT <= 4096) ? 6 : 4;
}
template <int EPT, int NT, bool STAGED, bool KEEPIDX = true>
__global__ void __launch_bounds__(NT, v2_min_ctas<EPT, NT, STAGED, KEEPIDX>())
norm_power_v2_kernel(const float2* __restrict__ spectra, long long pitch_in, int blocks_per_row, int nb, NormOut out,
                     unsigned* __restrict__ redo, unsigned* __restrict__ redo_count,
                     const char* __restrict__ lim_lo, const char* __restrict__ lim_hi, unsigned l2_ahead) {
    static_assert(EPT % 2 == 0 && EPT <= 32, "bucket indices are packed in pairs; hit mask has 16 + 16 bits");
    static_assert(NT % 32 == 0 && (EPT * NT) % 128 == 0, "sample stride");
    constexpr int B = EPT * NT;
    extern __shared__ __align__(128) unsigned char v2_raw[];
    unsigned char* stage = v2_raw;
    unsigned* hist = reinterpret_cast<unsigned*>(v2_raw + (STAGED ? (size_t)B * 8 + 16 : 0));
    V2Ctl& ctl = *reinterpret_cast<V2Ctl*>(hist + 2 * kV2NB);
    const int tid = threadIdx.x, warp = tid >> 5;
    // Bin of thread tid in round r: wb + 32·r.  Each warp owns a contiguous run of 32·EPT bins: four rounds of a warp are 128
    // consecutive bins = 32 consecutive group sums, which the output pass writes as one 128-byte line per store.
    const int wb = warp * (EPT * 32) + (tid & 31);
    const unsigned row = blockIdx.x / (unsigned)blocks_per_row;
    const unsigned jblk = blockIdx.x - row * (unsigned)blocks_per_row;
    const long long lo_bin = (long long)jblk * B;
    const float2* src = spectra + (long long)row * pitch_in + lo_bin;

    // ---- stage the block; zero the histograms meanwhile; warp 0 derives the bucket map from a sample
    const unsigned shift = (unsigned)(reinterpret_cast<uintptr_t>(src) & 15);          // 0 or 8
    const char* csrc = reinterpret_cast<const char*>(src) - shift;
    const unsigned nbytes = (unsigned)B * 8u + (shift ? 16u : 0u);
    const bool use_tma = STAGED && csrc >= lim_lo && csrc + nbytes <= lim_hi;
    const float2* sdat = STAGED ? reinterpret_cast<const float2*>(stage + shift) : src;
    // L2 look-ahead: ask for the block that the CTA `l2_ahead` launches behind this one will work on (about one wave of
    // resident CTAs later) to be brought into L2 now, with one bulk prefetch that occupies no register and no LSU slot.
    // That CTA's three passes then find their 8·B bytes in L2: the HBM stream is decoupled from the latency-bound phases.
    if (kV2L2Ahead<EPT, NT, STAGED>() && l2_ahead && tid == 0 && blockIdx.x + l2_ahead < gridDim.x) {
        const unsigned nxt = blockIdx.x + l2_ahead;
        const unsigned nrow = nxt / (unsigned)blocks_per_row;
        const char* a = reinterpret_cast<const char*>(spectra + (long long)nrow * pitch_in + (long long)(nxt - nrow * (unsigned)blocks_per_row) * B);
        const char* a16 = a - (reinterpret_cast<uintptr_t>(a) & 15);
        const unsigned nb16 = (unsigned)B * 8u + 16u;
        if (a16 >= lim_lo && a16 + nb16 <= lim_hi)
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(a16), "r"(nb16) : "memory");
    }
#if PULSCAN_V2_SAMPLE_AHEAD
    // Longer blocks: only the four runs of 32 bins that the later CTA's sample estimate reads (its first, latency-bound step)
    if (!STAGED && !kV2L2Ahead<EPT, NT, STAGED>() && l2_ahead && tid == 0 && blockIdx.x + l2_ahead < gridDim.x) {
        const unsigned nxt = blockIdx.x + l2_ahead;
        const unsigned nrow = nxt / (unsigned)blocks_per_row;
        const char* a = reinterpret_cast<const char*>(spectra + (long long)nrow * pitch_in + (long long)(nxt - nrow * (unsigned)blocks_per_row) * B);
        const char* a16 = a - (reinterpret_cast<uintptr_t>(a) & 15);
        if (a16 >= lim_lo && a16 + (unsigned)B * 8u + 16u <= lim_hi) {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(a16 + (size_t)k * (B / 4) * 8), "r"(272u) : "memory");
        }
    }
#endif
    if (tid == 0) {
        if (STAGED) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(v2_smem(&ctl.mbar)));
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        if (use_tma) v2_tma_issue(stage, csrc, nbytes, &ctl.mbar);
        ctl.fail = 0; ctl.cls_n[0][0] = 0; ctl.cls_n[0][1] = 0; ctl.cls_n[1][0] = 0; ctl.cls_n[1][1] = 0;
    }
    {
        uint4* hz = reinterpret_cast<uint4*>(hist);
#pragma unroll
        for (int i = tid; i < 2 * kV2NB / 4; i += NT) hz[i] = make_uint4(0, 0, 0, 0);
    }
    if (STAGED && !use_tma) {
        float2* sw = reinterpret_cast<float2*>(stage + shift);
#pragma unroll 4
        for (int r = 0; r < EPT; ++r) sw[wb + r * 32] = __ldg(src + wb + r * 32);
        __syncthreads();
    }
    if (warp == 0) {
        __syncwarp();                                  // lane 0 has initialised the barrier and ctl.fail
        if (use_tma) v2_mbar_wait(&ctl.mbar, 0);
        v2_estimate<B>(sdat, ctl);
    }
    __syncthreads();                                                                     // S1
    if (use_tma) v2_mbar_wait(&ctl.mbar, 0);           // already complete: makes the copied bytes visible to this thread
    bool bad = ctl.fail != 0;

    // ---- histogram pass: both components, bucket indices kept packed in pairs
    unsigned idxp[2][KEEPIDX ? EPT / 2 : 1];
    if (!bad) {
        const float sc0 = ctl.scale[0], sc1 = ctl.scale[1], of0 = ctl.off[0], of1 = ctl.off[1];
        const unsigned hb0 = v2_smem(hist), hb1 = v2_smem(hist + kV2NB);
#pragma unroll
        for (int q = 0; q < EPT / 2; ++q) {
            const float2 z0 = sdat[wb + (2 * q) * 32], z1 = sdat[wb + (2 * q + 1) * 32];
            const unsigned b00 = v2_bucket_bits(z0.x, sc0, of0), b01 = v2_bucket_bits(z1.x, sc0, of0);
            const unsigned b10 = v2_bucket_bits(z0.y, sc1, of1), b11 = v2_bucket_bits(z1.y, sc1, of1);
            v2_red_inc(hb0 + (b00 << 2)); v2_red_inc(hb0 + (b01 << 2));
            v2_red_inc(hb1 + (b10 << 2)); v2_red_inc(hb1 + (b11 << 2));
            if (KEEPIDX) {
                idxp[0][q] = __byte_perm(b00, b01, 0x5410);
                idxp[1][q] = __byte_perm(b10, b11, 0x5410);
            }
        }
    }
    __syncthreads();                                                                     // S2
    // ---- chunk totals (16 buckets each), rotated 16-byte reads so that a quarter-warp touches all bank groups
    if (!bad) {
        for (int id = tid; id < 2 * kV2NCH; id += NT) {
            const uint4* hp = reinterpret_cast<const uint4*>(hist) + id * 4;
            const int rot = (id >> 1) & 3;
            unsigned s = 0;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const uint4 x = hp[(q + rot) & 3];
                s += (x.x + x.y) + (x.z + x.w);
            }
            (&ctl.chunk_tot[0][0])[id] = s;
        }
    }
    __syncthreads();                                                                     // S3
    if (!bad && warp < 2) v2_locate<B>(ctl, hist + warp * kV2NB, warp);
    __syncthreads();                                                                     // S4
    bad = bad || ctl.fail != 0;
    // ---- gather: z = ||4·(idx − ⌊c2/2⌋)| − K| − K, member ⇔ |z| ≤ HW', on fp16 pairs (exact small-integer arithmetic).
    // The few hits (≈ 30 of 2·B values) are re-read, classified exactly (shell t = |2·bucket − c2|: median net t ≤ tm, MAD
    // shells t0 ≤ t ≤ tE; for odd c2 the test above is one shell too wide and the extra hits are dropped here) and appended
    // to their list, so that the ranking warps start from split lists.  The masks of both components are formed first and
    // their hits are read in pairs: a thread's re-reads (L2 hits at best) overlap instead of following one another.
    if (!bad) {
        const __half2 four = __float2half2_rn(4.0f);
        unsigned hm[2] = {0u, 0u};
        const unsigned u00 = ctl.hc2[0], u01 = ctl.hK[0], u02 = ctl.hHW[0], u10 = ctl.hc2[1], u11 = ctl.hK[1], u12 = ctl.hHW[1];
        const __half2 hc2[2] = {*reinterpret_cast<const __half2*>(&u00), *reinterpret_cast<const __half2*>(&u10)};
        const __half2 Kh[2] = {*reinterpret_cast<const __half2*>(&u01), *reinterpret_cast<const __half2*>(&u11)};
        const __half2 HWh[2] = {*reinterpret_cast<const __half2*>(&u02), *reinterpret_cast<const __half2*>(&u12)};
        const float sc0 = ctl.scale[0], sc1 = ctl.scale[1], of0 = ctl.off[0], of1 = ctl.off[1];
#pragma unroll
        for (int q = 0; q < EPT / 2; ++q) {
            unsigned ip[2];
            if (KEEPIDX) { ip[0] = idxp[0][q]; ip[1] = idxp[1][q]; }
            else {
                const float2 z0 = sdat[wb + (2 * q) * 32], z1 = sdat[wb + (2 * q + 1) * 32];
                ip[0] = __byte_perm(v2_bucket_bits(z0.x, sc0, of0), v2_bucket_bits(z1.x, sc0, of0), 0x5410);
                ip[1] = __byte_perm(v2_bucket_bits(z0.y, sc1, of1), v2_bucket_bits(z1.y, sc1, of1), 0x5410);
            }
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const __half2 ih = *reinterpret_cast<const __half2*>(&ip[c]);
                const __half2 d4 = __hfma2(ih, four, hc2[c]);
                const __half2 u = __hsub2(__habs2(d4), Kh[c]);
                const __half2 z = __hsub2(__habs2(u), Kh[c]);
                const unsigned mm = __hle2_mask(__habs2(z), HWh[c]);
                hm[c] |= mm & ((1u << q) | (1u << (16 + q)));
            }
        }
        auto put = [&](float val, int c) {
            const int tt = abs(2 * (int)(v2_bucket_bits(val, ctl.scale[c], ctl.off[c]) & 0xFFFFu) - ctl.c2[c]);
            const int k = tt <= ctl.tm[c] ? 0 : (tt >= ctl.t0[c] && tt <= ctl.tE[c]) ? 1 : -1;
            if (k >= 0) {
                const unsigned slot = atomicAdd(&ctl.cls_n[c][k], 1u);
                if (slot < (unsigned)kV2ClsCap) ctl.cls[c][k][slot] = val;
            }
        };
        // The warp's hits (≈ 15) are dealt to its lanes, one each, so that their re-reads make ONE round trip instead of one
        // per hit of the unluckiest lane: hit j belongs to the lane whose running count first exceeds j.
        const int lane = tid & 31;
        const int n0 = __popc(hm[0]), cnt = n0 + __popc(hm[1]);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        const int total = __shfl_sync(0xffffffffu, incl, 31);
        for (int j0 = 0; j0 < total; j0 += 32) {
            const int j = j0 + lane;
            int owner = 0;                                   // number of lanes whose running count is ≤ j (incl is non-decreasing)
#pragma unroll
            for (int step = 16; step > 0; step >>= 1) {
                const int v = __shfl_sync(0xffffffffu, incl, min(owner + step - 1, 31));
                if (v <= j) owner += step;
            }
            owner = min(owner, 31);
            const int oi = __shfl_sync(0xffffffffu, incl, owner), oc = __shfl_sync(0xffffffffu, cnt, owner);
            const int on0 = __shfl_sync(0xffffffffu, n0, owner);
            const unsigned om0 = __shfl_sync(0xffffffffu, hm[0], owner), om1 = __shfl_sync(0xffffffffu, hm[1], owner);
            if (j < total) {
                const int k = j - (oi - oc);                 // my hit is the k-th of that lane: component 0's first
                const int c = k < on0 ? 0 : 1;
                const int b = (int)__fns(c ? om1 : om0, 0, (c ? k - on0 : k) + 1);
                const float val = reinterpret_cast<const float*>(sdat + (wb - lane + owner) + (2 * (b & 15) + (b >> 4)) * 32)[c];
                put(val, c);
            }
        }
    }
    __syncthreads();                                                                     // S5
    if (!bad && warp < 2) v2_resolve<B>(ctl, warp);
    __syncthreads();                                                                     // S6
    bad = bad || ctl.fail != 0;
    if (!bad) {
        // x' = ((v − a) − h)·inv evaluated as fma(v − a, inv, −h·inv), as in the general path (norm_power.cuh)
        const float a0 = ctl.a[0], a1 = ctl.a[1], i0 = ctl.inv[0], i1 = ctl.inv[1];
        const float k0 = -ctl.h[0] * i0, k1 = -ctl.h[1] * i1;
        if (out.P) {
            float* dst = out.P + (long long)row * out.pitchP + lo_bin;
#pragma unroll
            for (int r = 0; r < EPT; ++r) dst[wb + r * 32] = norm_power_value(sdat[wb + r * 32], a0, i0, k0, a1, i1, k1);
        }
        if (out.G) {   // sums of aligned groups of four bins (lanes 4j..4j+3 hold a group), see norm_power.cuh
            float* g = out.G + (long long)row * out.pitchG + (lo_bin >> 2) + (wb >> 2);
            if constexpr (EPT % 4 == 0) {
#pragma unroll
                for (int r0 = 0; r0 < EPT; r0 += 4) {
                    const float e = quad_sums4(norm_power_value(sdat[wb + r0 * 32], a0, i0, k0, a1, i1, k1),
                                               norm_power_value(sdat[wb + (r0 + 1) * 32], a0, i0, k0, a1, i1, k1),
                                               norm_power_value(sdat[wb + (r0 + 2) * 32], a0, i0, k0, a1, i1, k1),
                                               norm_power_value(sdat[wb + (r0 + 3) * 32], a0, i0, k0, a1, i1, k1));
                    g[(r0 + (tid & 3)) * 8] = e;       // 32 consecutive group sums per warp and store: one 128-byte line
                }
            } else {
#pragma unroll
                for (int r = 0; r < EPT; ++r) {
                    const float e = quad_sum1(norm_power_value(sdat[wb + r * 32], a0, i0, k0, a1, i1, k1));
                    if ((tid & 3) == 0) g[r * 8] = e;
                }
            }
            if (tid == 0) {
                float* st = out.stats + ((long long)row * nb + jblk) * 8;
                st[0] = a0; st[1] = i0; st[2] = k0; st[3] = a1; st[4] = i1; st[5] = k1;
            }
        }
    } else if (tid == 0) {
        redo[atomicAdd(redo_count, 1u)] = blockIdx.x;   // the general path will do this block
        atomicAdd(redo_count + 2 + min(max(ctl.fail, 1), 5), 1u);   // counters[4..8]: why (see V2Ctl::fail)
    }
}

} // namespace pulscan
