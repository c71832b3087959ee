// step1.cuh — Step 1 of Alg. 1: the SU(2) update rules, and the counter-based
// Philox4x32-10 generator (PAPER.md:249 fn. 2) that the stochastic rules draw from.
//
// Input of every rule is the neighbourhood quaternion a = (a0,a1,a2,a3) of one SU(2) subgroup in
// the Cayley-Klein convention of Eq. (22): the local functional is
// g0 a0 - g1 a1 - g2 a2 - g3 a3 + const, maximal at conj(a)/|a| (Eq. (20)).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "su3.cuh"

namespace gf {

enum { ALGO_OR = 0, ALGO_SR = 1, ALGO_SA = 2, ALGO_MICRO = 3 };

// ---- Philox4x32-10 -------------------------------------------------------------------------
struct u32x4 {
    uint32_t x, y, z, w;
};

GF_DEV u32x4 philox4x32_10(u32x4 c, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        u32x4 n;
        n.x = hi1 ^ c.y ^ k0;
        n.y = lo1;
        n.z = hi0 ^ c.w ^ k1;
        n.w = lo0;
        c = n;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return c;
}

// counter = (site, sweep, subgroup | purpose << 8, trial), key = seed  (R19)
GF_DEV u32x4 rng_draw(uint64_t seed, uint32_t site, uint32_t sweep, int sub, int purpose, uint32_t trial) {
    u32x4 c;
    c.x = site;
    c.y = sweep;
    c.z = (uint32_t)sub | ((uint32_t)purpose << 8);
    c.w = trial;
    return philox4x32_10(c, (uint32_t)(seed & 0xffffffffull), (uint32_t)(seed >> 32));
}
// (w + 0.5) 2^-32, exactly: 2^52 + w assembled from its bit pattern, then one fused multiply-add
// (2^52 + w) 2^-32 - (2^20 - 2^-33); no integer-to-double conversion
GF_DEV double uniform01(uint32_t w) {
    return __fma_rn(__hiloint2double(0x43300000, (int)w), 0x1p-32, -(1048576.0 - 0x1p-33));
}

// ---- deterministic rules -------------------------------------------------------------------
GF_DEV float inv_sqrt(float x) { return 1.0f / sqrtf(x); }
GF_DEV double inv_sqrt(double x) { return rsqrt(x); }   // one MUFU.RSQ64H + Newton steps instead of sqrt and a division
GF_DEV float sqrt_t(float x) { return sqrtf(x); }
GF_DEV double sqrt_t(double x) { return sqrt(x); }

// Overrelaxation, Fig. A.11; omega = 1 is plain relaxation, Eq. (20).
template <class A>
GF_DEV void rule_or(const A a[4], A omega, A g[4]) {
    const A ai_sq = a[1] * a[1] + a[2] * a[2] + a[3] * a[3];
    const A a0_sq = a[0] * a[0];
    const A n = a0_sq + ai_sq;
    if (n == A(0)) {
        g[0] = A(1); g[1] = g[2] = g[3] = A(0);
        return;
    }
    A c, bc;
    if (sizeof(A) == 8) {
        // b = M/N with M = omega B + A', N = B + A'; c = 1/sqrt(B + b^2 A') = N r, bc = M r,
        // r = 1/sqrt(B N^2 + M^2 A'): the same numbers without the division (double: no under/overflow
        // for any sum of 2d unit-modulus links that is not exactly zero)
        const A m = omega * a0_sq + ai_sq;
        const A r = inv_sqrt(a0_sq * n * n + m * m * ai_sq);
        c = n * r;
        bc = m * r;
    } else {
        const A b = (omega * a0_sq + ai_sq) / n;
        c = inv_sqrt(a0_sq + b * b * ai_sq);
        bc = b * c;
    }
    g[0] = a[0] * c;
    g[1] = -a[1] * bc;
    g[2] = -a[2] * bc;
    g[3] = -a[3] * bc;
}

// Microcanonical step: exact square of the maximiser (R4).
template <class A>
GF_DEV void rule_micro(const A a[4], A g[4]) {
    const A n2 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2] + a[3] * a[3];
    if (n2 == A(0)) {
        g[0] = A(1); g[1] = g[2] = g[3] = A(0);
        return;
    }
    const A inv = inv_sqrt(n2);
    const A h0 = a[0] * inv, h1 = -a[1] * inv, h2 = -a[2] * inv, h3 = -a[3] * inv;
    g[0] = A(2) * h0 * h0 - A(1);
    g[1] = A(2) * h0 * h1;
    g[2] = A(2) * h0 * h2;
    g[3] = A(2) * h0 * h3;
}

// ---- heatbath (R14, R15, §6.8) ------------------------------------------------------
// Split in two phases.  hb_draws_* makes the Philox draws of trial 0 and of the direction and everything that follows
// from them alone (logarithms, trigonometric functions): none of it depends on the links, so the half-sweep kernel
// runs it while its cp.async gather is in flight.  hb_finish_* needs the local field and is short.  The retries of
// the rejection loops are evaluated by the 32 lanes of the warp together (hb_retry).  The values are those of the
// serial loop of the oracle (the draws are keyed by (site, sweep, subgroup, trial), R19).
//
// S = scalar type of the heatbath arithmetic: double on DP and MP contexts (Step 1 in double), float on
// SP contexts.  In float every accept/reject decision is taken with a guard band: where the float value of the
// decision variable is within a proven bound of its rounding error from the threshold, the trial is re-evaluated in
// double, so the decisions are the double-precision ones (for the float local field) and only the accepted value
// carries float rounding (~1e-7, inside the 5e-5 of BASELINE.json).
#define GF_HB_MAX_TRIALS 64
#define GF_FULL_WARP 0xffffffffu

template <class S>
struct HbDraw {
    // Landau/Coulomb: v[0] = L = ln r1 + cos^2(2 pi r2) ln r3, v[1] = r4^2, v[5] = |ln r1| + |ln r3| of Kennedy-Pendleton
    //                 trial 0 and v[6], v[7], v[8] the same of trial 1 (most lanes that reject trial 0 accept trial 1: the
    //                 warp-wide retry becomes rare); v[2..4] = uniform direction (sin th cos ph, sin th sin ph, cos th)
    // MAG:            v[0] = r1, v[1] = sin(2 pi r2), v[2] = cos(2 pi r2), v[3] = 1 - r1
    S v[9];
};

// (w + 0.5) 2^-32 in S; the float version rounds w to 24 bits (relative error 2^-24)
template <class S> GF_DEV S uniform_s(uint32_t w);
template <> GF_DEV double uniform_s<double>(uint32_t w) { return uniform01(w); }
template <> GF_DEV float uniform_s<float>(uint32_t w) { return __fmaf_rn((float)w, 0x1p-32f, 0x1p-33f); }

GF_DEV float log_s(float x) { return logf(x); }
GF_DEV double log_s(double x) { return log(x); }
// ln of a uniform in (0, 1].  float: the SFU's lg2 (2 ulp outside [1/2, 2], 2^-22 absolute inside: CUDA C Programming
// Guide, __log2f) times ln 2 - as good as logf for this purpose at a tenth of the instructions
GF_DEV float log_u(float x) { return __log2f(x) * 0.693147180559945309f; }
GF_DEV double log_u(double x) { return log(x); }
// cos^2(2 pi r) = 1/2 - 1/2 cos(2 pi c), c = frac(2 r) - 1/2 in [-1/2, 1/2); float: SFU cosine on [-pi, pi)
// (absolute error 2^-21.41 there, __cosf)
GF_DEV float cos2_2pi(float r) {
    float y = r + r;
    y = (y >= 1.0f) ? y - 1.0f : y;
    return __fmaf_rn(-0.5f, __cosf(6.283185307179586f * (y - 0.5f)), 0.5f);
}
GF_DEV double cos2_2pi(double r) { const double c = cospi(2.0 * r); return c * c; }
// (sin, cos)(2 pi r): pi-scaled functions (exact argument reduction)
GF_DEV void sincos_2pi(float r, float* s, float* c) { sincospif(2.0f * r, s, c); }
GF_DEV void sincos_2pi(double r, double* s, double* c) { sincospi(2.0 * r, s, c); }
GF_DEV float exp_s(float x) { return expf(x); }
GF_DEV double exp_s(double x) { return exp(x); }
GF_DEV float cospi_s(float x) { return cospif(x); }
GF_DEV double cospi_s(double x) { return cospi(x); }
GF_DEV void sincospi_s(float x, float* s, float* c) { sincospif(x, s, c); }
GF_DEV void sincospi_s(double x, double* s, double* c) { sincospi(x, s, c); }
GF_DEV float rsqrt_s(float x) { return rsqrtf(x); }
GF_DEV double rsqrt_s(double x) { return rsqrt(x); }
GF_DEV float max_s(float a, float b) { return fmaxf(a, b); }
GF_DEV double max_s(double a, double b) { return fmax(a, b); }
GF_DEV float min_s(float a, float b) { return fminf(a, b); }
GF_DEV double min_s(double a, double b) { return fmin(a, b); }
// sqrt(x) for x >= 0 as x rsqrt(x) (0 at 0)
template <class S>
GF_DEV S sqrt_pos(S x) { return x > S(0) ? x * rsqrt_s(x) : S(0); }

template <class S>
GF_DEV void hb_draws_landau(uint64_t seed, uint32_t site, uint32_t sweep, int sub, HbDraw<S>& d) {
    const u32x4 rd = rng_draw(seed, site, sweep, sub, 2, 0);
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const u32x4 r = rng_draw(seed, site, sweep, sub, 1, (uint32_t)t);
        const S r1 = uniform_s<S>(r.x), r2 = uniform_s<S>(r.y), r3 = uniform_s<S>(r.z), r4 = uniform_s<S>(r.w);
        const S l1 = log_u(r1), l3 = log_u(r3);
        d.v[t ? 6 : 0] = l1 + cos2_2pi(r2) * l3;
        d.v[t ? 7 : 1] = r4 * r4;
        if (sizeof(S) == 4) d.v[t ? 8 : 5] = -(l1 + l3);   // the guard band of the float decisions only
    }
    // cos th = 2 r5 - 1 = r5 - (1 - r5) and sin^2 th = 4 r5 (1 - r5), with 1 - r5 converted from the complemented
    // Philox word: no cancellation near the poles (in float 1 - cos^2 th would lose sin th there)
    const S r5 = uniform_s<S>(rd.x), r5c = uniform_s<S>(~rd.x);
    const S ct = r5 - r5c;
    S sphi, cphi;
    sincos_2pi(uniform_s<S>(rd.y), &sphi, &cphi);
    const S st = S(2) * sqrt_pos(r5 * r5c);
    d.v[2] = st * cphi;
    d.v[3] = st * sphi;
    d.v[4] = ct;
}
template <class S>
GF_DEV void hb_draws_mag(uint64_t seed, uint32_t site, uint32_t sweep, int sub, HbDraw<S>& d) {
    const u32x4 r = rng_draw(seed, site, sweep, sub, 1, 0);
    d.v[0] = uniform_s<S>(r.x);
    sincos_2pi(uniform_s<S>(r.y), &d.v[1], &d.v[2]);
    d.v[3] = uniform_s<S>(~r.x);   // 1 - r1 = ((2^32 - 1 - w) + 0.5) 2^-32, to full relative precision
}

// Guard bands of the float decisions (first-order bounds of the rounding error of the decision variable, with a
// factor >= 8 to spare).  Kennedy-Pendleton: v = 1 - delta/2 - r4^2, delta = -L/alpha; the logarithms are good to
// 3.6e-7 relative or 1.7e-7 absolute, cos^2 to 6e-7 (SFU 1.8e-7, argument 4 pi 2^-25), the uniforms to 2^-24
// relative: |error of L| <= 1e-6 (|ln r1| + |ln r3|) + 4e-7, so |error of v| <= 0.5e-6 (|ln r1| + |ln r3|)/alpha
// + 6e-7.  Creutz: v = w (2 - w) - r2^2 with w in [0, 2] good to 5e-7 relative: |error of v| <= 2.5e-6.
#define GF_HB_BAND_KP 1e-5f
#define GF_HB_BAND_CREUTZ 3e-5f

// one trial of the u0 sampler, u0 ~ sqrt(1-u0^2) exp(alpha u0): Kennedy-Pendleton (kp, alpha >= 2) or Creutz.
// Returns accepted?; w = 1 - u0.  aux = exp(-2 alpha) (Creutz only).
GF_DEV bool hb_trial(bool kp, double inv_alpha, double aux, const u32x4& r, double& w) {
    const double r1 = uniform01(r.x), r2 = uniform01(r.y);
    if (kp) {
        const double r3 = uniform01(r.z), r4 = uniform01(r.w);
        const double cs = cospi(2.0 * r2);
        w = -(log(r1) + cs * cs * log(r3)) * inv_alpha;
        return r4 * r4 <= 1.0 - 0.5 * w;
    }
    const double x = aux + (1.0 - aux) * r1;
    w = -log(x) * inv_alpha;
    return r2 * r2 <= w * (2.0 - w);
}
// the same in float, aux = 1 - exp(-2 alpha) (from expm1f); inside the guard band the trial is redone in double
GF_DEV bool hb_trial(bool kp, float inv_alpha, float aux, const u32x4& r, float& w) {
    const float r2 = uniform_s<float>(r.y);
    float v, band;
    if (kp) {
        const float r1 = uniform_s<float>(r.x), r3 = uniform_s<float>(r.z), r4 = uniform_s<float>(r.w);
        const float l1 = log_u(r1), l3 = log_u(r3);
        w = -(l1 + cos2_2pi(r2) * l3) * inv_alpha;
        v = 1.0f - 0.5f * w - r4 * r4;
        band = GF_HB_BAND_KP * (1.0f - (l1 + l3) * inv_alpha);
    } else {
        const float r1c = uniform_s<float>(~r.x);   // 1 - r1
        w = -log1pf(-aux * r1c) * inv_alpha;         // x = 1 - (1 - e^{-2 alpha}) (1 - r1)
        v = w * (2.0f - w) - r2 * r2;
        band = GF_HB_BAND_CREUTZ;
    }
    if (fabsf(v) > band) return v > 0.0f;
    double wd;
    const bool ok = hb_trial(kp, (double)inv_alpha, kp ? 0.0 : exp(-2.0 / (double)inv_alpha), r, wd);
    w = (float)wd;
    return ok;
}

// position of the k-th (0-based) set bit of m, k < popc(m)
GF_DEV int kth_set_bit(uint32_t m, int k) {
    int pos = 0, c;
    c = __popc(m & 0xffffu); if (k >= c) { pos += 16; k -= c; m >>= 16; }
    c = __popc(m & 0xffu);   if (k >= c) { pos += 8;  k -= c; m >>= 8; }
    c = __popc(m & 0xfu);    if (k >= c) { pos += 4;  k -= c; m >>= 4; }
    c = __popc(m & 0x3u);    if (k >= c) { pos += 2;  k -= c; m >>= 2; }
    c = (int)(m & 1u);       if (k >= c) pos += 1;
    return pos;
}

// The rejection loops, continued by the warp as a whole.  All 32 lanes call it together; a lane with pending = true
// still needs trials next_trial, next_trial + 1, ... (< GF_HB_MAX_TRIALS) of its own (site, subgroup) stream.  Few
// lanes are pending (the acceptance is 0.7 .. 0.996), so instead of every lane repeating the trial until the last
// one accepts (24 of 32 lanes active and 2.7 passes per subgroup in round 1), the 32 lanes evaluate 32 trials at
// once: the n pending lanes get g = 2^floor(log2(32 / n)) consecutive trials each, lane l evaluating trial
// next_trial + (l mod g) of the (l / g)-th pending lane, and the first accepted one in trial order stands.  After
// GF_HB_MAX_TRIALS rejected trials the last one stands, as in the serial loop.  Returns the lane's w = 1 - u0
// (unchanged for a lane that was not pending).  One copy in the binary: the kernels' instruction footprint matters.
template <class S>
static __device__ __noinline__ S hb_retry(bool pending, uint32_t next_trial, bool kp, S inv_alpha, S aux,
                                          uint64_t seed, uint32_t site, uint32_t sweep, int sub, S w) {
    const int lane = (int)(threadIdx.x & 31u);
    uint32_t rej = __ballot_sync(GF_FULL_WARP, pending);
    while (rej) {
        const int n = __popc(rej);
        const int lg = (n <= 1) ? 5 : 5 - (32 - __clz(n - 1));   // g = largest power of two <= 32 / n
        const int g = 1 << lg;
        const int q = lane >> lg, j = lane & (g - 1);
        const bool helper = q < n;
        const int src = helper ? kth_set_bit(rej, q) : 0;
        const uint32_t s_site = __shfl_sync(GF_FULL_WARP, site, src);
        const uint32_t s_next = __shfl_sync(GF_FULL_WARP, next_trial, src);
        const int s_kp = __shfl_sync(GF_FULL_WARP, (int)kp, src);
        const S s_ia = __shfl_sync(GF_FULL_WARP, inv_alpha, src);
        const S s_aux = __shfl_sync(GF_FULL_WARP, aux, src);
        const uint32_t trial = s_next + (uint32_t)j;
        bool ok = false;
        S v = S(0);
        if (helper && trial < GF_HB_MAX_TRIALS)
            ok = hb_trial(s_kp != 0, s_ia, s_aux, rng_draw(seed, s_site, sweep, sub, 1, trial), v);
        const uint32_t okm = __ballot_sync(GF_FULL_WARP, ok);
        int take = -1;
        if (pending) {
            const int first = __popc(rej & ((1u << lane) - 1u)) << lg;   // first lane of this lane's group
            const uint32_t mine = (okm >> first) & (lg == 5 ? 0xffffffffu : ((1u << g) - 1u));
            if (mine) take = first + __ffs((int)mine) - 1;
            else if (next_trial + (uint32_t)g >= GF_HB_MAX_TRIALS) take = first + (int)(GF_HB_MAX_TRIALS - 1 - next_trial);
            else next_trial += (uint32_t)g;
        }
        const S got = __shfl_sync(GF_FULL_WARP, v, take < 0 ? lane : take);
        if (take >= 0) { w = got; pending = false; }
        rej = __ballot_sync(GF_FULL_WARP, pending);
    }
    return w;
}

// Landau/Coulomb: P(g) ~ exp(Re tr[gK]/T) (Eq. (30)).  u = g g_hat^-1 has
// u0 ~ sqrt(1-u0^2) exp(alpha u0), alpha = |a|/T: Kennedy-Pendleton (alpha >= 2) or Creutz.
// Every lane of the warp must call it (hb_retry).
template <class S>
GF_DEV void hb_finish_landau(const S a[4], S T, const HbDraw<S>& d, uint64_t seed, uint32_t site,
                             uint32_t sweep, int sub, S g[4]) {
    const S n2 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2] + a[3] * a[3];
    const bool zero = n2 == S(0);
    // one reciprocal square root and one reciprocal instead of a square root and six divisions.  The oracle writes
    // the same quantities with sqrt and /: the values agree to an ulp or two, the accept decisions but for events
    // of probability ~1e-16 (double).
    const S inv_norm = rsqrt_s(zero ? S(1) : n2);
    const S norm = n2 * inv_norm;
    const S alpha = norm * (S(1) / T);
    const S inv_alpha = T * inv_norm;
    const S h0 = a[0] * inv_norm, h1 = -a[1] * inv_norm, h2 = -a[2] * inv_norm, h3 = -a[3] * inv_norm;
    const bool kp = alpha >= S(2);
    // trials 0 and 1 of Kennedy-Pendleton from the precomputed draws (w = delta = 1 - u0, accepted iff
    // v = 1 - delta/2 - r4^2 >= 0); in float a trial inside the guard band is left open and redone by hb_retry
    const S w0 = -d.v[0] * inv_alpha, w1 = -d.v[6] * inv_alpha;
    const S v0 = S(1) - S(0.5) * w0 - d.v[1], v1 = S(1) - S(0.5) * w1 - d.v[7];
    bool acc0, rej0, acc1, rej1;
    if (sizeof(S) == 4) {
        const S b0 = (S)GF_HB_BAND_KP * (S(1) + d.v[5] * inv_alpha), b1 = (S)GF_HB_BAND_KP * (S(1) + d.v[8] * inv_alpha);
        acc0 = v0 > b0; rej0 = v0 < -b0; acc1 = v1 > b1; rej1 = v1 < -b1;
    } else {
        acc0 = v0 >= S(0); rej0 = !acc0; acc1 = v1 >= S(0); rej1 = !acc1;
    }
    S w = acc0 ? w0 : w1;
    const bool pending = !zero && !(kp && (acc0 || (rej0 && acc1)));
    if (__any_sync(GF_FULL_WARP, pending)) {
        // first trial that is still open: 0 for a Creutz lane
        const uint32_t next = (!kp || !rej0) ? 0u : (!rej1 ? 1u : 2u);
        S aux = S(0);
        if (!kp) aux = (sizeof(S) == 4) ? (S)(-expm1f(-2.0f * (float)alpha)) : exp_s(S(-2) * alpha);
        w = hb_retry<S>(pending, next, kp, inv_alpha, aux, seed, site, sweep, sub, w);
    }
    w = min_s(S(2), max_s(S(0), w));   // u0 in [-1, 1]
    const S u0 = S(1) - w;
    const S rad = sqrt_pos(w * (S(2) - w));   // sqrt(1 - u0^2) without the cancellation
    const S u1 = rad * d.v[2], u2 = rad * d.v[3], u3 = rad * d.v[4];
    // g = u * g_hat as 2x2 matrices of Eq. (22): (pq)_0 = p0 q0 - p.q, (pq)_vec = p0 q + q0 p - p x q
    const S q0 = u0 * h0 - u1 * h1 - u2 * h2 - u3 * h3;
    const S q1 = u0 * h1 + h0 * u1 - (u2 * h3 - u3 * h2);
    const S q2 = u0 * h2 + h0 * u2 - (u3 * h1 - u1 * h3);
    const S q3 = u0 * h3 + h0 * u3 - (u1 * h2 - u2 * h1);
    const S rn = rsqrt_s(q0 * q0 + q1 * q1 + q2 * q2 + q3 * q3);
    g[0] = zero ? S(1) : q0 * rn;
    g[1] = zero ? S(0) : q1 * rn;
    g[2] = zero ? S(0) : q2 * rn;
    g[3] = zero ? S(0) : q3 * rn;
}

// whole heatbath in one call, in double (SU(2) input generator, Wilson heatbath); every lane of the warp must call it
GF_DEV void rule_heatbath_landau(const double a[4], double T, uint64_t seed, uint32_t site, uint32_t sweep,
                                 int sub, double g[4]) {
    HbDraw<double> d;
    hb_draws_landau<double>(seed, site, sweep, sub, d);
    hb_finish_landau<double>(a, T, d, seed, site, sweep, sub, g);
}

// MAG: f = const + phi.X with phi on S^2, X = (E,F,D); sample phi ~ exp(phi.X/T), closed-form CDF:
// cos(gamma) = 1 + (T/lambda) ln(1 - r1 (1 - e^{-2 lambda/T})).
GF_DEV double hb_mag_one_minus_cg(double r1, double /*r1c*/, double lam, double inv_lam, double T) {
    return -(T * inv_lam) * log(1.0 - r1 * (1.0 - exp(-2.0 * lam * (1.0 / T))));
}
// float: the argument of the logarithm without cancellation — 1 - r1 q (q = 1 - e^{-y} from expm1f) through log1pf
// where r1 q < 1/2, else as (1 - r1) + r1 e^{-y} with 1 - r1 converted from the complemented Philox word
GF_DEV float hb_mag_one_minus_cg(float r1, float r1c, float lam, float inv_lam, float T) {
    const float y = 2.0f * lam / T;
    const float t = -r1 * expm1f(-y);
    const float lg = (t < 0.5f) ? log1pf(-t) : logf(__fmaf_rn(r1, expf(-y), r1c));
    return -(T * inv_lam) * lg;
}

template <class S>
GF_DEV void hb_finish_mag(S D, S E, S F, S T, const HbDraw<S>& d, S g[4]) {
    const S n2 = D * D + E * E + F * F;
    const bool zero = n2 == S(0);
    const S inv_lam = rsqrt_s(zero ? S(1) : n2);
    const S lam = n2 * inv_lam;
    const S w = min_s(S(2), max_s(S(0), hb_mag_one_minus_cg(d.v[0], d.v[3], lam, inv_lam, T)));   // 1 - cos(gamma)
    const S cg = S(1) - w;
    const S sg = sqrt_pos(w * (S(2) - w));
    const S X0 = E * inv_lam, X1 = F * inv_lam, X2 = D * inv_lam;
    // frame about X: e1 = normalise(z x X) (y if degenerate), e2 = X x e1
    const S n1sq = X0 * X0 + X1 * X1;
    const bool degenerate = n1sq < (sizeof(S) == 4 ? S(1e-36) : S(1e-300));
    const S rn1 = rsqrt_s(degenerate ? S(1) : n1sq);
    const S e10 = degenerate ? S(0) : -X1 * rn1, e11 = degenerate ? S(1) : X0 * rn1;
    const S e20 = -X2 * e11, e21 = X2 * e10, e22 = X0 * e11 - X1 * e10;
    const S sa = d.v[1], ca = d.v[2];
    const S p0 = cg * X0 + sg * (ca * e10 + sa * e20);
    const S p1 = cg * X1 + sg * (ca * e11 + sa * e21);
    const S p2 = cg * X2 + sg * (sa * e22);
    const S h = S(0.5) * (S(1) + p2);
    const bool south = h < (sizeof(S) == 4 ? S(1e-36) : S(1e-300));
    const S rh = rsqrt_s(south ? S(1) : h);
    const S g0 = h * rh, hg = S(0.5) * rh;
    const S g1 = p0 * hg, g2 = p1 * hg;
    const S rn = rsqrt_s(g0 * g0 + g1 * g1 + g2 * g2);
    g[0] = zero ? S(1) : (south ? S(0) : g0 * rn);
    g[1] = zero ? S(0) : (south ? S(1) : g1 * rn);
    g[2] = (zero || south) ? S(0) : g2 * rn;
    g[3] = S(0);
}

}  // namespace gf
