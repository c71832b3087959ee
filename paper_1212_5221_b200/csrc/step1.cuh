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
GF_DEV double uniform01(uint32_t w) { return ((double)w + 0.5) * (1.0 / 4294967296.0); }

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

// ---- heatbath (always double; R14, R15) -------------------------------------------
#define GF_TWO_PI 6.283185307179586476925286766559
#define GF_HB_MAX_TRIALS 64

// Landau/Coulomb: P(g) ~ exp(Re tr[gK]/T) (Eq. (30)).  u = g g_hat^-1 has
// u0 ~ sqrt(1-u0^2) exp(alpha u0), alpha = |a|/T: Kennedy-Pendleton (alpha >= 2) or Creutz.
GF_DEV void rule_heatbath_landau(const double a[4], double T, uint64_t seed, uint32_t site, uint32_t sweep,
                                 int sub, double g[4]) {
    const double n2 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2] + a[3] * a[3];
    if (n2 == 0.0) {
        g[0] = 1.0; g[1] = g[2] = g[3] = 0.0;
        return;
    }
    // one reciprocal square root and one reciprocal instead of a square root and six divisions; pi-scaled
    // trigonometric functions (exact argument reduction).  The oracle writes the same quantities with sqrt, / and
    // cos(2 pi r): the values agree to an ulp or two, the accept decisions but for events of probability ~1e-16.
    const double inv_norm = rsqrt(n2);
    const double norm = n2 * inv_norm;
    const double alpha = norm * (1.0 / T);
    const double inv_alpha = T * inv_norm;
    const double h0 = a[0] * inv_norm, h1 = -a[1] * inv_norm, h2 = -a[2] * inv_norm, h3 = -a[3] * inv_norm;
    double u0 = 1.0;
    if (alpha >= 2.0) {
        for (uint32_t trial = 0; trial < GF_HB_MAX_TRIALS; ++trial) {
            const u32x4 r = rng_draw(seed, site, sweep, sub, 1, trial);
            const double r1 = uniform01(r.x), r2 = uniform01(r.y), r3 = uniform01(r.z), r4 = uniform01(r.w);
            const double cs = cospi(2.0 * r2);
            const double delta = -(log(r1) + cs * cs * log(r3)) * inv_alpha;
            u0 = 1.0 - delta;
            if (r4 * r4 <= 1.0 - 0.5 * delta) break;
        }
    } else {
        const double em = exp(-2.0 * alpha);
        for (uint32_t trial = 0; trial < GF_HB_MAX_TRIALS; ++trial) {
            const u32x4 r = rng_draw(seed, site, sweep, sub, 1, trial);
            const double r1 = uniform01(r.x), r2 = uniform01(r.y);
            const double x = em + (1.0 - em) * r1;
            u0 = 1.0 + log(x) * inv_alpha;
            if (r2 * r2 <= 1.0 - u0 * u0) break;
        }
    }
    u0 = fmin(1.0, fmax(-1.0, u0));
    const u32x4 rd = rng_draw(seed, site, sweep, sub, 2, 0);
    const double ct = 2.0 * uniform01(rd.x) - 1.0;
    double sphi, cphi;
    sincospi(2.0 * uniform01(rd.y), &sphi, &cphi);
    const double st = sqrt(fmax(0.0, 1.0 - ct * ct));
    const double rad = sqrt(fmax(0.0, 1.0 - u0 * u0));
    const double u1 = rad * st * cphi, u2 = rad * st * sphi, u3 = rad * ct;
    // g = u * g_hat as 2x2 matrices of Eq. (22): (pq)_0 = p0 q0 - p.q, (pq)_vec = p0 q + q0 p - p x q
    const double q0 = u0 * h0 - u1 * h1 - u2 * h2 - u3 * h3;
    const double q1 = u0 * h1 + h0 * u1 - (u2 * h3 - u3 * h2);
    const double q2 = u0 * h2 + h0 * u2 - (u3 * h1 - u1 * h3);
    const double q3 = u0 * h3 + h0 * u3 - (u1 * h2 - u2 * h1);
    const double rn = rsqrt(q0 * q0 + q1 * q1 + q2 * q2 + q3 * q3);
    g[0] = q0 * rn; g[1] = q1 * rn; g[2] = q2 * rn; g[3] = q3 * rn;
}

// MAG: f = const + phi.X with phi on S^2, X = (E,F,D); sample phi ~ exp(phi.X/T), closed-form CDF.
GF_DEV void rule_heatbath_mag(double D, double E, double F, double T, uint64_t seed, uint32_t site,
                              uint32_t sweep, int sub, double g[4]) {
    const double lam = sqrt(D * D + E * E + F * F);
    if (lam == 0.0) {
        g[0] = 1.0; g[1] = g[2] = g[3] = 0.0;
        return;
    }
    const u32x4 r = rng_draw(seed, site, sweep, sub, 1, 0);
    const double r1 = uniform01(r.x), r2 = uniform01(r.y);
    const double inv_lam = 1.0 / lam;
    double cg = 1.0 + (T * inv_lam) * log(1.0 - r1 * (1.0 - exp(-2.0 * lam / T)));
    cg = fmin(1.0, fmax(-1.0, cg));
    const double sg = sqrt(fmax(0.0, 1.0 - cg * cg));
    const double X0 = E * inv_lam, X1 = F * inv_lam, X2 = D * inv_lam;
    double e10 = -X1, e11 = X0, e12 = 0.0;
    const double n1 = sqrt(e10 * e10 + e11 * e11);
    if (n1 < 1e-150) {
        e10 = 0.0; e11 = 1.0;
    } else {
        e10 /= n1; e11 /= n1;
    }
    const double e20 = X1 * e12 - X2 * e11, e21 = X2 * e10 - X0 * e12, e22 = X0 * e11 - X1 * e10;
    double sa, ca;
    sincospi(2.0 * r2, &sa, &ca);
    const double p0 = cg * X0 + sg * (ca * e10 + sa * e20);
    const double p1 = cg * X1 + sg * (ca * e11 + sa * e21);
    const double p2 = cg * X2 + sg * (ca * e12 + sa * e22);
    const double h = 0.5 * (1.0 + p2);
    if (h < 1e-300) {
        g[0] = 0.0; g[1] = 1.0; g[2] = 0.0; g[3] = 0.0;
        return;
    }
    const double g0 = sqrt(h);
    const double hg = 0.5 / g0;
    const double g1 = p0 * hg, g2 = p1 * hg;
    const double rn = rsqrt(g0 * g0 + g1 * g1 + g2 * g2);
    g[0] = g0 * rn; g[1] = g1 * rn; g[2] = g2 * rn; g[3] = 0.0;
}

}  // namespace gf
