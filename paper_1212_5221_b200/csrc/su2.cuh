// su2.cuh — the gauge group SU(2): links as quaternions.
//
// An SU(2) matrix is U = u0 1 + i (u1 s1 + u2 s2 + u3 s3) (Cayley-Klein form, Eq. (15)/(23),
// PAPER.md:124, 181): four reals, and the second row of the matrix is (-conj b, conj a) of the first
// row (a, b) = (u0 + i u3, u2 + i u1) — the N_c = 2 analogue of the 12-real storage of PAPER.md:351.
// HBM holds the first row, (Re a, Im a, Re b, Im b) = (u0, u3, u2, u1): one float4 or two double2 per
// link, in the parity-split vector planes of layout.cuh with RECON = 4:
//     links[parity][mu][chunk][cb],   16 bytes per chunk.
#pragma once
#include <cuda_runtime.h>

#include "layout.cuh"
#include "su3.cuh"

namespace gf {

template <class T>
struct Quat {
    T v[4];   // (u0, u1, u2, u3)
};

// r = g u  (matrix product in Cayley-Klein components):
//   r0 = g0 u0 - g.u,   r_vec = g0 u_vec + u0 g_vec - g_vec x u_vec
template <class T>
GF_DEV Quat<T> qmul(const Quat<T>& g, const Quat<T>& u) {
    Quat<T> r;
    r.v[0] = fma_t(-g.v[3], u.v[3], fma_t(-g.v[2], u.v[2], fma_t(-g.v[1], u.v[1], g.v[0] * u.v[0])));
    r.v[1] = fma_t(g.v[3], u.v[2], fma_t(-g.v[2], u.v[3], fma_t(u.v[0], g.v[1], g.v[0] * u.v[1])));
    r.v[2] = fma_t(g.v[1], u.v[3], fma_t(-g.v[3], u.v[1], fma_t(u.v[0], g.v[2], g.v[0] * u.v[2])));
    r.v[3] = fma_t(g.v[2], u.v[1], fma_t(-g.v[1], u.v[2], fma_t(u.v[0], g.v[3], g.v[0] * u.v[3])));
    return r;
}
// r = u g^dagger:  r0 = u0 g0 + u.g,   r_vec = g0 u_vec - u0 g_vec + u_vec x g_vec
template <class T>
GF_DEV Quat<T> qmul_dagger(const Quat<T>& u, const Quat<T>& g) {
    Quat<T> r;
    r.v[0] = fma_t(u.v[3], g.v[3], fma_t(u.v[2], g.v[2], fma_t(u.v[1], g.v[1], u.v[0] * g.v[0])));
    r.v[1] = fma_t(-u.v[3], g.v[2], fma_t(u.v[2], g.v[3], fma_t(-u.v[0], g.v[1], g.v[0] * u.v[1])));
    r.v[2] = fma_t(-u.v[1], g.v[3], fma_t(u.v[3], g.v[1], fma_t(-u.v[0], g.v[2], g.v[0] * u.v[2])));
    r.v[3] = fma_t(-u.v[2], g.v[1], fma_t(u.v[1], g.v[2], fma_t(-u.v[0], g.v[3], g.v[0] * u.v[3])));
    return r;
}
template <class T>
GF_DEV Quat<T> qconj(const Quat<T>& u) {
    Quat<T> r;
    r.v[0] = u.v[0]; r.v[1] = -u.v[1]; r.v[2] = -u.v[2]; r.v[3] = -u.v[3];
    return r;
}

// ---- HBM <-> registers: stored order (u0, u3, u2, u1) ------------------------------------------
GF_DEV void global_get_q(const char* plane0, int64_t Vh, int64_t cb, Quat<float>& q) {
    const float4 c = *reinterpret_cast<const float4*>(plane0 + cb * 16);
    q.v[0] = c.x; q.v[3] = c.y; q.v[2] = c.z; q.v[1] = c.w;
}
GF_DEV void global_get_q(const char* plane0, int64_t Vh, int64_t cb, Quat<double>& q) {
    const double2 c0 = *reinterpret_cast<const double2*>(plane0 + cb * 16);
    const double2 c1 = *reinterpret_cast<const double2*>(plane0 + 16 * Vh + cb * 16);
    q.v[0] = c0.x; q.v[3] = c0.y; q.v[2] = c1.x; q.v[1] = c1.y;
}
GF_DEV void global_put_q(char* plane0, int64_t Vh, int64_t cb, const Quat<float>& q) {
    *reinterpret_cast<float4*>(plane0 + cb * 16) = make_float4(q.v[0], q.v[3], q.v[2], q.v[1]);
}
GF_DEV void global_put_q(char* plane0, int64_t Vh, int64_t cb, const Quat<double>& q) {
    *reinterpret_cast<double2*>(plane0 + cb * 16) = make_double2(q.v[0], q.v[3]);
    *reinterpret_cast<double2*>(plane0 + 16 * Vh + cb * 16) = make_double2(q.v[2], q.v[1]);
}

// ---- neighbourhood summaries ---------------------------------------------------------------------
// Landau/Coulomb (Eq. (19)/(20)): a = quaternion of 2 K(x), the un-normalised form of
// Fig. A.10: a += 2 u for U_mu(x), a += 2 conj(w) for U_mu(x-mu)^dagger.
template <class A, class T>
GF_DEV void su2_acc_landau(A a[4], const Quat<T>& u, const Quat<T>& w) {
    a[0] += (A)2 * ((A)u.v[0] + (A)w.v[0]);
#pragma unroll
    for (int k = 1; k < 4; ++k) a[k] += (A)2 * ((A)u.v[k] - (A)w.v[k]);
}
// MAG (Eqs. (26)-(28), D per DESIGN.md R12): up link u, down link w entering as w^dagger
template <class A, class T>
GF_DEV void su2_acc_mag(A& D, A& E, A& F, const Quat<T>& uq, const Quat<T>& wq) {
    const A u0 = (A)uq.v[0], u1 = (A)uq.v[1], u2 = (A)uq.v[2], u3 = (A)uq.v[3];
    const A w0 = (A)wq.v[0], w1 = (A)wq.v[1], w2 = (A)wq.v[2], w3 = (A)wq.v[3];
    D += u0 * u0 + u3 * u3 - u1 * u1 - u2 * u2;
    D += w0 * w0 + w3 * w3 - w1 * w1 - w2 * w2;
    E += (A)2 * (-u0 * u1 - u2 * u3) + (A)2 * (w0 * w1 - w2 * w3);
    F += (A)2 * (-u0 * u2 + u1 * u3) + (A)2 * (w0 * w2 + w1 * w3);
}
// sum_i |U_ii|^2 = 2 (u0^2 + u3^2)   (Eq. (11))
template <class A, class T>
GF_DEV A su2_diag2(const Quat<T>& u) {
    return (A)2 * ((A)u.v[0] * (A)u.v[0] + (A)u.v[3] * (A)u.v[3]);
}

}  // namespace gf
