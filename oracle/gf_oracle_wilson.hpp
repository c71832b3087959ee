// =====================================================================================
// gf_oracle_wilson.hpp — CPU ORACLE for the input generator: thermalised
// SU(3) configurations of the Wilson gauge action, standing in for the paper's beta = 5.7 32^4
// ensemble, which is not available.  TEST INFRASTRUCTURE, NOT THE PRODUCT;
// included by gf_oracle.cpp after its own definitions (Philox, heatbath rule, Mat3, Lattice).
//
// The paper does not describe how its configurations were made (standard lattice practice); this is
// the textbook Cabibbo-Marinari pseudo-heatbath (ref. [31] of the paper is the SU(2)-subgroup method):
//   S = beta sum_P (1 - Re tr U_P / 3);  for a link U_mu(x) with staple sum
//   A = sum_{nu != mu} [ U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag + U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu) ]
//   the weight is exp((beta/3) Re tr[U A]).  For the subgroups (0,1),(0,2),(1,2) in turn: W = U A, a = the
//   un-normalised quaternion of W's sub-block (Fig. A.10), g drawn with P(g) ~ exp((beta/3)(g0 a0 - g.a)) —
//   the Landau heatbath rule of gf_oracle.cpp at temperature T = 3/beta — and U <- g~ U.
// Order of a sweep: for mu = 0..3, for parity = even, odd: all links U_mu(x) with x of that parity (they
// share no plaquette).  Random numbers: counter (site, 4*sweep_index + mu, sub | purpose << 8, trial).
// The paper gives nothing to compare this generator with: "parity unpinned" against the paper (R30), pinned
// by the mathematics below and oracle <-> GPU.
// Pins (tests/test_oracle_wilson.py): plaquette against an independent NumPy evaluation; strong-coupling
// <P> = beta/18 + beta^2/216; weak-coupling 1 - <P> -> 2/beta; beta -> infinity raises every local action
// term monotonically; unitarity; SU(2)-subgroup single-link law (u0 density) through the pinned rule.
// =====================================================================================
#pragma once

namespace {

template <class R>
inline Mat3<R> mat_mul(const Mat3<R>& a, const Mat3<R>& b) {
    Mat3<R> c;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            std::complex<R> acc(0, 0);
            for (int k = 0; k < 3; ++k) acc += a.m[i][k] * b.m[k][j];
            c.m[i][j] = acc;
        }
    return c;
}
template <class R>
inline Mat3<R> mat_dag(const Mat3<R>& a) {
    Mat3<R> c;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c.m[i][j] = std::conj(a.m[j][i]);
    return c;
}

inline int64_t site_shift2(const Lattice& L, const int c[4], int mu, int dmu, int nu, int dnu) {
    int d[4] = {c[0], c[1], c[2], c[3]};
    const int n[4] = {L.Nt, L.Nx, L.Ny, L.Nz};
    d[mu] = (d[mu] + dmu + n[mu]) % n[mu];
    d[nu] = (d[nu] + dnu + n[nu]) % n[nu];
    return L.site(d[0], d[1], d[2], d[3]);
}

// staple sum A of the link U_mu(x), x = c
template <class R>
inline Mat3<R> staple_sum(const R* links, const Lattice& L, const int c[4], int mu) {
    Mat3<R> A;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) A.m[i][j] = std::complex<R>(0, 0);
    const int64_t x = L.site(c[0], c[1], c[2], c[3]);
    const int64_t xmu = site_shift2(L, c, mu, +1, mu, 0);
    for (int nu = 0; nu < 4; ++nu) {
        if (nu == mu) continue;
        const int64_t xnu = site_shift2(L, c, nu, +1, nu, 0);
        const int64_t xmnu = site_shift2(L, c, nu, -1, nu, 0);
        const int64_t xmu_mnu = site_shift2(L, c, mu, +1, nu, -1);
        // upper: U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
        Mat3<R> up = mat_mul<R>(mat_mul<R>(load<R>(link_ptr(links, xmu, nu)), mat_dag<R>(load<R>(link_ptr(links, xnu, mu)))),
                                mat_dag<R>(load<R>(link_ptr(links, x, nu))));
        // lower: U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu)
        Mat3<R> lo = mat_mul<R>(mat_mul<R>(mat_dag<R>(load<R>(link_ptr(links, xmu_mnu, nu))),
                                           mat_dag<R>(load<R>(link_ptr(links, xmnu, mu)))),
                                load<R>(link_ptr(links, xmnu, nu)));
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) A.m[i][j] += up.m[i][j] + lo.m[i][j];
    }
    return A;
}

template <class R>
void wilson_heatbath_sweep(R* links, const Lattice& L, double beta, uint64_t seed, uint32_t sweep_index) {
    const double T = 3.0 / beta;
    for (int mu = 0; mu < 4; ++mu)
        for (int parity = 0; parity < 2; ++parity) {
#pragma omp parallel for collapse(2) schedule(static) if (L.V() >= OMP_MIN_SITES)
            for (int t = 0; t < L.Nt; ++t)
                for (int x = 0; x < L.Nx; ++x)
                    for (int y = 0; y < L.Ny; ++y)
                        for (int z = 0; z < L.Nz; ++z) {
                            if (((t + x + y + z) & 1) != parity) continue;
                            const int c[4] = {t, x, y, z};
                            const int64_t s = L.site(t, x, y, z);
                            Mat3<R> U = load<R>(link_ptr(links, s, mu));
                            const Mat3<R> A = staple_sum<R>(links, L, c, mu);
                            for (int sg = 0; sg < 3; ++sg) {
                                const int i = SUB_I[sg], j = SUB_J[sg];
                                const Mat3<R> W = mat_mul<R>(U, A);
                                double a[4] = {0, 0, 0, 0}, g[4];
                                add_quaternion<R, double>(a, W, i, j);
                                rule_heatbath_landau(a, T, seed, (uint32_t)s, 4u * sweep_index + (uint32_t)mu, sg, g);
                                R gr[4] = {(R)g[0], (R)g[1], (R)g[2], (R)g[3]};
                                left_mul_subgroup<R>(U, gr, i, j);
                            }
                            store<R>(link_ptr(links, s, mu), U);
                        }
        }
}

// average plaquette <Re tr U_P> / 3 over the 6 V plaquettes
template <class R>
double plaquette_mean(const R* links, const Lattice& L) {
    double tot = 0.0;
    for (int t = 0; t < L.Nt; ++t)
        for (int x = 0; x < L.Nx; ++x)
            for (int y = 0; y < L.Ny; ++y)
                for (int z = 0; z < L.Nz; ++z) {
                    const int c[4] = {t, x, y, z};
                    const int64_t s = L.site(t, x, y, z);
                    for (int mu = 0; mu < 4; ++mu)
                        for (int nu = mu + 1; nu < 4; ++nu) {
                            const int64_t xmu = site_shift2(L, c, mu, +1, mu, 0), xnu = site_shift2(L, c, nu, +1, nu, 0);
                            Mat3<R> P = mat_mul<R>(mat_mul<R>(load<R>(link_ptr(links, s, mu)), load<R>(link_ptr(links, xmu, nu))),
                                                   mat_mul<R>(mat_dag<R>(load<R>(link_ptr(links, xnu, mu))),
                                                              mat_dag<R>(load<R>(link_ptr(links, s, nu)))));
                            tot += (double)P.m[0][0].real() + (double)P.m[1][1].real() + (double)P.m[2][2].real();
                        }
                }
    return tot / (3.0 * 6.0 * (double)L.V());
}

// ---- the same for the gauge group SU(2): one "subgroup", weight exp((beta/2) Re tr[U A]), T = 2/beta ----
template <class R>
inline Mat2<R> staple_sum2(const R* links, const Lattice& L, const int c[4], int mu) {
    Mat2<R> A;
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) A.m[i][j] = std::complex<R>(0, 0);
    const int64_t x = L.site(c[0], c[1], c[2], c[3]);
    const int64_t xmu = site_shift2(L, c, mu, +1, mu, 0);
    for (int nu = 0; nu < 4; ++nu) {
        if (nu == mu) continue;
        const int64_t xnu = site_shift2(L, c, nu, +1, nu, 0), xmnu = site_shift2(L, c, nu, -1, nu, 0);
        const int64_t xmu_mnu = site_shift2(L, c, mu, +1, nu, -1);
        Mat2<R> up = mul2<R>(mul2<R>(load2<R>(link_ptr2(links, xmu, nu)), dagger2<R>(load2<R>(link_ptr2(links, xnu, mu)))),
                             dagger2<R>(load2<R>(link_ptr2(links, x, nu))));
        Mat2<R> lo = mul2<R>(mul2<R>(dagger2<R>(load2<R>(link_ptr2(links, xmu_mnu, nu))),
                                     dagger2<R>(load2<R>(link_ptr2(links, xmnu, mu)))),
                             load2<R>(link_ptr2(links, xmnu, nu)));
        for (int i = 0; i < 2; ++i)
            for (int j = 0; j < 2; ++j) A.m[i][j] += up.m[i][j] + lo.m[i][j];
    }
    return A;
}

template <class R>
void wilson_heatbath_sweep2(R* links, const Lattice& L, double beta, uint64_t seed, uint32_t sweep_index) {
    const double T = 2.0 / beta;
    for (int mu = 0; mu < 4; ++mu)
        for (int parity = 0; parity < 2; ++parity)
            for (int t = 0; t < L.Nt; ++t)
                for (int x = 0; x < L.Nx; ++x)
                    for (int y = 0; y < L.Ny; ++y)
                        for (int z = 0; z < L.Nz; ++z) {
                            if (((t + x + y + z) & 1) != parity) continue;
                            const int c[4] = {t, x, y, z};
                            const int64_t s = L.site(t, x, y, z);
                            Mat2<R> U = load2<R>(link_ptr2(links, s, mu));
                            const Mat2<R> W = mul2<R>(U, staple_sum2<R>(links, L, c, mu));
                            double a[4] = {0, 0, 0, 0}, g[4];
                            add_quaternion2<R, double>(a, W);
                            rule_heatbath_landau(a, T, seed, (uint32_t)s, 4u * sweep_index + (uint32_t)mu, 0, g);
                            R gr[4] = {(R)g[0], (R)g[1], (R)g[2], (R)g[3]};
                            store2<R>(link_ptr2(links, s, mu), mul2<R>(su2_matrix<R>(gr), U));
                        }
}

template <class R>
double plaquette_mean2(const R* links, const Lattice& L) {
    double tot = 0.0;
    for (int t = 0; t < L.Nt; ++t)
        for (int x = 0; x < L.Nx; ++x)
            for (int y = 0; y < L.Ny; ++y)
                for (int z = 0; z < L.Nz; ++z) {
                    const int c[4] = {t, x, y, z};
                    const int64_t s = L.site(t, x, y, z);
                    for (int mu = 0; mu < 4; ++mu)
                        for (int nu = mu + 1; nu < 4; ++nu) {
                            const int64_t xmu = site_shift2(L, c, mu, +1, mu, 0), xnu = site_shift2(L, c, nu, +1, nu, 0);
                            Mat2<R> P = mul2<R>(mul2<R>(load2<R>(link_ptr2(links, s, mu)), load2<R>(link_ptr2(links, xmu, nu))),
                                                mul2<R>(dagger2<R>(load2<R>(link_ptr2(links, xnu, mu))),
                                                        dagger2<R>(load2<R>(link_ptr2(links, s, nu)))));
                            tot += (double)P.m[0][0].real() + (double)P.m[1][1].real();
                        }
                }
    return tot / (2.0 * 6.0 * (double)L.V());
}

}  // namespace

extern "C" {

int gfo_wilson_heatbath_d(double* links, const int* dims, double beta, uint64_t seed, uint32_t sweep_index) {
    if (!dims_ok(dims) || !(beta > 0)) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    wilson_heatbath_sweep<double>(links, L, beta, seed, sweep_index);
    return 0;
}
int gfo_wilson_heatbath_f(float* links, const int* dims, double beta, uint64_t seed, uint32_t sweep_index) {
    if (!dims_ok(dims) || !(beta > 0)) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    wilson_heatbath_sweep<float>(links, L, beta, seed, sweep_index);
    return 0;
}
double gfo_plaquette_d(const double* links, const int* dims) {
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    return plaquette_mean<double>(links, L);
}
double gfo_plaquette_f(const float* links, const int* dims) {
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    return plaquette_mean<float>(links, L);
}
int gfo2_wilson_heatbath_d(double* links, const int* dims, double beta, uint64_t seed, uint32_t sweep_index) {
    if (!dims_ok(dims) || !(beta > 0)) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    wilson_heatbath_sweep2<double>(links, L, beta, seed, sweep_index);
    return 0;
}
int gfo2_wilson_heatbath_f(float* links, const int* dims, double beta, uint64_t seed, uint32_t sweep_index) {
    if (!dims_ok(dims) || !(beta > 0)) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    wilson_heatbath_sweep2<float>(links, L, beta, seed, sweep_index);
    return 0;
}
double gfo2_plaquette_d(const double* links, const int* dims) {
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    return plaquette_mean2<double>(links, L);
}
double gfo2_plaquette_f(const float* links, const int* dims) {
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    return plaquette_mean2<float>(links, L);
}
// staple sum of one link, for the pins
void gfo_staple_d(const double* links, const int* dims, int t, int x, int y, int z, int mu, double* out18) {
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    const int c[4] = {t, x, y, z};
    store<double>(out18, staple_sum<double>(links, L, c, mu));
}

}  // extern "C"
