// =====================================================================================
// gf_oracle_su2.hpp — CPU ORACLE for the gauge group SU(2).
//
// TEST INFRASTRUCTURE, NOT THE PRODUCT (see the header of gf_oracle.cpp, which includes this file
// after its own definitions: the Philox generator, the update rules on the neighbourhood quaternion
// and the Lattice indexer are shared inside the oracle; nothing here is shared with the CUDA path).
//
// The paper states its local problems for SU(2) first (Eq. (20); Eqs. (21)-(29)
// PAPER.md:170-213; theta of Eqs. (12)-(13) PAPER.md:109-113) and reaches SU(3) through the SU(2)
// subgroups; with N_c = 2 there is one "subgroup", the group itself.  Written on std::complex 2x2
// matrices, link by link:  links[t][x][y][z][mu][i][j][re,im], i,j in {0,1} (8 reals per link),
// transforms [t][x][y][z][i][j][re,im].
//
// Pins (tests/test_oracle_su2.py): brute force of Step 1 over a dense SU(2) grid (Landau and MAG),
// Eq. (8) == 2 Eq. (11) - 1, theta = 0 iff stationary, plaquette invariance, unitarity/det, monotone F,
// pure gauge -> F = 1, microcanonical invariance, embedding of an Abelian field (closed form).
// =====================================================================================
#pragma once

namespace {

template <class R>
struct Mat2 {
    std::complex<R> m[2][2];
};
template <class R>
inline Mat2<R> load2(const R* p) {
    Mat2<R> a;
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) a.m[i][j] = std::complex<R>(p[(i * 2 + j) * 2], p[(i * 2 + j) * 2 + 1]);
    return a;
}
template <class R>
inline void store2(R* p, const Mat2<R>& a) {
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) {
            p[(i * 2 + j) * 2] = a.m[i][j].real();
            p[(i * 2 + j) * 2 + 1] = a.m[i][j].imag();
        }
}
template <class R>
inline R* link_ptr2(R* links, int64_t site, int mu) { return links + (site * 4 + mu) * 8; }
template <class R>
inline const R* link_ptr2(const R* links, int64_t site, int mu) { return links + (site * 4 + mu) * 8; }

// Cayley-Klein components of Eq. (15)/(23), from the first row and the second
// row's average (for an exact SU(2) matrix both rows give the same numbers): the un-normalised
// quaternion of Fig. A.10 with (i,j) = (0,1), i.e. TWICE (u0,u1,u2,u3).
template <class R, class A>
inline void add_quaternion2(A q[4], const Mat2<R>& W) {
    q[0] += (A)W.m[0][0].real() + (A)W.m[1][1].real();
    q[3] += (A)W.m[0][0].imag() - (A)W.m[1][1].imag();
    q[2] += (A)W.m[0][1].real() - (A)W.m[1][0].real();
    q[1] += (A)W.m[0][1].imag() + (A)W.m[1][0].imag();
}
template <class R, class A>
inline void add_quaternion2_dagger(A q[4], const Mat2<R>& W) {   // the same for W^dagger
    q[0] += (A)W.m[0][0].real() + (A)W.m[1][1].real();
    q[3] += -(A)W.m[0][0].imag() + (A)W.m[1][1].imag();
    q[2] += (A)W.m[1][0].real() - (A)W.m[0][1].real();
    q[1] += -(A)W.m[1][0].imag() - (A)W.m[0][1].imag();
}

// D, E, F of Eqs. (26)-(28) for one link in Cayley-Klein components u (Eq. (23)),
// with D as corrected in reading R12: D = u0^2 + u3^2 - u1^2 - u2^2.  A down link U_mu(x-mu) enters
// the local functional through W^dagger sigma_3 W (Eq. (12)), i.e. as the up-link
// expressions evaluated on W^dagger, whose components are (w0, -w1, -w2, -w3).
template <class A>
inline void add_mag2(A& D, A& E, A& F, A u0, A u1, A u2, A u3) {
    D += u0 * u0 + u3 * u3 - u1 * u1 - u2 * u2;
    E += (A)2 * (-u0 * u1 - u2 * u3);
    F += (A)2 * (-u0 * u2 + u1 * u3);
}
template <class R, class A>
inline void cayley_klein(const Mat2<R>& W, A u[4]) {   // Eq. (23): first row of the matrix
    u[0] = (A)W.m[0][0].real(); u[3] = (A)W.m[0][0].imag();
    u[2] = (A)W.m[0][1].real(); u[1] = (A)W.m[0][1].imag();
}

// the 2x2 matrix of Eq. (22)
template <class R>
inline Mat2<R> su2_matrix(const R g[4]) {
    Mat2<R> m;
    m.m[0][0] = std::complex<R>(g[0], g[3]);
    m.m[0][1] = std::complex<R>(g[2], g[1]);
    m.m[1][0] = std::complex<R>(-g[2], g[1]);
    m.m[1][1] = std::complex<R>(g[0], -g[3]);
    return m;
}
template <class R>
inline Mat2<R> mul2(const Mat2<R>& a, const Mat2<R>& b) {
    Mat2<R> c;
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) c.m[i][j] = a.m[i][0] * b.m[0][j] + a.m[i][1] * b.m[1][j];
    return c;
}
template <class R>
inline Mat2<R> dagger2(const Mat2<R>& a) {
    Mat2<R> c;
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) c.m[i][j] = std::conj(a.m[j][i]);
    return c;
}

// One site update, N_c = 2: Step 1 on the whole group (Eq. (20) / Eq. (29)), Step 2 on the 2d links.
template <class R, class A>
inline void site_update2(Mat2<R>* up, Mat2<R>* dn, int nd, int gauge, int algo, double param, uint64_t seed,
                         uint32_t site_index, uint32_t sweep_index, Mat2<R>* gtot) {
    A a[4] = {0, 0, 0, 0};
    A Dm = 0, Em = 0, Fm = 0;
    if (gauge == MAG) {
        for (int m = 0; m < nd; ++m) {
            A u[4], w[4];
            cayley_klein<R, A>(up[m], u);
            cayley_klein<R, A>(dn[m], w);
            add_mag2<A>(Dm, Em, Fm, u[0], u[1], u[2], u[3]);
            add_mag2<A>(Dm, Em, Fm, w[0], -w[1], -w[2], -w[3]);
        }
        A lam = std::sqrt(Dm * Dm + Em * Em + Fm * Fm);   // Eq. (29)
        a[0] = Dm + lam; a[1] = -Em; a[2] = -Fm; a[3] = 0;
    } else {
        for (int m = 0; m < nd; ++m) {
            add_quaternion2<R, A>(a, up[m]);
            add_quaternion2_dagger<R, A>(a, dn[m]);
        }
    }
    A g[4];
    if (algo == ALGO_OR) {
        rule_or<A>(a, (A)param, g);
    } else if (algo == ALGO_MICRO) {
        rule_micro<A>(a, g);
    } else if (algo == ALGO_SR) {
        double u = u01(draw(seed, site_index, sweep_index, 0, 0, 0).v[0]);
        if (u < param) rule_micro<A>(a, g);
        else rule_or<A>(a, (A)1, g);
    } else {
        double gd[4];
        if (gauge == MAG) {
            rule_heatbath_mag((double)Dm, (double)Em, (double)Fm, param, seed, site_index, sweep_index, 0, gd);
        } else {
            double ad[4] = {(double)a[0], (double)a[1], (double)a[2], (double)a[3]};
            rule_heatbath_landau(ad, param, seed, site_index, sweep_index, 0, gd);
        }
        for (int k = 0; k < 4; ++k) g[k] = (A)gd[k];
    }
    R gr[4] = {(R)g[0], (R)g[1], (R)g[2], (R)g[3]};
    const Mat2<R> G = su2_matrix<R>(gr), Gd = dagger2<R>(G);
    for (int m = 0; m < nd; ++m) {
        up[m] = mul2<R>(G, up[m]);     // U_mu(x) <- g U_mu(x)
        dn[m] = mul2<R>(dn[m], Gd);    // U_mu(x-mu) <- U_mu(x-mu) g^dagger
    }
    if (gtot) *gtot = mul2<R>(G, *gtot);
}

template <class R, class A>
void half_sweep2(R* links, const Lattice& L, int parity, int gauge, int algo, double param, uint64_t seed,
                 uint32_t sweep_index, R* gtot) {
    const int mu0 = (gauge == COULOMB) ? 1 : 0;
    const int nd = 4 - mu0;
#pragma omp parallel for collapse(2) schedule(static) if (L.V() >= OMP_MIN_SITES)
    for (int t = 0; t < L.Nt; ++t)
        for (int x = 0; x < L.Nx; ++x)
            for (int y = 0; y < L.Ny; ++y)
                for (int z = 0; z < L.Nz; ++z) {
                    int p = (gauge == COULOMB) ? ((x + y + z) & 1) : ((t + x + y + z) & 1);
                    if (p != parity) continue;
                    int64_t s = L.site(t, x, y, z);
                    Mat2<R> up[4], dn[4], gt;
                    int64_t sdn[4];
                    for (int m = 0; m < nd; ++m) {
                        int mu = mu0 + m;
                        sdn[m] = L.shifted(t, x, y, z, mu, -1);
                        up[m] = load2<R>(link_ptr2(links, s, mu));
                        dn[m] = load2<R>(link_ptr2(links, sdn[m], mu));
                    }
                    if (gtot) gt = load2<R>(gtot + s * 8);
                    site_update2<R, A>(up, dn, nd, gauge, algo, param, seed, (uint32_t)s, sweep_index,
                                       gtot ? &gt : nullptr);
                    for (int m = 0; m < nd; ++m) {
                        int mu = mu0 + m;
                        store2<R>(link_ptr2(links, s, mu), up[m]);
                        store2<R>(link_ptr2(links, sdn[m], mu), dn[m]);
                    }
                    if (gtot) store2<R>(gtot + s * 8, gt);
                }
}

// F and theta for N_c = 2.  Landau/Coulomb: Eq. (4), Eqs. (6)-(7) with A = [(U - U^dag)/2i]_traceless.
// MAG: F of Eq. (11); theta of Eq. (13) with X(x) of Eq. (12) formed from the matrices.
// out[0] = F, out[1] = theta, out[2] = F of Eq. (8) (MAG only; = 2 Eq. (11) - 1 on SU(2) links).
template <class R>
void measure2(const R* links, const Lattice& L, int gauge, double* out, double* theta_slice, double* F_slice) {
    typedef std::complex<double> C;
    const int mu0 = (gauge == COULOMB) ? 1 : 0;
    const int nd = 4 - mu0;
    std::vector<double> fs(L.Nt, 0.0), ths(L.Nt, 0.0), f8(L.Nt, 0.0);
#pragma omp parallel for schedule(static) if (L.V() >= OMP_MIN_SITES)
    for (int t = 0; t < L.Nt; ++t) {
        double f_acc = 0, th_acc = 0, f8_acc = 0;
        for (int x = 0; x < L.Nx; ++x)
            for (int y = 0; y < L.Ny; ++y)
                for (int z = 0; z < L.Nz; ++z) {
                    int64_t s = L.site(t, x, y, z);
                    C X[2][2] = {{C(0, 0), C(0, 0)}, {C(0, 0), C(0, 0)}};
                    for (int mu = mu0; mu < 4; ++mu) {
                        Mat2<R> Ur = load2<R>(link_ptr2(links, s, mu));
                        Mat2<R> Wr = load2<R>(link_ptr2(links, L.shifted(t, x, y, z, mu, -1), mu));
                        C U[2][2], W[2][2];
                        for (int i = 0; i < 2; ++i)
                            for (int j = 0; j < 2; ++j) { U[i][j] = C(Ur.m[i][j]); W[i][j] = C(Wr.m[i][j]); }
                        if (gauge == MAG) {
                            const double s3[2] = {1.0, -1.0};
                            for (int i = 0; i < 2; ++i) f_acc += std::norm(U[i][i]);
                            for (int i = 0; i < 2; ++i)      // tr[sigma3 U sigma3 U^dag] = sum_ij s_i s_j |U_ij|^2
                                for (int j = 0; j < 2; ++j) f8_acc += s3[i] * s3[j] * std::norm(U[i][j]);
                            for (int i = 0; i < 2; ++i)      // Eq. (12): U sigma3 U^dag + W^dag sigma3 W
                                for (int j = 0; j < 2; ++j)
                                    for (int k = 0; k < 2; ++k)
                                        X[i][j] += U[i][k] * s3[k] * std::conj(U[j][k]) + std::conj(W[k][i]) * s3[k] * W[k][j];
                        } else {
                            f_acc += U[0][0].real() + U[1][1].real();
                            for (int w = 0; w < 2; ++w) {
                                C(*M)[2] = (w == 0) ? U : W;
                                C A[2][2];
                                for (int i = 0; i < 2; ++i)
                                    for (int j = 0; j < 2; ++j) A[i][j] = (M[i][j] - std::conj(M[j][i])) / C(0, 2);
                                C trA = A[0][0] + A[1][1];
                                A[0][0] -= trA / 2.0; A[1][1] -= trA / 2.0;
                                const double sign = (w == 0) ? 1.0 : -1.0;
                                for (int i = 0; i < 2; ++i)
                                    for (int j = 0; j < 2; ++j) X[i][j] += sign * A[i][j];   // X holds Delta(x)
                            }
                        }
                    }
                    if (gauge == MAG) th_acc += std::norm(X[0][1]);   // Eq. (13)
                    else
                        for (int i = 0; i < 2; ++i)
                            for (int j = 0; j < 2; ++j) th_acc += std::norm(X[i][j]);   // tr[Delta Delta^dag]
                }
        fs[t] = f_acc; ths[t] = th_acc; f8[t] = f8_acc;
    }
    const double Vs = (double)L.Nx * L.Ny * L.Nz, V = (double)L.V();
    double Fsum = 0, Th = 0, F8 = 0;
    for (int t = 0; t < L.Nt; ++t) {
        Fsum += fs[t]; Th += ths[t]; F8 += f8[t];
        if (theta_slice) theta_slice[t] = ths[t] / (2.0 * Vs);
        if (F_slice) F_slice[t] = fs[t] / (2.0 * nd * Vs);
    }
    out[0] = Fsum / (2.0 * nd * V);
    out[1] = Th / (2.0 * V);
    out[2] = F8 / (2.0 * nd * V);
}

// Reprojection to SU(2): first row normalised in double, second row (-conj b, conj a) — the N_c = 2
// analogue of "third row = (u x v)^*" (reading R20).
template <class R>
void reunitarize2(R* mats, int64_t n) {
    for (int64_t k = 0; k < n; ++k) {
        R* p = mats + k * 8;
        std::complex<double> a(p[0], p[1]), b(p[2], p[3]);
        const double nrm = 1.0 / std::sqrt(std::norm(a) + std::norm(b));
        a *= nrm; b *= nrm;
        p[0] = (R)a.real(); p[1] = (R)a.imag(); p[2] = (R)b.real(); p[3] = (R)b.imag();
        p[4] = (R)(-b.real()); p[5] = (R)b.imag(); p[6] = (R)a.real(); p[7] = (R)(-a.imag());
    }
}

template <class R>
void coulomb_finalize2(R* links, const R* gtot, const Lattice& L) {
    for (int t = 0; t < L.Nt; ++t)
        for (int x = 0; x < L.Nx; ++x)
            for (int y = 0; y < L.Ny; ++y)
                for (int z = 0; z < L.Nz; ++z) {
                    int64_t s = L.site(t, x, y, z), sf = L.shifted(t, x, y, z, 0, +1);
                    Mat2<R> G = load2<R>(gtot + s * 8), H = load2<R>(gtot + sf * 8);
                    Mat2<R> U = load2<R>(link_ptr2(links, s, 0));
                    store2<R>(link_ptr2(links, s, 0), mul2<R>(mul2<R>(G, U), dagger2<R>(H)));
                }
}

template <class R>
int sweep2_dispatch(R* links, const int* dims, int parity_mask, int gauge, int algo, double param, uint64_t seed,
                    uint32_t sweep_index, int step1_double, R* gtot) {
    if (!dims_ok(dims) || gauge < 0 || gauge > 2 || algo < 0 || algo > 3) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    for (int p = 0; p < 2; ++p) {
        if (!(parity_mask & (1 << p))) continue;
        if (step1_double) half_sweep2<R, double>(links, L, p, gauge, algo, param, seed, sweep_index, gtot);
        else half_sweep2<R, R>(links, L, p, gauge, algo, param, seed, sweep_index, gtot);
    }
    return 0;
}

}  // namespace

extern "C" {

int gfo2_sweep_d(double* links, const int* dims, int parity_mask, int gauge, int algo, double param, uint64_t seed,
                 uint32_t sweep_index, double* gtot) {
    return sweep2_dispatch<double>(links, dims, parity_mask, gauge, algo, param, seed, sweep_index, 1, gtot);
}
int gfo2_sweep_f(float* links, const int* dims, int parity_mask, int gauge, int algo, double param, uint64_t seed,
                 uint32_t sweep_index, int step1_double, float* gtot) {
    return sweep2_dispatch<float>(links, dims, parity_mask, gauge, algo, param, seed, sweep_index, step1_double, gtot);
}
int gfo2_measure_d(const double* links, const int* dims, int gauge, double* out3, double* theta_slice, double* F_slice) {
    if (!dims_ok(dims)) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    measure2<double>(links, L, gauge, out3, theta_slice, F_slice);
    return 0;
}
int gfo2_measure_f(const float* links, const int* dims, int gauge, double* out3, double* theta_slice, double* F_slice) {
    if (!dims_ok(dims)) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    measure2<float>(links, L, gauge, out3, theta_slice, F_slice);
    return 0;
}
void gfo2_reunitarize_d(double* mats, int64_t n) { reunitarize2<double>(mats, n); }
void gfo2_reunitarize_f(float* mats, int64_t n) { reunitarize2<float>(mats, n); }
int gfo2_coulomb_finalize_d(double* links, const double* gtot, const int* dims) {
    if (!dims_ok(dims)) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    coulomb_finalize2<double>(links, gtot, L);
    return 0;
}
int gfo2_coulomb_finalize_f(float* links, const float* gtot, const int* dims) {
    if (!dims_ok(dims)) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    coulomb_finalize2<float>(links, gtot, L);
    return 0;
}
// one site from caller-gathered links: up/dn = nd matrices of 8 reals
void gfo2_site_update_d(double* up, double* dn, int nd, int gauge, int algo, double param, uint64_t seed,
                        uint32_t site_index, uint32_t sweep_index) {
    Mat2<double> u[4], d[4];
    for (int m = 0; m < nd; ++m) { u[m] = load2<double>(up + m * 8); d[m] = load2<double>(dn + m * 8); }
    site_update2<double, double>(u, d, nd, gauge, algo, param, seed, site_index, sweep_index, nullptr);
    for (int m = 0; m < nd; ++m) { store2<double>(up + m * 8, u[m]); store2<double>(dn + m * 8, d[m]); }
}
// Haar on SU(2) (uniform on S^3): first row (a, b) = two complex standard normals — Box-Muller on the
// Philox uniforms of counter (site, 0, 0 | 3 << 8, 0), as in gfo_haar_field_d with k = 0 — normalised;
// second row (-conj b, conj a).  h: [V][2][2][2] doubles.
void gfo2_haar_field_d(double* h, const int* dims, uint64_t seed) {
    const int64_t V = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
    const double two_pi = 6.283185307179586477;
    for (int64_t s = 0; s < V; ++s) {
        double* p = h + s * 8;
        Philox4 w = draw(seed, (uint32_t)s, 0u, 0, 3, 0u);
        const double r0 = std::sqrt(-2.0 * std::log(u01(w.v[0]))), r1 = std::sqrt(-2.0 * std::log(u01(w.v[2])));
        p[0] = r0 * std::cos(two_pi * u01(w.v[1]));
        p[1] = r0 * std::sin(two_pi * u01(w.v[1]));
        p[2] = r1 * std::cos(two_pi * u01(w.v[3]));
        p[3] = r1 * std::sin(two_pi * u01(w.v[3]));
    }
    reunitarize2<double>(h, V);
}

}  // extern "C"
