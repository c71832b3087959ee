// =====================================================================================
// gf_oracle.cpp — CPU ORACLE for SU(3) lattice gauge fixing (arxiv/paper_1212_5221).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, by-the-book
// implementation of the paper's Alg. 1, written on std::complex 3x3
// matrices in the natural StandardPattern order, link by link and subgroup
// by subgroup exactly as the paper states it.  It shares no code with the CUDA path
// (paper_1212_5221_b200/csrc) and must never be imported by it: only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may call it.
//
// Layout: links[t][x][y][z][mu][i][j][re,im]   mu = 0 temporal, 1,2,3 = x,y,z
//         ("StandardPattern: t,x,y,z,mu,i,j,c"; PAPER.md:450 U_0 temporal).
// dims are passed as (Nt, Nx, Ny, Nz).
//
// Readings of the paper where it is silent/garbled are those of DESIGN.md §3 (R1..R20);
// each function cites the passage it follows.
//
// Parity pins (tests/test_oracle_*.py): pure gauge -> F=1, theta->0; plaquette invariance;
// unitarity/det; monotone F at omega=1; exact F-invariance of microcanonical sweeps;
// one-site brute force of Step 1 (Landau and MAG); Coulomb slice == standalone 3-d problem;
// heatbath histograms vs closed-form densities, T->0 limit; Philox known answers; theta_MAG (both forms) vs
// Eq. (12) evaluated with NumPy matrices on a rough field and vs the N_c = 2 value on embedded SU(2) links.
// "parity unpinned" items (no value in the paper pins them; any fixed choice is a valid
// algorithm): subgroup order (R6), MAG heatbath construction (R15), Philox keying (R19).
// =====================================================================================
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum Gauge { LANDAU = 0, COULOMB = 1, MAG = 2 };
enum Algo { ALGO_OR = 0, ALGO_SR = 1, ALGO_SA = 2, ALGO_MICRO = 3 };

// OpenMP over the sites of one parity only where the lattice is big enough to pay for the fork
const int64_t OMP_MIN_SITES = 32768;

// ---------------------------------------------------------------------------------
// Philox4x32-10 (Random123, PAPER.md:249 fn. 2, ref. [32] PAPER.md:672).  Reading R19.
// ---------------------------------------------------------------------------------
struct Philox4 {
    uint32_t v[4];
};

inline Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                             uint32_t k1) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;   // multipliers
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;   // Weyl key increments
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    Philox4 r;
    r.v[0] = c0; r.v[1] = c1; r.v[2] = c2; r.v[3] = c3;
    return r;
}

// uniform in (0,1): (u32 + 0.5) * 2^-32, evaluated in double in all precision modes (R19)
inline double u01(uint32_t w) { return ((double)w + 0.5) * (1.0 / 4294967296.0); }

// draw for (site, sweep, subgroup, purpose, trial): counter = (site, sweep, sub | purpose<<8, trial)
inline Philox4 draw(uint64_t seed, uint32_t site, uint32_t sweep, int sub, int purpose,
                    uint32_t trial) {
    return philox4x32_10(site, sweep, (uint32_t)sub | ((uint32_t)purpose << 8), trial,
                         (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32));
}

// ---------------------------------------------------------------------------------
// 3x3 complex matrices
// ---------------------------------------------------------------------------------
template <class R>
struct Mat3 {
    std::complex<R> m[3][3];
};

template <class R>
inline Mat3<R> load(const R* p) {
    Mat3<R> a;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) a.m[i][j] = std::complex<R>(p[(i * 3 + j) * 2], p[(i * 3 + j) * 2 + 1]);
    return a;
}
template <class R>
inline void store(R* p, const Mat3<R>& a) {
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            p[(i * 3 + j) * 2] = a.m[i][j].real();
            p[(i * 3 + j) * 2 + 1] = a.m[i][j].imag();
        }
}

struct Lattice {
    int Nt, Nx, Ny, Nz;
    int64_t V() const { return (int64_t)Nt * Nx * Ny * Nz; }
    int64_t site(int t, int x, int y, int z) const { return (((int64_t)t * Nx + x) * Ny + y) * Nz + z; }
    // neighbour of (t,x,y,z) displaced by dir (+1/-1) along mu, periodic
    int64_t shifted(int t, int x, int y, int z, int mu, int dir) const {
        int c[4] = {t, x, y, z};
        const int n[4] = {Nt, Nx, Ny, Nz};
        c[mu] = (c[mu] + dir + n[mu]) % n[mu];
        return site(c[0], c[1], c[2], c[3]);
    }
};

template <class R>
inline R* link_ptr(R* links, int64_t site, int mu) { return links + (site * 4 + mu) * 18; }
template <class R>
inline const R* link_ptr(const R* links, int64_t site, int mu) { return links + (site * 4 + mu) * 18; }

// ---------------------------------------------------------------------------------
// Fig. A.10 with its lost signs restored (reading R1), in the
// Cayley-Klein convention of Eq. (15)/(22):
//   W_sub = [[q0 + i q3, q2 + i q1], [-q2 + i q1, q0 - i q3]]  (times 2, un-normalised)
// ---------------------------------------------------------------------------------
template <class R, class A>
inline void add_quaternion(A q[4], const Mat3<R>& W, int i, int j) {
    q[0] += (A)W.m[i][i].real() + (A)W.m[j][j].real();
    q[3] += (A)W.m[i][i].imag() - (A)W.m[j][j].imag();
    q[2] += (A)W.m[i][j].real() - (A)W.m[j][i].real();
    q[1] += (A)W.m[i][j].imag() + (A)W.m[j][i].imag();
}
// the same for W^dagger without forming it: (W^dag)_ab = conj(W_ba)
template <class R, class A>
inline void add_quaternion_dagger(A q[4], const Mat3<R>& W, int i, int j) {
    q[0] += (A)W.m[i][i].real() + (A)W.m[j][j].real();
    q[3] += -(A)W.m[i][i].imag() + (A)W.m[j][j].imag();
    q[2] += (A)W.m[j][i].real() - (A)W.m[i][j].real();
    q[1] += -(A)W.m[j][i].imag() - (A)W.m[i][j].imag();
}

// ---------------------------------------------------------------------------------
// MAG local quadratic form, SU(3) analogue of Eqs. (24)-(28) derived
// from the functional actually used, Eq. (11) (reading R12):
//   f(g) = const + g^T [[D,E,F],[E,-D,0],[F,0,-D]] g,   g = (g0,g1,g2), g3 = 0.
// up-link W = U_mu(x) enters as g W, down-link W = U_mu(x-mu) as W g^dagger.
// ---------------------------------------------------------------------------------
template <class R, class A>
inline void add_mag_up(A& a, A& b, A& E, A& F, const Mat3<R>& W, int i, int j) {
    typedef std::complex<A> C;
    C ii(W.m[i][i]), jj(W.m[j][j]), ij(W.m[i][j]), ji(W.m[j][i]);
    a += std::norm(ii) + std::norm(jj);
    b += std::norm(ij) + std::norm(ji);
    C s = ji * std::conj(ii) + ij * std::conj(jj);
    C d = ji * std::conj(ii) - ij * std::conj(jj);
    E += -s.imag();
    F += d.real();
}
template <class R, class A>
inline void add_mag_down(A& a, A& b, A& E, A& F, const Mat3<R>& W, int i, int j) {
    typedef std::complex<A> C;
    C ii(W.m[i][i]), jj(W.m[j][j]), ij(W.m[i][j]), ji(W.m[j][i]);
    a += std::norm(ii) + std::norm(jj);
    b += std::norm(ij) + std::norm(ji);
    C s = ij * std::conj(ii) + ji * std::conj(jj);
    C d = ij * std::conj(ii) - ji * std::conj(jj);
    E += s.imag();
    F += d.real();
}

// ---------------------------------------------------------------------------------
// Step 1 update rules.  Input: the accumulated quaternion a (Landau/Coulomb: Eq. (19)
// PAPER.md:154 summed as quaternions; MAG: a = (D+lambda, -E, -F, 0)).
// The local functional is g0 a0 - g1 a1 - g2 a2 - g3 a3 (+const), maximised by
// g_hat = conj(a)/|a| = (a0,-a1,-a2,-a3)/|a|, which is Eq. (20) in the subgroup.
// Output: the SU(2) element g = (g0,g1,g2,g3) in the convention of Eq. (22).
// ---------------------------------------------------------------------------------

// Overrelaxation, Fig. A.11 verbatim; omega=1 is plain relaxation.
template <class A>
inline void rule_or(const A a[4], A omega, A g[4]) {
    A ai_sq = a[1] * a[1] + a[2] * a[2] + a[3] * a[3];
    A a0_sq = a[0] * a[0];
    if (a0_sq + ai_sq == (A)0) { g[0] = 1; g[1] = g[2] = g[3] = 0; return; }
    A b = (omega * a0_sq + ai_sq) / (a0_sq + ai_sq);
    A c = (A)1 / std::sqrt(a0_sq + b * b * ai_sq);
    g[0] = a[0] * c;
    g[1] = -a[1] * (b * c);
    g[2] = -a[2] * (b * c);
    g[3] = -a[3] * (b * c);
}

// Microcanonical step: the exact square of g_hat (reading R4).
template <class A>
inline void rule_micro(const A a[4], A g[4]) {
    A n2 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2] + a[3] * a[3];
    if (n2 == (A)0) { g[0] = 1; g[1] = g[2] = g[3] = 0; return; }
    A inv = (A)1 / std::sqrt(n2);
    A h0 = a[0] * inv, h1 = -a[1] * inv, h2 = -a[2] * inv, h3 = -a[3] * inv;
    g[0] = (A)2 * h0 * h0 - (A)1;
    g[1] = (A)2 * h0 * h1;
    g[2] = (A)2 * h0 * h2;
    g[3] = (A)2 * h0 * h3;
}

// quaternion product in the convention of Eq. (22): M(p)M(q), M(g) = g0 + i g.sigma
inline void qmul(const double p[4], const double q[4], double r[4]) {
    r[0] = p[0] * q[0] - p[1] * q[1] - p[2] * q[2] - p[3] * q[3];
    r[1] = p[0] * q[1] + q[0] * p[1] - (p[2] * q[3] - p[3] * q[2]);
    r[2] = p[0] * q[2] + q[0] * p[2] - (p[3] * q[1] - p[1] * q[3]);
    r[3] = p[0] * q[3] + q[0] * p[3] - (p[1] * q[2] - p[2] * q[1]);
}

const double TWO_PI = 6.283185307179586476925286766559;
const int HB_MAX_TRIALS = 64;

// Heatbath for Landau/Coulomb at temperature T (Eq. (30); reading R14):
// P(g) ~ exp(Re tr[g K]/T).  With u = g * g_hat^{-1}: density of u0 ~ sqrt(1-u0^2) exp(alpha u0),
// alpha = |a|/T.  Kennedy-Pendleton for alpha >= 2, Creutz for alpha < 2; all in double.
inline void rule_heatbath_landau(const double a[4], double T, uint64_t seed, uint32_t site,
                                 uint32_t sweep, int sub, double g[4]) {
    double n2 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2] + a[3] * a[3];
    if (n2 == 0.0) { g[0] = 1; g[1] = g[2] = g[3] = 0; return; }
    double norm = std::sqrt(n2);
    double alpha = norm / T;
    double ghat[4] = {a[0] / norm, -a[1] / norm, -a[2] / norm, -a[3] / norm};
    double u0 = 1.0;
    if (alpha >= 2.0) {
        for (uint32_t trial = 0; trial < (uint32_t)HB_MAX_TRIALS; ++trial) {
            Philox4 r = draw(seed, site, sweep, sub, 1, trial);
            double r1 = u01(r.v[0]), r2 = u01(r.v[1]), r3 = u01(r.v[2]), r4 = u01(r.v[3]);
            double cs = std::cos(TWO_PI * r2);
            double delta = -(std::log(r1) + cs * cs * std::log(r3)) / alpha;
            u0 = 1.0 - delta;
            if (r4 * r4 <= 1.0 - 0.5 * delta) break;
        }
    } else {
        double em = std::exp(-2.0 * alpha);
        for (uint32_t trial = 0; trial < (uint32_t)HB_MAX_TRIALS; ++trial) {
            Philox4 r = draw(seed, site, sweep, sub, 1, trial);
            double r1 = u01(r.v[0]), r2 = u01(r.v[1]);
            double x = em + (1.0 - em) * r1;
            u0 = 1.0 + std::log(x) / alpha;
            if (r2 * r2 <= 1.0 - u0 * u0) break;
        }
    }
    if (u0 > 1.0) u0 = 1.0;
    if (u0 < -1.0) u0 = -1.0;
    Philox4 rd = draw(seed, site, sweep, sub, 2, 0);
    double ct = 2.0 * u01(rd.v[0]) - 1.0;
    double phi = TWO_PI * u01(rd.v[1]);
    double st = std::sqrt(std::fmax(0.0, 1.0 - ct * ct));
    double rad = std::sqrt(std::fmax(0.0, 1.0 - u0 * u0));
    double u[4] = {u0, rad * st * std::cos(phi), rad * st * std::sin(phi), rad * ct};
    double r[4];
    qmul(u, ghat, r);
    double rn = 1.0 / std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2] + r[3] * r[3]);
    for (int k = 0; k < 4; ++k) g[k] = r[k] * rn;
}

// Heatbath for MAG (paper silent; reading R15 = our construction):
// with g0 = cos(al), (g1,g2) = sin(al)(cos(be), sin(be)):  f = const + phi.X,
// phi = (sin 2al cos be, sin 2al sin be, cos 2al) on S^2, X = (E,F,D), |X| = lambda.
// Sample phi ~ exp(phi.X/T) on S^2 (closed-form inverse CDF), no rejection.
inline void rule_heatbath_mag(double D, double E, double F, double T, uint64_t seed, uint32_t site,
                              uint32_t sweep, int sub, double g[4]) {
    double lam = std::sqrt(D * D + E * E + F * F);
    if (lam == 0.0) { g[0] = 1; g[1] = g[2] = g[3] = 0; return; }
    Philox4 r = draw(seed, site, sweep, sub, 1, 0);
    double r1 = u01(r.v[0]), r2 = u01(r.v[1]);
    double cg = 1.0 + (T / lam) * std::log(1.0 - r1 * (1.0 - std::exp(-2.0 * lam / T)));
    if (cg < -1.0) cg = -1.0;
    if (cg > 1.0) cg = 1.0;
    double sg = std::sqrt(std::fmax(0.0, 1.0 - cg * cg));
    double X[3] = {E / lam, F / lam, D / lam};
    // e1 = normalise(z_hat x X_hat) = (-X1, X0, 0)/|.|, y_hat if degenerate; e2 = X_hat x e1
    double e1[3] = {-X[1], X[0], 0.0};
    double n1 = std::sqrt(e1[0] * e1[0] + e1[1] * e1[1]);
    if (n1 < 1e-150) { e1[0] = 0.0; e1[1] = 1.0; e1[2] = 0.0; }
    else { e1[0] /= n1; e1[1] /= n1; }
    double e2[3] = {X[1] * e1[2] - X[2] * e1[1], X[2] * e1[0] - X[0] * e1[2], X[0] * e1[1] - X[1] * e1[0]};
    double az = TWO_PI * r2;
    double ca = std::cos(az), sa = std::sin(az);
    double phi[3];
    for (int k = 0; k < 3; ++k) phi[k] = cg * X[k] + sg * (ca * e1[k] + sa * e2[k]);
    double h = 0.5 * (1.0 + phi[2]);
    if (h < 1e-300) { g[0] = 0; g[1] = 1; g[2] = 0; g[3] = 0; return; }
    double g0 = std::sqrt(h);
    double g1 = phi[0] / (2.0 * g0), g2 = phi[1] / (2.0 * g0);
    double rn = 1.0 / std::sqrt(g0 * g0 + g1 * g1 + g2 * g2);
    g[0] = g0 * rn; g[1] = g1 * rn; g[2] = g2 * rn; g[3] = 0.0;
}

// ---------------------------------------------------------------------------------
// Step 2 (Fig. A.9, body missing -> reading R2):
// left multiplication by the SU(2) element embedded in rows (i,j) via Eq. (22) PAPER.md:178,
// per column k: 4 complex mul + 2 complex add.
// ---------------------------------------------------------------------------------
template <class R>
inline void left_mul_subgroup(Mat3<R>& U, const R g[4], int i, int j) {
    typedef std::complex<R> C;
    C g00(g[0], g[3]), g01(g[2], g[1]), g10(-g[2], g[1]), g11(g[0], -g[3]);
    for (int k = 0; k < 3; ++k) {
        C ui = U.m[i][k], uj = U.m[j][k];
        U.m[i][k] = g00 * ui + g01 * uj;
        U.m[j][k] = g10 * ui + g11 * uj;
    }
}
// right multiplication by the dagger: U <- U g~^dagger, acts on columns (i,j)
template <class R>
inline void right_mul_subgroup_dagger(Mat3<R>& U, const R g[4], int i, int j) {
    typedef std::complex<R> C;
    // g^dagger = [[conj g00, conj g10],[conj g01, conj g11]]
    C d00(g[0], -g[3]), d01(-g[2], -g[1]), d10(g[2], -g[1]), d11(g[0], g[3]);
    for (int k = 0; k < 3; ++k) {
        C ui = U.m[k][i], uj = U.m[k][j];
        U.m[k][i] = ui * d00 + uj * d10;
        U.m[k][j] = ui * d01 + uj * d11;
    }
}

const int SUB_I[3] = {0, 0, 1};   // subgroup order (0,1),(0,2),(1,2), one pass (reading R6)
const int SUB_J[3] = {1, 2, 2};

// ---------------------------------------------------------------------------------
// One site update = the body of Alg. 1's "for all x of sublattice".
// up[mu], dn[mu] are the 2d links U_mu(x), U_mu(x-mu) (mu over `dirs`), modified in place.
// R = storage/Step-2 type; A = Step-1 type (double for MP/DP, float for SP).
// ---------------------------------------------------------------------------------
template <class R, class A>
inline void site_update(Mat3<R>* up, Mat3<R>* dn, int nd, int gauge, int algo, double param,
                        uint64_t seed, uint32_t site_index, uint32_t sweep_index, Mat3<R>* gtot) {
    for (int s = 0; s < 3; ++s) {
        const int i = SUB_I[s], j = SUB_J[s];
        A a[4] = {0, 0, 0, 0};
        A Dm = 0, Em = 0, Fm = 0;
        // ---- Step 1: local optimisation ----
        if (gauge == MAG) {
            A sa = 0, sb = 0;
            for (int m = 0; m < nd; ++m) {
                add_mag_up<R, A>(sa, sb, Em, Fm, up[m], i, j);
                add_mag_down<R, A>(sa, sb, Em, Fm, dn[m], i, j);
            }
            Dm = (sa - sb) / (A)2;
            A lam = std::sqrt(Dm * Dm + Em * Em + Fm * Fm);   // Eq. (29)
            a[0] = Dm + lam; a[1] = -Em; a[2] = -Fm; a[3] = 0;
        } else {
            for (int m = 0; m < nd; ++m) {
                add_quaternion<R, A>(a, up[m], i, j);
                add_quaternion_dagger<R, A>(a, dn[m], i, j);
            }
        }
        A g[4];
        if (algo == ALGO_OR) {
            rule_or<A>(a, (A)param, g);
        } else if (algo == ALGO_MICRO) {
            rule_micro<A>(a, g);
        } else if (algo == ALGO_SR) {
            // stochastic relaxation: g^2 with probability p, else g
            double u = u01(draw(seed, site_index, sweep_index, s, 0, 0).v[0]);
            if (u < param) rule_micro<A>(a, g);
            else rule_or<A>(a, (A)1, g);
        } else {   // ALGO_SA: heatbath at temperature T = param, scalar math in double (R14/R15)
            double gd[4];
            if (gauge == MAG) {
                rule_heatbath_mag((double)Dm, (double)Em, (double)Fm, param, seed, site_index, sweep_index, s, gd);
            } else {
                double ad[4] = {(double)a[0], (double)a[1], (double)a[2], (double)a[3]};
                rule_heatbath_landau(ad, param, seed, site_index, sweep_index, s, gd);
            }
            for (int k = 0; k < 4; ++k) g[k] = (A)gd[k];
        }
        R gr[4] = {(R)g[0], (R)g[1], (R)g[2], (R)g[3]};
        // ---- Step 2: apply g to U_mu(x), U_mu(x-mu) ----
        for (int m = 0; m < nd; ++m) {
            left_mul_subgroup<R>(up[m], gr, i, j);
            right_mul_subgroup_dagger<R>(dn[m], gr, i, j);
        }
        if (gtot) left_mul_subgroup<R>(*gtot, gr, i, j);
    }
}

// ---------------------------------------------------------------------------------
// Half sweep over one parity (Alg. 1 "for sublattice = even, odd").
// Landau/MAG: parity = (t+x+y+z)&1 (PAPER.md:293 fn. 3).  Coulomb: (x+y+z)&1 in every
// time-slice, mu restricted to spatial directions (reading R21).
// ---------------------------------------------------------------------------------
template <class R, class A>
void half_sweep(R* links, const Lattice& L, int parity, int gauge, int algo, double param,
                uint64_t seed, uint32_t sweep_index, R* gtot) {
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
                    Mat3<R> up[4], dn[4], gt;
                    int64_t sdn[4];
                    for (int m = 0; m < nd; ++m) {
                        int mu = mu0 + m;
                        sdn[m] = L.shifted(t, x, y, z, mu, -1);
                        up[m] = load<R>(link_ptr(links, s, mu));
                        dn[m] = load<R>(link_ptr(links, sdn[m], mu));
                    }
                    if (gtot) gt = load<R>(gtot + s * 18);
                    site_update<R, A>(up, dn, nd, gauge, algo, param, seed, (uint32_t)s, sweep_index,
                                      gtot ? &gt : nullptr);
                    for (int m = 0; m < nd; ++m) {
                        int mu = mu0 + m;
                        store<R>(link_ptr(links, s, mu), up[m]);
                        store<R>(link_ptr(links, sdn[m], mu), dn[m]);
                    }
                    if (gtot) store<R>(gtot + s * 18, gt);
                }
}

// ---------------------------------------------------------------------------------
// F and theta (Eq. 4, 80-82 Eqs. 6-7; MAG PAPER.md:102 Eq. 11 and reading R11).
// Always accumulated in double (BASELINE.json: "DP reductions").
// out[0]=F, out[1]=theta, out[2]=theta_literal (MAG only: |sum_s X^s_12|^2 form of Eq. 16);
// theta_slice[t] (Coulomb/any gauge: per-time-slice theta with V -> Nx Ny Nz), F_slice[t].
// ---------------------------------------------------------------------------------
template <class R>
void measure(const R* links, const Lattice& L, int gauge, double* out, double* theta_slice,
             double* F_slice) {
    const int mu0 = (gauge == COULOMB) ? 1 : 0;
    const int nd = 4 - mu0;
    std::vector<double> fs(L.Nt, 0.0), ths(L.Nt, 0.0), thl(L.Nt, 0.0);
    typedef std::complex<double> C;
#pragma omp parallel for schedule(static) if (L.V() >= OMP_MIN_SITES)
    for (int t = 0; t < L.Nt; ++t) {
        double f_acc = 0, th_acc = 0, thl_acc = 0;
        for (int x = 0; x < L.Nx; ++x)
            for (int y = 0; y < L.Ny; ++y)
                for (int z = 0; z < L.Nz; ++z) {
                    int64_t s = L.site(t, x, y, z);
                    if (gauge == MAG) {
                        // F: sum_i |U_ii|^2 over the links starting at x (Eq. 11)
                        for (int mu = 0; mu < 4; ++mu) {
                            Mat3<R> U = load<R>(link_ptr(links, s, mu));
                            for (int i = 0; i < 3; ++i) f_acc += std::norm(C(U.m[i][i]));
                        }
                        // theta: per subgroup X^s_12 = F_s + i E_s (reading R11)
                        C lit(0, 0);
                        for (int sgi = 0; sgi < 3; ++sgi) {
                            double a = 0, b = 0, E = 0, F = 0;
                            for (int mu = 0; mu < 4; ++mu) {
                                Mat3<R> U = load<R>(link_ptr(links, s, mu));
                                Mat3<R> W = load<R>(link_ptr(links, L.shifted(t, x, y, z, mu, -1), mu));
                                add_mag_up<R, double>(a, b, E, F, U, SUB_I[sgi], SUB_J[sgi]);
                                add_mag_down<R, double>(a, b, E, F, W, SUB_I[sgi], SUB_J[sgi]);
                            }
                            th_acc += E * E + F * F;
                            lit += C(F, E);
                        }
                        thl_acc += std::norm(lit);
                    } else {
                        // Delta(x) = sum_mu A_mu(x) - A_mu(x-mu),  A = [(U - U^dag)/2i]_traceless (R8)
                        C Dl[3][3];
                        for (int i = 0; i < 3; ++i)
                            for (int j = 0; j < 3; ++j) Dl[i][j] = C(0, 0);
                        for (int mu = mu0; mu < 4; ++mu) {
                            Mat3<R> U = load<R>(link_ptr(links, s, mu));
                            Mat3<R> W = load<R>(link_ptr(links, L.shifted(t, x, y, z, mu, -1), mu));
                            double tr = 0;
                            for (int i = 0; i < 3; ++i) tr += (double)U.m[i][i].real();
                            f_acc += tr;
                            const Mat3<R>* Ms[2] = {&U, &W};
                            for (int w = 0; w < 2; ++w) {
                                const Mat3<R>& M = *Ms[w];
                                C A[3][3];
                                C trA(0, 0);
                                for (int i = 0; i < 3; ++i)
                                    for (int j = 0; j < 3; ++j)
                                        A[i][j] = (C(M.m[i][j]) - std::conj(C(M.m[j][i]))) / C(0, 2);
                                for (int i = 0; i < 3; ++i) trA += A[i][i];
                                for (int i = 0; i < 3; ++i) A[i][i] -= trA / 3.0;
                                double sign = (w == 0) ? 1.0 : -1.0;
                                for (int i = 0; i < 3; ++i)
                                    for (int j = 0; j < 3; ++j) Dl[i][j] += sign * A[i][j];
                            }
                        }
                        double n = 0;   // tr[Delta Delta^dag] = sum |Delta_ij|^2
                        for (int i = 0; i < 3; ++i)
                            for (int j = 0; j < 3; ++j) n += std::norm(Dl[i][j]);
                        th_acc += n;
                    }
                }
        fs[t] = f_acc; ths[t] = th_acc; thl[t] = thl_acc;
    }
    double Vs = (double)L.Nx * L.Ny * L.Nz;
    double Fsum = 0, Th = 0, ThL = 0;
    for (int t = 0; t < L.Nt; ++t) {
        Fsum += fs[t]; Th += ths[t]; ThL += thl[t];
        if (theta_slice) theta_slice[t] = ths[t] / (3.0 * Vs);
        if (F_slice) F_slice[t] = fs[t] / (3.0 * nd * Vs);
    }
    double V = (double)L.V();
    out[0] = Fsum / (3.0 * nd * V);
    out[1] = Th / (3.0 * V);
    out[2] = ThL / (3.0 * V);
}

// ---------------------------------------------------------------------------------
// Reprojection to SU(3) (method unstated -> reading R20): Gram-Schmidt on rows
// 0,1 in double, third row = (u x v)^* (PAPER.md:351), rounded to the storage type.
// ---------------------------------------------------------------------------------
template <class R>
void reunitarize(R* mats, int64_t n) {
    typedef std::complex<double> C;
#pragma omp parallel for schedule(static) if (n >= 4 * OMP_MIN_SITES)
    for (int64_t k = 0; k < n; ++k) {
        R* p = mats + k * 18;
        C u[3], v[3], w[3];
        for (int j = 0; j < 3; ++j) {
            u[j] = C(p[j * 2], p[j * 2 + 1]);
            v[j] = C(p[(3 + j) * 2], p[(3 + j) * 2 + 1]);
        }
        double nu = 0;
        for (int j = 0; j < 3; ++j) nu += std::norm(u[j]);
        nu = 1.0 / std::sqrt(nu);
        for (int j = 0; j < 3; ++j) u[j] *= nu;
        C uv(0, 0);
        for (int j = 0; j < 3; ++j) uv += std::conj(u[j]) * v[j];
        for (int j = 0; j < 3; ++j) v[j] -= uv * u[j];
        double nv = 0;
        for (int j = 0; j < 3; ++j) nv += std::norm(v[j]);
        nv = 1.0 / std::sqrt(nv);
        for (int j = 0; j < 3; ++j) v[j] *= nv;
        w[0] = std::conj(u[1] * v[2] - u[2] * v[1]);
        w[1] = std::conj(u[2] * v[0] - u[0] * v[2]);
        w[2] = std::conj(u[0] * v[1] - u[1] * v[0]);
        for (int j = 0; j < 3; ++j) {
            p[j * 2] = (R)u[j].real();        p[j * 2 + 1] = (R)u[j].imag();
            p[(3 + j) * 2] = (R)v[j].real();  p[(3 + j) * 2 + 1] = (R)v[j].imag();
            p[(6 + j) * 2] = (R)w[j].real();  p[(6 + j) * 2 + 1] = (R)w[j].imag();
        }
    }
}

// Coulomb finalisation (reading R22): U_0(x,t) <- G(x,t) U_0(x,t) G(x,t+1)^dag
template <class R>
void coulomb_finalize(R* links, const R* gtot, const Lattice& L) {
    typedef std::complex<R> C;
#pragma omp parallel for collapse(2) schedule(static) if (L.V() >= OMP_MIN_SITES)
    for (int t = 0; t < L.Nt; ++t)
        for (int x = 0; x < L.Nx; ++x)
            for (int y = 0; y < L.Ny; ++y)
                for (int z = 0; z < L.Nz; ++z) {
                    int64_t s = L.site(t, x, y, z);
                    int64_t sf = L.shifted(t, x, y, z, 0, +1);
                    Mat3<R> U = load<R>(link_ptr(links, s, 0));
                    Mat3<R> G = load<R>(gtot + s * 18);
                    Mat3<R> H = load<R>(gtot + sf * 18);
                    Mat3<R> T, O;
                    for (int i = 0; i < 3; ++i)
                        for (int j = 0; j < 3; ++j) {
                            C acc(0, 0);
                            for (int k = 0; k < 3; ++k) acc += G.m[i][k] * U.m[k][j];
                            T.m[i][j] = acc;
                        }
                    for (int i = 0; i < 3; ++i)
                        for (int j = 0; j < 3; ++j) {
                            C acc(0, 0);
                            for (int k = 0; k < 3; ++k) acc += T.m[i][k] * std::conj(H.m[j][k]);
                            O.m[i][j] = acc;
                        }
                    store<R>(link_ptr(links, s, 0), O);
                }
}

inline bool dims_ok(const int* d) {
    for (int k = 0; k < 4; ++k)
        if (d[k] < 2 || (d[k] & 1)) return false;   // odd extents break the colouring (R24)
    return true;
}

template <class R>
int sweep_dispatch(R* links, const int* dims, int parity_mask, int gauge, int algo, double param,
                   uint64_t seed, uint32_t sweep_index, int step1_double, R* gtot) {
    if (!dims_ok(dims) || gauge < 0 || gauge > 2 || algo < 0 || algo > 3) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    for (int p = 0; p < 2; ++p) {   // even first (Alg. 1; reading R7)
        if (!(parity_mask & (1 << p))) continue;
        if (step1_double) half_sweep<R, double>(links, L, p, gauge, algo, param, seed, sweep_index, gtot);
        else half_sweep<R, R>(links, L, p, gauge, algo, param, seed, sweep_index, gtot);
    }
    return 0;
}

}  // namespace

// =====================================================================================
// C interface (ctypes; see oracle/gf_oracle.py).  dims = (Nt, Nx, Ny, Nz).
// parity_mask: bit0 = even half-sweep, bit1 = odd half-sweep (3 = full sweep, even first).
// step1_double: 0 = Step 1 in the storage type, 1 = Step 1 in double (MP).
// =====================================================================================
extern "C" {

int gfo_sweep_d(double* links, const int* dims, int parity_mask, int gauge, int algo, double param,
                uint64_t seed, uint32_t sweep_index, double* gtot) {
    return sweep_dispatch<double>(links, dims, parity_mask, gauge, algo, param, seed, sweep_index, 1, gtot);
}
int gfo_sweep_f(float* links, const int* dims, int parity_mask, int gauge, int algo, double param,
                uint64_t seed, uint32_t sweep_index, int step1_double, float* gtot) {
    return sweep_dispatch<float>(links, dims, parity_mask, gauge, algo, param, seed, sweep_index,
                                 step1_double, gtot);
}

int gfo_measure_d(const double* links, const int* dims, int gauge, double* out3, double* theta_slice,
                  double* F_slice) {
    if (!dims_ok(dims)) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    measure<double>(links, L, gauge, out3, theta_slice, F_slice);
    return 0;
}
int gfo_measure_f(const float* links, const int* dims, int gauge, double* out3, double* theta_slice,
                  double* F_slice) {
    if (!dims_ok(dims)) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    measure<float>(links, L, gauge, out3, theta_slice, F_slice);
    return 0;
}

void gfo_reunitarize_d(double* mats, int64_t n) { reunitarize<double>(mats, n); }
void gfo_reunitarize_f(float* mats, int64_t n) { reunitarize<float>(mats, n); }

int gfo_coulomb_finalize_d(double* links, const double* gtot, const int* dims) {
    if (!dims_ok(dims)) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    coulomb_finalize<double>(links, gtot, L);
    return 0;
}
int gfo_coulomb_finalize_f(float* links, const float* gtot, const int* dims) {
    if (!dims_ok(dims)) return -1;
    Lattice L = {dims[0], dims[1], dims[2], dims[3]};
    coulomb_finalize<float>(links, gtot, L);
    return 0;
}

// One site update on caller-gathered links: up/dn = nd matrices of 18 reals each
// (nd = 4: mu = 0..3; nd = 3: mu = 1..3).  Used for sampled parity at sizes where a whole-lattice
// oracle sweep is too slow, and by the one-site brute-force pins.
void gfo_site_update_d(double* up, double* dn, int nd, int gauge, int algo, double param, uint64_t seed,
                       uint32_t site_index, uint32_t sweep_index, double* gtot) {
    Mat3<double> u[4], d[4], gt;
    for (int m = 0; m < nd; ++m) { u[m] = load<double>(up + m * 18); d[m] = load<double>(dn + m * 18); }
    if (gtot) gt = load<double>(gtot);
    site_update<double, double>(u, d, nd, gauge, algo, param, seed, site_index, sweep_index, gtot ? &gt : nullptr);
    for (int m = 0; m < nd; ++m) { store<double>(up + m * 18, u[m]); store<double>(dn + m * 18, d[m]); }
    if (gtot) store<double>(gtot, gt);
}
void gfo_site_update_f(float* up, float* dn, int nd, int gauge, int algo, double param, uint64_t seed,
                       uint32_t site_index, uint32_t sweep_index, int step1_double, float* gtot) {
    Mat3<float> u[4], d[4], gt;
    for (int m = 0; m < nd; ++m) { u[m] = load<float>(up + m * 18); d[m] = load<float>(dn + m * 18); }
    if (gtot) gt = load<float>(gtot);
    if (step1_double)
        site_update<float, double>(u, d, nd, gauge, algo, param, seed, site_index, sweep_index, gtot ? &gt : nullptr);
    else
        site_update<float, float>(u, d, nd, gauge, algo, param, seed, site_index, sweep_index, gtot ? &gt : nullptr);
    for (int m = 0; m < nd; ++m) { store<float>(up + m * 18, u[m]); store<float>(dn + m * 18, d[m]); }
    if (gtot) store<float>(gtot, gt);
}

// ---- pieces of Step 1 exposed for the pins ----
void gfo_philox4x32_10(const uint32_t* ctr4, const uint32_t* key2, uint32_t* out4) {
    Philox4 r = philox4x32_10(ctr4[0], ctr4[1], ctr4[2], ctr4[3], key2[0], key2[1]);
    for (int k = 0; k < 4; ++k) out4[k] = r.v[k];
}
void gfo_draw(uint64_t seed, uint32_t site, uint32_t sweep, int sub, int purpose, uint32_t trial,
              uint32_t* out4, double* uni4) {
    Philox4 r = draw(seed, site, sweep, sub, purpose, trial);
    for (int k = 0; k < 4; ++k) { out4[k] = r.v[k]; uni4[k] = u01(r.v[k]); }
}
// quaternion of the neighbourhood for subgroup (i,j): Landau form; up/dn as in gfo_site_update
void gfo_local_quaternion_d(const double* up, const double* dn, int nd, int i, int j, double* a4) {
    double a[4] = {0, 0, 0, 0};
    for (int m = 0; m < nd; ++m) {
        Mat3<double> U = load<double>(up + m * 18), W = load<double>(dn + m * 18);
        add_quaternion<double, double>(a, U, i, j);
        add_quaternion_dagger<double, double>(a, W, i, j);
    }
    for (int k = 0; k < 4; ++k) a4[k] = a[k];
}
// D, E, F of the MAG quadratic form for subgroup (i,j)
void gfo_local_mag_def_d(const double* up, const double* dn, int nd, int i, int j, double* def3) {
    double a = 0, b = 0, E = 0, F = 0;
    for (int m = 0; m < nd; ++m) {
        Mat3<double> U = load<double>(up + m * 18), W = load<double>(dn + m * 18);
        add_mag_up<double, double>(a, b, E, F, U, i, j);
        add_mag_down<double, double>(a, b, E, F, W, i, j);
    }
    def3[0] = (a - b) / 2; def3[1] = E; def3[2] = F;
}
void gfo_rule_or_d(const double* a4, double omega, double* g4) { rule_or<double>(a4, omega, g4); }
void gfo_rule_micro_d(const double* a4, double* g4) { rule_micro<double>(a4, g4); }
void gfo_rule_heatbath_landau(const double* a4, double T, uint64_t seed, uint32_t site, uint32_t sweep,
                              int sub, double* g4) {
    rule_heatbath_landau(a4, T, seed, site, sweep, sub, g4);
}
void gfo_rule_heatbath_mag(double D, double E, double F, double T, uint64_t seed, uint32_t site,
                           uint32_t sweep, int sub, double* g4) {
    rule_heatbath_mag(D, E, F, T, seed, site, sweep, sub, g4);
}
// apply the embedded subgroup element: which = 0 left (g U), 1 right-dagger (U g^dag)
void gfo_apply_subgroup_d(double* mat18, const double* g4, int i, int j, int which) {
    Mat3<double> U = load<double>(mat18);
    if (which == 0) left_mul_subgroup<double>(U, g4, i, j);
    else right_mul_subgroup_dagger<double>(U, g4, i, j);
    store<double>(mat18, U);
}

// Random start on the gauge orbit (reading R27; how the paper drew its starts is not stated:
// the Haar law is pinned by its moments, the Philox keying is "parity unpinned"): h(x) Haar on SU(3) from two rows of
// complex standard normals, Box-Muller on the Philox uniforms of counter (site, 0, k | 3<<8, 0), k=0..2:
// normals 4k..4k+3 = sqrt(-2 ln u0)(cos, sin)(2 pi u1), sqrt(-2 ln u2)(cos, sin)(2 pi u3); then the
// Gram-Schmidt reprojection above.  h: [V][3][3][2] doubles in site order.
void gfo_haar_field_d(double* h, const int* dims, uint64_t seed) {
    const int64_t V = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
    const double two_pi = 6.283185307179586477;
    for (int64_t s = 0; s < V; ++s) {
        double* p = h + s * 18;
        for (int k = 0; k < 3; ++k) {
            Philox4 w = draw(seed, (uint32_t)s, 0u, k, 3, 0u);
            const double r0 = std::sqrt(-2.0 * std::log(u01(w.v[0]))), r1 = std::sqrt(-2.0 * std::log(u01(w.v[2])));
            p[4 * k] = r0 * std::cos(two_pi * u01(w.v[1]));
            p[4 * k + 1] = r0 * std::sin(two_pi * u01(w.v[1]));
            p[4 * k + 2] = r1 * std::cos(two_pi * u01(w.v[3]));
            p[4 * k + 3] = r1 * std::sin(two_pi * u01(w.v[3]));
        }
        for (int k = 12; k < 18; ++k) p[k] = 0.0;
    }
    reunitarize<double>(h, V);
}

int gfo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"

// the N_c = 2 oracle uses the generator, rules and indexer defined above
#include "gf_oracle_su2.hpp"

// the input generator's oracle: Wilson-action heatbath, plaquette
#include "gf_oracle_wilson.hpp"
