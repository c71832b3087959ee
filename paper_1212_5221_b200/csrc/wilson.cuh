// wilson.cuh — input generator: thermalised SU(3) configurations of the Wilson
// gauge action, standing in for the paper's beta = 5.7 ensemble, and the plaquette.
//
// Cabibbo-Marinari pseudo-heatbath (the SU(2)-subgroup method of the paper's ref. [31]): for a link U_mu(x)
// with staple sum A the weight is exp((beta/3) Re tr[U A]); for the subgroups (0,1),(0,2),(1,2) in turn,
// W = U A, a = un-normalised quaternion of W's sub-block (Fig. A.10), g drawn by the Landau heatbath rule
// (step1.cuh) at temperature T = 3/beta, U <- g~ U (and W <- g~ W).  One launch updates the links of one
// direction mu on the sites of one parity (they share no plaquette); one thread per link; Philox counter
// (site, 4*sweep_index + mu, sub | purpose << 8, trial), key seed + copy.  Scalar heatbath math in double.
#pragma once
#include "aux_kernels.cuh"
#include "step1.cuh"
#include "su2.cuh"

namespace gf {

// out = T^dagger M
template <class T>
GF_DEV void mul_dagger_left(const Mat<T>& Tm, const Mat<T>& M, Mat<T>& out) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T re = T(0), im = T(0);
#pragma unroll
            for (int k = 0; k < 3; ++k) {   // conj(T_ki) M_kj
                re = fma_t(Tm.v[RE(k, i)], M.v[RE(k, j)], re);
                re = fma_t(Tm.v[IM(k, i)], M.v[IM(k, j)], re);
                im = fma_t(Tm.v[RE(k, i)], M.v[IM(k, j)], im);
                im = fma_t(-Tm.v[IM(k, i)], M.v[RE(k, j)], im);
            }
            out.v[RE(i, j)] = re;
            out.v[IM(i, j)] = im;
        }
}

struct SiteCoord {
    int c[4];   // t, x, y, z
};
// checkerboard index of the site displaced by (d_mu along mu, d_nu along nu), periodic
GF_DEV int64_t cb_shift(const Dims& d, const SiteCoord& s, int mu, int dmu, int nu, int dnu) {
    int c[4] = {s.c[0], s.c[1], s.c[2], s.c[3]};
    const int n[4] = {d.Nt, d.Nx, d.Ny, d.Nz};
    c[mu] += dmu; if (c[mu] >= n[mu]) c[mu] -= n[mu]; if (c[mu] < 0) c[mu] += n[mu];
    c[nu] += dnu; if (c[nu] >= n[nu]) c[nu] -= n[nu]; if (c[nu] < 0) c[nu] += n[nu];
    return ((((int64_t)c[0] * d.Nx + c[1]) * d.Ny + c[2]) * d.Nz + c[3]) >> 1;
}

// the heatbath runs in the storage type, as in the half-sweep kernel (step1.cuh: float with guard-banded decisions on
// SP contexts, double on DP contexts)
template <int I, int J, int S, class R>
GF_DEV void wilson_subgroup(Mat<R>& W, Mat<R>& U, double T, uint64_t seed, uint32_t site, uint32_t sweep,
                            const HbDraw<R>& pre) {
    R a[4], g[4];
    a[0] = W.v[RE(I, I)] + W.v[RE(J, J)];
    a[3] = W.v[IM(I, I)] - W.v[IM(J, J)];
    a[2] = W.v[RE(I, J)] - W.v[RE(J, I)];
    a[1] = W.v[IM(I, J)] + W.v[IM(J, I)];
    hb_finish_landau<R>(a, (R)T, pre, seed, site, sweep, S, g);
    sub_left<I, J>(W, g);
    sub_left<I, J>(U, g);
}

// grid = (ceil(Vsh / block), ncopies * Nt); links U_mu(x) for x of parity `parity`
#ifndef GF_HB_MIN_CTAS
#define GF_HB_MIN_CTAS 2
#endif
template <class R, int RECON>
__global__ void __launch_bounds__(128, GF_HB_MIN_CTAS) wilson_heatbath_kernel(char* links_all, Dims d, int mu, int parity, double beta,
                                                              uint64_t seed0, uint32_t sweep_index, int64_t copy_bytes) {
    typedef Layout<R, RECON> L;
    const int Nzh = d.Nz >> 1;
    const int Vsh = d.Nx * d.Ny * Nzh;
    const int64_t Vh = (int64_t)d.Nt * Vsh;
    // threads past the end of the slice redo the last site without storing: the heatbath's retries are evaluated by
    // whole warps (step1.cuh, hb_retry)
    const int i_raw = blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = i_raw < Vsh;
    const int i = active ? i_raw : Vsh - 1;
    const int copy = blockIdx.y / d.Nt;
    const int t = blockIdx.y - copy * d.Nt;
    char* links = links_all + copy * copy_bytes;
    int rem = i;
    const int zh = rem % Nzh; rem /= Nzh;
    const int y = rem % d.Ny;
    const int x = rem / d.Ny;
    const int r = (t + x + y + parity) & 1;
    SiteCoord s;
    s.c[0] = t; s.c[1] = x; s.c[2] = y; s.c[3] = 2 * zh + r;
    const int64_t cb = (int64_t)t * Vsh + i;
    const uint32_t site = (uint32_t)(((t * d.Nx + x) * d.Ny + y) * d.Nz + s.c[3]);
    const int q = 1 - parity;   // parity of the sites one step away

    const double T = 3.0 / beta;
    const uint64_t seed = seed0 + (uint64_t)copy;
    const uint32_t sw = 4u * sweep_index + (uint32_t)mu;
    Mat<R> U, A;
    global_get<R, RECON>(links + L::link_offset(parity, mu, Vh), Vh, cb, U);
    // the link-independent part of the three heatbath draws (step1.cuh) while the first loads are in flight
    HbDraw<R> pre[3];
#pragma unroll 1
    for (int k = 0; k < 3; ++k) hb_draws_landau<R>(seed, site, sw, k, pre[k]);
    set_zero(A);
    const int64_t cb_mu = cb_shift(d, s, mu, +1, mu, 0);
#pragma unroll 1
    for (int nu = 0; nu < 4; ++nu) {
        if (nu == mu) continue;
        Mat<R> a, b, c, T1, T2;
        // upper staple: U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
        global_get<R, RECON>(links + L::link_offset(q, nu, Vh), Vh, cb_mu, a);
        global_get<R, RECON>(links + L::link_offset(q, mu, Vh), Vh, cb_shift(d, s, nu, +1, nu, 0), b);
        global_get<R, RECON>(links + L::link_offset(parity, nu, Vh), Vh, cb, c);
        mul_right_dagger<3>(a, b, T1);
        mul_right_dagger<3>(T1, c, T2);
#pragma unroll
        for (int k = 0; k < 18; ++k) A.v[k] += T2.v[k];
        // lower staple: U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu) = [U_mu(x-nu) U_nu(x+mu-nu)]^dag U_nu(x-nu)
        const int64_t cb_mnu = cb_shift(d, s, nu, -1, nu, 0);
        global_get<R, RECON>(links + L::link_offset(parity, nu, Vh), Vh, cb_shift(d, s, mu, +1, nu, -1), a);
        global_get<R, RECON>(links + L::link_offset(q, mu, Vh), Vh, cb_mnu, b);
        global_get<R, RECON>(links + L::link_offset(q, nu, Vh), Vh, cb_mnu, c);
        mul_left<3>(b, a, T1);
        mul_dagger_left(T1, c, T2);
#pragma unroll
        for (int k = 0; k < 18; ++k) A.v[k] += T2.v[k];
    }
    Mat<R> W;
    mul_left<3>(U, A, W);
    wilson_subgroup<0, 1, 0>(W, U, T, seed, site, sw, pre[0]);
    wilson_subgroup<0, 2, 1>(W, U, T, seed, site, sw, pre[1]);
    wilson_subgroup<1, 2, 2>(W, U, T, seed, site, sw, pre[2]);
    if (active) global_put<R, RECON>(links + L::link_offset(parity, mu, Vh), Vh, cb, U);
}

// sum over the 6 plaquettes at x of Re tr U_P: grid (ceil(Vsh/block), ncopies*Nt, 2) like measure_kernel;
// partial[...][0] = sum, [1] = 0
template <class R, int RECON>
// t-shards: U_nu(x + t_hat) of the last slice is the first slice of the link store above (links_up, Vh_up sites per
// parity; shards hold one copy); not sharded: the store itself (periodic wrap)
__global__ void plaquette_kernel(const char* links, Dims d, double* partial, int64_t copy_bytes, const char* links_up,
                                 int64_t Vh_up) {
    typedef Layout<R, RECON> L;
    const int Nzh = d.Nz >> 1;
    const int Vsh = d.Nx * d.Ny * Nzh;
    const int64_t Vh = (int64_t)d.Nt * Vsh;
    const int copy = blockIdx.y / d.Nt;
    const int t = blockIdx.y - copy * d.Nt, par = blockIdx.z;
    links += copy * copy_bytes;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double acc = 0.0, zero = 0.0;
    if (i < Vsh) {
        int rem = i;
        const int zh = rem % Nzh; rem /= Nzh;
        const int y = rem % d.Ny;
        const int x = rem / d.Ny;
        SiteCoord s;
        s.c[0] = t; s.c[1] = x; s.c[2] = y; s.c[3] = 2 * zh + ((t + x + y + par) & 1);
        const int64_t cb = (int64_t)t * Vsh + i;
#pragma unroll 1
        for (int mu = 0; mu < 4; ++mu)
#pragma unroll 1
            for (int nu = mu + 1; nu < 4; ++nu) {
                Mat<R> a, b, T1, T2;
                global_get<R, RECON>(links + L::link_offset(par, mu, Vh), Vh, cb, a);
                if (mu == 0 && t == d.Nt - 1)     // same (x, y, z) in slice 0 of the store above: in-slice index i
                    global_get<R, RECON>(links_up + copy * copy_bytes + L::link_offset(1 - par, nu, Vh_up), Vh_up, (int64_t)i, b);
                else
                    global_get<R, RECON>(links + L::link_offset(1 - par, nu, Vh), Vh, cb_shift(d, s, mu, +1, mu, 0), b);
                mul_left<3>(a, b, T1);                                   // U_mu(x) U_nu(x+mu)
                global_get<R, RECON>(links + L::link_offset(1 - par, mu, Vh), Vh, cb_shift(d, s, nu, +1, nu, 0), a);
                mul_right_dagger<3>(T1, a, T2);                          // ... U_mu(x+nu)^dag
                global_get<R, RECON>(links + L::link_offset(par, nu, Vh), Vh, cb, b);
                // Re tr[T2 b^dag] = sum_ij Re(T2_ij conj(b_ij))
#pragma unroll
                for (int k = 0; k < 18; ++k) acc += (double)T2.v[k] * (double)b.v[k];
            }
    }
    block_sum2(acc, zero);
    if (threadIdx.x == 0) {
        const int64_t bidx = ((int64_t)(blockIdx.y * 2 + par)) * gridDim.x + blockIdx.x;
        partial[2 * bidx] = acc;
        partial[2 * bidx + 1] = 0.0;
    }
}

// ---- the same for the gauge group SU(2) (links as quaternions, su2.cuh): weight exp((beta/2) Re tr[U A]) ----
template <class R>
__global__ void __launch_bounds__(128) wilson_heatbath2_kernel(char* links_all, Dims d, int mu, int parity, double beta,
                                                               uint64_t seed0, uint32_t sweep_index, int64_t copy_bytes) {
    typedef Layout<R, 4> L;
    const int Nzh = d.Nz >> 1;
    const int Vsh = d.Nx * d.Ny * Nzh;
    const int64_t Vh = (int64_t)d.Nt * Vsh;
    const int i_raw = blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = i_raw < Vsh;     // whole warps stay (hb_retry)
    const int i = active ? i_raw : Vsh - 1;
    const int copy = blockIdx.y / d.Nt;
    const int t = blockIdx.y - copy * d.Nt;
    char* links = links_all + copy * copy_bytes;
    int rem = i;
    const int zh = rem % Nzh; rem /= Nzh;
    const int y = rem % d.Ny;
    const int x = rem / d.Ny;
    SiteCoord s;
    s.c[0] = t; s.c[1] = x; s.c[2] = y; s.c[3] = 2 * zh + ((t + x + y + parity) & 1);
    const int64_t cb = (int64_t)t * Vsh + i;
    const uint32_t site = (uint32_t)(((t * d.Nx + x) * d.Ny + y) * d.Nz + s.c[3]);
    const int q = 1 - parity;
    Quat<R> U, a, b, c;
    global_get_q(links + L::link_offset(parity, mu, Vh), Vh, cb, U);
    HbDraw<R> pre;   // the link-independent part of the heatbath draw while the loads are in flight
    hb_draws_landau<R>(seed0 + (uint64_t)copy, site, 4u * sweep_index + (uint32_t)mu, 0, pre);
    R A[4] = {R(0), R(0), R(0), R(0)};
    const int64_t cb_mu = cb_shift(d, s, mu, +1, mu, 0);
#pragma unroll 1
    for (int nu = 0; nu < 4; ++nu) {
        if (nu == mu) continue;
        global_get_q(links + L::link_offset(q, nu, Vh), Vh, cb_mu, a);
        global_get_q(links + L::link_offset(q, mu, Vh), Vh, cb_shift(d, s, nu, +1, nu, 0), b);
        global_get_q(links + L::link_offset(parity, nu, Vh), Vh, cb, c);
        Quat<R> st = qmul_dagger(qmul_dagger(a, b), c);              // U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
#pragma unroll
        for (int k = 0; k < 4; ++k) A[k] += st.v[k];
        const int64_t cb_mnu = cb_shift(d, s, nu, -1, nu, 0);
        global_get_q(links + L::link_offset(parity, nu, Vh), Vh, cb_shift(d, s, mu, +1, nu, -1), a);
        global_get_q(links + L::link_offset(q, mu, Vh), Vh, cb_mnu, b);
        global_get_q(links + L::link_offset(q, nu, Vh), Vh, cb_mnu, c);
        st = qmul(qconj(qmul(b, a)), c);                             // [U_mu(x-nu) U_nu(x+mu-nu)]^dag U_nu(x-nu)
#pragma unroll
        for (int k = 0; k < 4; ++k) A[k] += st.v[k];
    }
    Quat<R> Aq;
#pragma unroll
    for (int k = 0; k < 4; ++k) Aq.v[k] = A[k];
    const Quat<R> W = qmul(U, Aq);                                   // the product is bilinear: A need not be unit
    const R aw[4] = {R(2) * W.v[0], R(2) * W.v[1], R(2) * W.v[2], R(2) * W.v[3]};
    Quat<R> g;
    hb_finish_landau<R>(aw, (R)(2.0 / beta), pre, seed0 + (uint64_t)copy, site, 4u * sweep_index + (uint32_t)mu, 0, g.v);
    if (active) global_put_q(links + L::link_offset(parity, mu, Vh), Vh, cb, qmul(g, U));
}

template <class R>
__global__ void plaquette2_kernel(const char* links, Dims d, double* partial, int64_t copy_bytes) {
    typedef Layout<R, 4> L;
    const int Nzh = d.Nz >> 1;
    const int Vsh = d.Nx * d.Ny * Nzh;
    const int64_t Vh = (int64_t)d.Nt * Vsh;
    const int copy = blockIdx.y / d.Nt;
    const int t = blockIdx.y - copy * d.Nt, par = blockIdx.z;
    links += copy * copy_bytes;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double acc = 0.0, zero = 0.0;
    if (i < Vsh) {
        int rem = i;
        const int zh = rem % Nzh; rem /= Nzh;
        const int y = rem % d.Ny;
        const int x = rem / d.Ny;
        SiteCoord s;
        s.c[0] = t; s.c[1] = x; s.c[2] = y; s.c[3] = 2 * zh + ((t + x + y + par) & 1);
        const int64_t cb = (int64_t)t * Vsh + i;
#pragma unroll 1
        for (int mu = 0; mu < 4; ++mu)
#pragma unroll 1
            for (int nu = mu + 1; nu < 4; ++nu) {
                Quat<R> a, b, c, e;
                global_get_q(links + L::link_offset(par, mu, Vh), Vh, cb, a);
                global_get_q(links + L::link_offset(1 - par, nu, Vh), Vh, cb_shift(d, s, mu, +1, mu, 0), b);
                global_get_q(links + L::link_offset(1 - par, mu, Vh), Vh, cb_shift(d, s, nu, +1, nu, 0), c);
                global_get_q(links + L::link_offset(par, nu, Vh), Vh, cb, e);
                const Quat<R> P = qmul_dagger(qmul_dagger(qmul(a, b), c), e);
                acc += 2.0 * (double)P.v[0];                        // Re tr of the SU(2) matrix
            }
    }
    block_sum2(acc, zero);
    if (threadIdx.x == 0) {
        const int64_t bidx = ((int64_t)(blockIdx.y * 2 + par)) * gridDim.x + blockIdx.x;
        partial[2 * bidx] = acc;
        partial[2 * bidx + 1] = 0.0;
    }
}

}  // namespace gf
