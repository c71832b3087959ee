// aux_kernels.cuh — everything on the path that is not the half-sweep itself:
//   layout conversion StandardPattern <-> device store (gf_set_links / gf_get_links),
//   F / theta reductions, reunitarisation (a10),
//   Coulomb finalisation of the temporal links (a12).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "layout.cuh"
#include "su3.cuh"
#include "sweep.cuh"

namespace gf {

struct Dims {
    int Nt, Nx, Ny, Nz;
};
GF_DEV int64_t Vh_of(const Dims& d) { return (int64_t)d.Nt * d.Nx * d.Ny * d.Nz / 2; }

// lexicographic site index s = ((t*Nx + x)*Ny + y)*Nz + z  ->  parity, checkerboard index
GF_DEV void site_to_cb(const Dims& d, int64_t s, int& par, int& cb) {
    int64_t rem = s;
    const int z = (int)(rem % d.Nz); rem /= d.Nz;
    const int y = (int)(rem % d.Ny); rem /= d.Ny;
    const int x = (int)(rem % d.Nx);
    const int t = (int)(rem / d.Nx);
    par = (t + x + y + z) & 1;
    cb = (int)(s >> 1);
}

// ---- StandardPattern (AoS, element type E) -> device store (R, RECON) ------------------------
// one thread per link (site, mu); src points at the first link of site `site0`
template <class E, class R, int RECON>
__global__ void convert_in_kernel(const E* __restrict__ src, char* links, Dims d, int64_t site0, int64_t nsites) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nsites * 4) return;
    const int64_t s = site0 + (i >> 2);
    const int mu = (int)(i & 3);
    const int64_t Vh = (int64_t)d.Nt * d.Nx * d.Ny * d.Nz / 2;
    int par, cb;
    site_to_cb(d, s, par, cb);
    Mat<R> m;
    const E* p = src + i * 18;
#pragma unroll
    for (int k = 0; k < 18; ++k) m.v[k] = (R)p[k];
    global_put<R, RECON>(links + Layout<R, RECON>::link_offset(par, mu, Vh), Vh, cb, m);
}
template <class E, class R, int RECON>
__global__ void convert_out_kernel(E* __restrict__ dst, const char* links, Dims d, int64_t site0, int64_t nsites) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nsites * 4) return;
    const int64_t s = site0 + (i >> 2);
    const int mu = (int)(i & 3);
    const int64_t Vh = (int64_t)d.Nt * d.Nx * d.Ny * d.Nz / 2;
    int par, cb;
    site_to_cb(d, s, par, cb);
    Mat<R> m;
    global_get<R, RECON>(links + Layout<R, RECON>::link_offset(par, mu, Vh), Vh, cb, m);
    E* p = dst + i * 18;
#pragma unroll
    for (int k = 0; k < 18; ++k) p[k] = (E)m.v[k];
}
// one-matrix-per-site field (tracked transform), always 18 reals
template <class E, class R>
__global__ void field_out_kernel(E* __restrict__ dst, const char* field, Dims d, int64_t site0, int64_t nsites) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nsites) return;
    const int64_t s = site0 + i;
    const int64_t Vh = (int64_t)d.Nt * d.Nx * d.Ny * d.Nz / 2;
    int par, cb;
    site_to_cb(d, s, par, cb);
    Mat<R> m;
    global_get<R, 18>(field + Layout<R, 18>::site_offset(par, Vh), Vh, cb, m);
    E* p = dst + i * 18;
#pragma unroll
    for (int k = 0; k < 18; ++k) p[k] = (E)m.v[k];
}
template <class R>
__global__ void field_identity_kernel(char* field, int64_t Vh) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * Vh) return;
    const int par = (int)(i / Vh);
    const int cb = (int)(i % Vh);
    Mat<R> m;
    set_identity(m);
    global_put<R, 18>(field + Layout<R, 18>::site_offset(par, Vh), Vh, cb, m);
}

// ---- reunitarisation: Gram-Schmidt on rows 0,1 in double, row 2 = (u x v)^* ------------------
GF_DEV void gram_schmidt(Mat<double>& m) {
    double nu = 0.0;
#pragma unroll
    for (int j = 0; j < 3; ++j) nu += m.v[RE(0, j)] * m.v[RE(0, j)] + m.v[IM(0, j)] * m.v[IM(0, j)];
    nu = 1.0 / sqrt(nu);
#pragma unroll
    for (int j = 0; j < 3; ++j) { m.v[RE(0, j)] *= nu; m.v[IM(0, j)] *= nu; }
    double pr = 0.0, pi = 0.0;   // u^dagger v
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        pr += m.v[RE(0, j)] * m.v[RE(1, j)] + m.v[IM(0, j)] * m.v[IM(1, j)];
        pi += m.v[RE(0, j)] * m.v[IM(1, j)] - m.v[IM(0, j)] * m.v[RE(1, j)];
    }
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const double ur = m.v[RE(0, j)], ui = m.v[IM(0, j)];
        m.v[RE(1, j)] -= pr * ur - pi * ui;
        m.v[IM(1, j)] -= pr * ui + pi * ur;
    }
    double nv = 0.0;
#pragma unroll
    for (int j = 0; j < 3; ++j) nv += m.v[RE(1, j)] * m.v[RE(1, j)] + m.v[IM(1, j)] * m.v[IM(1, j)];
    nv = 1.0 / sqrt(nv);
#pragma unroll
    for (int j = 0; j < 3; ++j) { m.v[RE(1, j)] *= nv; m.v[IM(1, j)] *= nv; }
    reconstruct_row2(m);
}

// nmats matrices stored as planes [slot][chunk][cb] with `slot_bytes` = RECON*sizeof(R)*Vh between slots
// blockIdx.y = gauge copy, copy_bytes apart
template <class R, int RECON>
__global__ void reunit_kernel(char* base, int64_t Vh, int nslots, int64_t copy_bytes) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (int64_t)nslots * Vh) return;
    base += blockIdx.y * copy_bytes;
    const int slot = (int)(i / Vh);
    const int cb = (int)(i % Vh);
    char* p0 = base + (int64_t)slot * Layout<R, RECON>::LINK_BYTES * Vh;
    Mat<R> m;
    global_get<R, RECON>(p0, Vh, cb, m);   // RECON=12: row 2 rebuilt here, overwritten below
    Mat<double> w;
#pragma unroll
    for (int k = 0; k < 18; ++k) w.v[k] = (double)m.v[k];
    gram_schmidt(w);
#pragma unroll
    for (int k = 0; k < 18; ++k) m.v[k] = (R)w.v[k];
    global_put<R, RECON>(p0, Vh, cb, m);
}

// ---- F and theta ---------------------------------------------------------------------------
// grid = (2 * ceil(Vsh / block), ncopies*Nt): one thread per site of parity blockIdx.x & 1 in (gauge copy,
// time-slice) blockIdx.y.  Each block writes one (F-term, theta-term) pair; slice_reduce_kernel sums them in a
// fixed order, so results are bit-reproducible.  All arithmetic in double (BASELINE.json).
GF_DEV double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}
GF_DEV void block_sum2(double& a, double& b) {
    __shared__ double sa[32], sb[32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    a = warp_sum(a);
    b = warp_sum(b);
    if (lane == 0) { sa[w] = a; sb[w] = b; }
    __syncthreads();
    if (w == 0) {
        a = lane < nw ? sa[lane] : 0.0;
        b = lane < nw ? sb[lane] : 0.0;
        a = warp_sum(a);
        b = warp_sum(b);
    }
}

// t-shards: sh.links_dn is the store that holds the slice below this store's first one (its last
// slice, Nt_dn - 1); not sharded: the store itself (periodic wrap).
struct ShardDn {
    const char* links_dn;
    int64_t Vh_dn, copy_bytes_dn;
    int Nt_dn;
};

template <class R, int RECON, int GAUGE>
__global__ void measure_kernel(const char* links, Dims d, double* partial, int64_t copy_bytes, ShardDn sh, int mag_eq16) {
    typedef Layout<R, RECON> L;
    constexpr int MU0 = (GAUGE == GAUGE_COULOMB) ? 1 : 0;
    const int Nzh = d.Nz >> 1;
    const int Vsh = d.Nx * d.Ny * Nzh;
    const int64_t Vh = (int64_t)d.Nt * Vsh;
    const int copy = blockIdx.y / d.Nt;
    // both parities of a tile in neighbouring CTAs (blockIdx.x = 2 tile + parity): a link is read once as the up link
    // of its origin and once as the down link of its end point, and the second read then is an L2 hit unless the two
    // sites are a whole time-slice apart
    const int t = blockIdx.y - copy * d.Nt, par = (int)(blockIdx.x & 1u);
    const int bx = (int)(blockIdx.x >> 1), gx = (int)(gridDim.x >> 1);
    links += copy * copy_bytes;
    const int i = bx * blockDim.x + threadIdx.x;
    double f_term = 0.0, th_term = 0.0;
    if (i < Vsh) {
        const int cb = t * Vsh + i;
        int rem = i;
        const int zh = rem % Nzh; rem /= Nzh;
        const int y = rem % d.Ny;
        const int x = rem / d.Ny;
        const int r = (t + x + y + par) & 1;
        const int sy = Nzh, sx = Nzh * d.Ny, st = Vsh;
        int cbn[4];
        cbn[0] = cb + (t ? -st : (d.Nt - 1) * st);
        cbn[1] = cb + (x ? -sx : (d.Nx - 1) * sx);
        cbn[2] = cb + (y ? -sy : (d.Ny - 1) * sy);
        cbn[3] = r ? cb : (zh ? cb - 1 : cb + Nzh - 1);
        Mat<double> K;
        Herm<double> M[3];
        if (GAUGE == GAUGE_MAG) { set_zero(M[0]); set_zero(M[1]); set_zero(M[2]); }
        else set_zero(K);
#pragma unroll
        for (int mu = MU0; mu < 4; ++mu) {
            Mat<R> U;
            global_get<R, RECON>(links + L::link_offset(par, mu, Vh), Vh, cb, U);
            if (GAUGE == GAUGE_MAG) {
#pragma unroll
                for (int k = 0; k < 3; ++k)
                    f_term += (double)U.v[RE(k, k)] * (double)U.v[RE(k, k)] + (double)U.v[IM(k, k)] * (double)U.v[IM(k, k)];
                mag_acc_up<0>(M[0], U); mag_acc_up<1>(M[1], U); mag_acc_up<2>(M[2], U);
            } else {
                f_term += (double)U.v[RE(0, 0)] + (double)U.v[RE(1, 1)] + (double)U.v[RE(2, 2)];
                acc_plain(K, U);
            }
            if (mu == 0 && t == 0)   // x - t_hat of the first slice: last slice of the store below
                global_get<R, RECON>(sh.links_dn + copy * sh.copy_bytes_dn + L::link_offset(1 - par, 0, sh.Vh_dn), sh.Vh_dn,
                                     (int64_t)(sh.Nt_dn - 1) * Vsh + i, U);
            else
                global_get<R, RECON>(links + L::link_offset(1 - par, mu, Vh), Vh, cbn[mu], U);
            if (GAUGE == GAUGE_MAG) { mag_acc_down<0>(M[0], U); mag_acc_down<1>(M[1], U); mag_acc_down<2>(M[2], U); }
            else acc_dagger(K, U);
        }
        if (GAUGE == GAUGE_MAG) {
            // theta: sum over the three subgroups of |X^s_12|^2 = E_s^2 + F_s^2 (R11)
            // mag_eq16: Eq. (16) as printed, |X_12 + Y_12 + Z_12|^2 with the sum over the subgroups
            // INSIDE the modulus: not a norm (it can vanish away from a maximum), reported for comparison with the paper
            const int SI[3] = {0, 0, 1}, SJ[3] = {1, 2, 2};
            double Es = 0.0, Fs = 0.0;
#pragma unroll
            for (int s = 0; s < 3; ++s) {
                const double E = M[SI[s]].o[2 * s + 1] - M[SJ[s]].o[2 * s + 1];
                const double F = M[SI[s]].o[2 * s] - M[SJ[s]].o[2 * s];
                th_term += E * E + F * F;
                Es += E; Fs += F;
            }
            if (mag_eq16) th_term = Es * Es + Fs * Fs;
        } else {
            // Delta = traceless[(K - K^dag)/2i] (Eqs. (6)); tr[Delta Delta^dag] (Eq. (7))
            double sum = 0.0, tr = 0.0;
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = 0; b < 3; ++b) {
                    const double xr = K.v[RE(a, b)] - K.v[RE(b, a)];
                    const double xi = K.v[IM(a, b)] + K.v[IM(b, a)];
                    sum += 0.25 * (xr * xr + xi * xi);
                    if (a == b) tr += 0.5 * xi;   // (X/2i)_aa = Im-part
                }
            th_term = fmax(0.0, sum - tr * tr / 3.0);
        }
    }
    block_sum2(f_term, th_term);
    if (threadIdx.x == 0) {
        const int64_t b = ((int64_t)(blockIdx.y * 2 + par)) * gx + bx;
        partial[2 * b] = f_term;
        partial[2 * b + 1] = th_term;
    }
}

// one block per (copy, time-slice) (Nt here = ncopies*Nt): out[t] = sum of F terms, out[Nt + t] = sum of theta terms
__global__ void slice_reduce_kernel(const double* partial, int blocks_per_slice, int Nt, double* out) {
    const int t = blockIdx.x;
    double a = 0.0, b = 0.0;
    for (int k = threadIdx.x; k < blocks_per_slice; k += blockDim.x) {
        a += partial[2 * ((int64_t)t * blocks_per_slice + k)];
        b += partial[2 * ((int64_t)t * blocks_per_slice + k) + 1];
    }
    block_sum2(a, b);
    if (threadIdx.x == 0) { out[t] = a; out[Nt + t] = b; }
}

// fused-reduction partials of the half-sweep kernels: partial[t][gx][3] -> out[t][3], one block per
// time-slice, fixed summation order (bit-reproducible)
__global__ void red_reduce_kernel(const double* partial, int gx, double* out) {
    const int t = blockIdx.x;
    double a = 0.0, b = 0.0, c = 0.0;
    for (int k = threadIdx.x; k < gx; k += blockDim.x) {
        const double* p = partial + ((size_t)t * gx + k) * 3;
        a += p[0]; b += p[1]; c += p[2];
    }
    block_sum2(a, b);
    __syncthreads();
    double dummy = 0.0;
    block_sum2(c, dummy);
    if (threadIdx.x == 0) { out[3 * t] = a; out[3 * t + 1] = b; out[3 * t + 2] = c; }
}

// ---- Coulomb finalisation: U_0(x) <- R(x) U_0(x) R(x+t)^dag, R = g_tot g_applied^dag -----------
// t-shards: g(x + t_hat) of the last slice is the first slice of the transform store above (gtot_up / gapp_up with
// Vh_up sites per parity); not sharded: the store itself (periodic wrap).
struct ShardUp {
    const char* gtot_up;
    const char* gapp_up;
    int64_t Vh_up, copy_bytes_up;
};

template <class R, int RECON>
__global__ void coulomb_finalize_kernel(char* links, const char* gtot, const char* gapp, Dims d,
                                        int64_t copy_links_bytes, int64_t copy_field_bytes, ShardUp sh) {
    links += blockIdx.y * copy_links_bytes;   // blockIdx.y = gauge copy
    gtot += blockIdx.y * copy_field_bytes;
    if (gapp) gapp += blockIdx.y * copy_field_bytes;
    const int Nzh = d.Nz >> 1;
    const int Vsh = d.Nx * d.Ny * Nzh;
    const int64_t Vh = (int64_t)d.Nt * Vsh;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * Vh) return;
    const int par = (int)(i / Vh);
    const int cb = (int)(i % Vh);
    const int t = cb / Vsh;
    const bool top = t == d.Nt - 1;
    const int64_t cbf = top ? cb - (int64_t)(d.Nt - 1) * Vsh : cb + Vsh;   // x + t_hat, other parity (top: slice 0 above)
    const char* gt_f = top ? sh.gtot_up + blockIdx.y * sh.copy_bytes_up : gtot;
    const char* ga_f = top ? (sh.gapp_up ? sh.gapp_up + blockIdx.y * sh.copy_bytes_up : nullptr) : gapp;
    const int64_t Vh_f = top ? sh.Vh_up : Vh;
    Mat<R> U, Ga, Gb, T, O;
    global_get<R, 18>(gtot + Layout<R, 18>::site_offset(par, Vh), Vh, cb, Ga);
    global_get<R, 18>(gt_f + Layout<R, 18>::site_offset(1 - par, Vh_f), Vh_f, cbf, Gb);
    if (gapp) {
        Mat<R> P;
        global_get<R, 18>(gapp + Layout<R, 18>::site_offset(par, Vh), Vh, cb, P);
        mul_right_dagger<3>(Ga, P, T); Ga = T;
        global_get<R, 18>(ga_f + Layout<R, 18>::site_offset(1 - par, Vh_f), Vh_f, cbf, P);
        mul_right_dagger<3>(Gb, P, T); Gb = T;
    }
    char* p0 = links + Layout<R, RECON>::link_offset(par, 0, Vh);
    global_get<R, RECON>(p0, Vh, cb, U);
    mul_left<3>(Ga, U, T);
    mul_right_dagger<3>(T, Gb, O);
    global_put<R, RECON>(p0, Vh, cb, O);
}

// ---- unitarity measure of Eq. (33): |1 - det U| per link ---------------------------
// one thread per stored link (slot = (parity, mu), cb), blockIdx.y = gauge copy; partial[(copy*gridDim.x + bx)*2]
// = (sum, max) of the block.  With RECON = 12 the third row is the rebuilt one (what every kernel uses).
template <class R, int RECON>
__global__ void unitarity_kernel(const char* base, int64_t Vh, int64_t copy_bytes, double* partial) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double dev = 0.0;
    if (i < 8 * Vh) {
        const char* p0 = base + blockIdx.y * copy_bytes + (i / Vh) * Layout<R, RECON>::LINK_BYTES * Vh;
        Mat<R> m;
        global_get<R, RECON>(p0, Vh, i % Vh, m);
        double dr = 0.0, di = 0.0;   // det = sum_j U_0j (U_1a U_2b - U_1b U_2a), (j,a,b) cyclic
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const int a = (j + 1) % 3, b = (j + 2) % 3;
            const double cr = (double)m.v[RE(1, a)] * m.v[RE(2, b)] - (double)m.v[IM(1, a)] * m.v[IM(2, b)] -
                              ((double)m.v[RE(1, b)] * m.v[RE(2, a)] - (double)m.v[IM(1, b)] * m.v[IM(2, a)]);
            const double ci = (double)m.v[RE(1, a)] * m.v[IM(2, b)] + (double)m.v[IM(1, a)] * m.v[RE(2, b)] -
                              ((double)m.v[RE(1, b)] * m.v[IM(2, a)] + (double)m.v[IM(1, b)] * m.v[RE(2, a)]);
            dr += (double)m.v[RE(0, j)] * cr - (double)m.v[IM(0, j)] * ci;
            di += (double)m.v[RE(0, j)] * ci + (double)m.v[IM(0, j)] * cr;
        }
        dev = sqrt((1.0 - dr) * (1.0 - dr) + di * di);
    }
    __shared__ double smax[32];
    double mx = dev;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o));
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) smax[w] = mx;
    double zero = 0.0;
    block_sum2(dev, zero);   // contains a __syncthreads after smax is written
    if (threadIdx.x == 0) {
        double m2 = 0.0;
        for (int k = 0; k < nw; ++k) m2 = fmax(m2, smax[k]);
        double* p = partial + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 2;
        p[0] = dev; p[1] = m2;
    }
}
// one block per copy: out[copy*2] = sum, out[copy*2+1] = max over the copy's nblocks partials
__global__ void unitarity_reduce_kernel(const double* partial, int nblocks, double* out) {
    __shared__ double smax[32];
    double s = 0.0, mx = 0.0;
    for (int k = threadIdx.x; k < nblocks; k += blockDim.x) {
        const double* p = partial + ((size_t)blockIdx.x * nblocks + k) * 2;
        s += p[0];
        mx = fmax(mx, p[1]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o));
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) smax[w] = mx;
    double zero = 0.0;
    block_sum2(s, zero);
    if (threadIdx.x == 0) {
        double m2 = 0.0;
        for (int k = 0; k < nw; ++k) m2 = fmax(m2, smax[k]);
        out[blockIdx.x * 2] = s; out[blockIdx.x * 2 + 1] = m2;
    }
}

// ---- random start on the gauge orbit (R27) ------------------------
// h(x) Haar-distributed on SU(3): two rows of independent complex standard normals (Box-Muller on
// Philox uniforms, counter = (site, 0, k | 3 << 8, 0), k = 0..2, key = seed + copy), Gram-Schmidt,
// third row (u x v)^*.  All in double.  One thread per site; field layout [copy][p][chunk][cb].
// h of one site: a function of (seed, lexicographic index of the site in the WHOLE lattice) alone
GF_DEV void haar_su3(uint64_t seed, uint32_t site, Mat<double>& h) {
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const u32x4 w = rng_draw(seed, site, 0u, k, 3, 0u);
        const double r0 = sqrt(-2.0 * log(uniform01(w.x))), r1 = sqrt(-2.0 * log(uniform01(w.z)));
        double s0, c0, s1, c1;
        sincos(6.283185307179586477 * uniform01(w.y), &s0, &c0);
        sincos(6.283185307179586477 * uniform01(w.w), &s1, &c1);
        h.v[4 * k] = r0 * c0; h.v[4 * k + 1] = r0 * s0; h.v[4 * k + 2] = r1 * c1; h.v[4 * k + 3] = r1 * s1;
    }
#pragma unroll
    for (int k = 12; k < 18; ++k) h.v[k] = 0.0;
    gram_schmidt(h);
}

// site_off: lexicographic index of this store's first site in the whole lattice (t-shards: t0 Nx Ny Nz; else 0)
template <class R>
__global__ void haar_field_kernel(char* field, Dims d, uint64_t seed, int64_t copy_bytes, int64_t site_off) {
    const int64_t V = (int64_t)d.Nt * d.Nx * d.Ny * d.Nz;
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= V) return;
    const int copy = blockIdx.y;
    int par, cb;
    site_to_cb(d, s, par, cb);
    Mat<double> h;
    haar_su3(seed + (uint64_t)copy, (uint32_t)(s + site_off), h);
    Mat<R> o;
#pragma unroll
    for (int k = 0; k < 18; ++k) o.v[k] = (R)h.v[k];
    global_put<R, 18>(field + copy * copy_bytes + Layout<R, 18>::site_offset(par, Vh_of(d)), Vh_of(d), cb, o);
}

// U_mu(x) <- h(x) U_mu(x) h(x+mu)^dagger (Eq. (1)) and, when tracked, g(x) <- h(x) g(x).
// One thread per site (parity blockIdx.z, copy blockIdx.y).
// t-shards: h(x + t_hat) of the last slice belongs to the store above and is recomputed here from its site index
// (top_site0 >= 0: lexicographic index, in the whole lattice, of the first site of the slice above; -1: not sharded)
template <class R, int RECON>
__global__ void gauge_apply_kernel(char* links, char* gtot, const char* hfield, Dims d, int64_t copy_links_bytes,
                                   int64_t copy_field_bytes, uint64_t seed, int64_t top_site0) {
    typedef Layout<R, RECON> L;
    const int Nzh = d.Nz >> 1;
    const int Vsh = d.Nx * d.Ny * Nzh;
    const int64_t Vh = (int64_t)d.Nt * Vsh;
    const int64_t cb = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= Vh) return;
    const int par = blockIdx.z;
    links += blockIdx.y * copy_links_bytes;
    hfield += blockIdx.y * copy_field_bytes;
    int64_t rem = cb;
    const int zh = (int)(rem % Nzh); rem /= Nzh;
    const int y = (int)(rem % d.Ny); rem /= d.Ny;
    const int x = (int)(rem % d.Nx);
    const int t = (int)(rem / d.Nx);
    const int r = (t + x + y + par) & 1;   // z = 2 zh + r
    // checkerboard index of x + mu (other parity)
    int64_t cbf[4];
    cbf[0] = cb + ((t == d.Nt - 1) ? -(int64_t)(d.Nt - 1) * Vsh : (int64_t)Vsh);
    cbf[1] = cb + ((x == d.Nx - 1) ? -(d.Nx - 1) * Nzh * d.Ny : Nzh * d.Ny);
    cbf[2] = cb + ((y == d.Ny - 1) ? -(d.Ny - 1) * Nzh : Nzh);
    cbf[3] = r ? ((zh == Nzh - 1) ? cb - (Nzh - 1) : cb + 1) : cb;
    Mat<R> h, hf, U, T, O;
    global_get<R, 18>(hfield + Layout<R, 18>::site_offset(par, Vh), Vh, cb, h);
#pragma unroll 1
    for (int mu = 0; mu < 4; ++mu) {
        if (mu == 0 && top_site0 >= 0 && t == d.Nt - 1) {
            Mat<double> hd;
            haar_su3(seed + (uint64_t)blockIdx.y, (uint32_t)(top_site0 + ((int64_t)x * d.Ny + y) * d.Nz + 2 * zh + r), hd);
#pragma unroll
            for (int k = 0; k < 18; ++k) hf.v[k] = (R)hd.v[k];
        } else {
            global_get<R, 18>(hfield + Layout<R, 18>::site_offset(1 - par, Vh), Vh, cbf[mu], hf);
        }
        char* p0 = links + L::link_offset(par, mu, Vh);
        global_get<R, RECON>(p0, Vh, cb, U);
        mul_left<3>(h, U, T);
        mul_right_dagger<3>(T, hf, O);
        global_put<R, RECON>(p0, Vh, cb, O);
    }
    if (gtot) {
        char* g0 = gtot + blockIdx.y * copy_field_bytes + Layout<R, 18>::site_offset(par, Vh);
        global_get<R, 18>(g0, Vh, cb, U);
        mul_left<3>(h, U, O);
        global_put<R, 18>(g0, Vh, cb, O);
    }
}

}  // namespace gf
