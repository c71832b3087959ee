// aux_su2.cuh — the kernels around the SU(2) half-sweep: layout conversion,
// F / theta reductions, reunitarisation, Coulomb finalisation, random start on the gauge orbit.
// Same grids and batching (blockIdx.y = gauge copy or copy*Nt + t) as their SU(3) counterparts in
// aux_kernels.cuh.  Host layout: links[t][x][y][z][mu][i][j][re,im], i,j in {0,1} (8 reals per link),
// transforms [t][x][y][z][i][j][re,im]; only the first row is read, the second is (-conj b, conj a).
#pragma once
#include "aux_kernels.cuh"
#include "su2.cuh"

namespace gf {

template <class E, class R>
GF_DEV void quat_from_host(const E* p, Quat<R>& q) {
    q.v[0] = (R)p[0]; q.v[3] = (R)p[1]; q.v[2] = (R)p[2]; q.v[1] = (R)p[3];
}
template <class E, class R>
GF_DEV void quat_to_host(E* p, const Quat<R>& q) {
    p[0] = (E)q.v[0]; p[1] = (E)q.v[3]; p[2] = (E)q.v[2]; p[3] = (E)q.v[1];        // ( u0 + i u3,  u2 + i u1)
    p[4] = (E)(-q.v[2]); p[5] = (E)q.v[1]; p[6] = (E)q.v[0]; p[7] = (E)(-q.v[3]);   // (-u2 + i u1,  u0 - i u3)
}

template <class E, class R>
__global__ void convert_in2_kernel(const E* __restrict__ src, char* links, Dims d, int64_t site0, int64_t nsites) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nsites * 4) return;
    const int64_t s = site0 + (i >> 2);
    const int mu = (int)(i & 3);
    const int64_t Vh = Vh_of(d);
    int par, cb;
    site_to_cb(d, s, par, cb);
    Quat<R> q;
    quat_from_host<E, R>(src + i * 8, q);
    global_put_q(links + Layout<R, 4>::link_offset(par, mu, Vh), Vh, cb, q);
}
template <class E, class R>
__global__ void convert_out2_kernel(E* __restrict__ dst, const char* links, Dims d, int64_t site0, int64_t nsites) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nsites * 4) return;
    const int64_t s = site0 + (i >> 2);
    const int mu = (int)(i & 3);
    const int64_t Vh = Vh_of(d);
    int par, cb;
    site_to_cb(d, s, par, cb);
    Quat<R> q;
    global_get_q(links + Layout<R, 4>::link_offset(par, mu, Vh), Vh, cb, q);
    quat_to_host<E, R>(dst + i * 8, q);
}
template <class E, class R>
__global__ void field_out2_kernel(E* __restrict__ dst, const char* field, Dims d, int64_t site0, int64_t nsites) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nsites) return;
    const int64_t Vh = Vh_of(d);
    int par, cb;
    site_to_cb(d, site0 + i, par, cb);
    Quat<R> q;
    global_get_q(field + Layout<R, 4>::site_offset(par, Vh), Vh, cb, q);
    quat_to_host<E, R>(dst + i * 8, q);
}
template <class R>
__global__ void field_identity2_kernel(char* field, int64_t Vh) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * Vh) return;
    Quat<R> q;
    q.v[0] = R(1); q.v[1] = q.v[2] = q.v[3] = R(0);
    global_put_q(field + Layout<R, 4>::site_offset((int)(i / Vh), Vh), Vh, i % Vh, q);
}

// reprojection onto SU(2): the quaternion normalised in double (R20 for N_c = 2)
template <class R>
__global__ void reunit2_kernel(char* base, int64_t Vh, int nslots, int64_t copy_bytes) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (int64_t)nslots * Vh) return;
    char* p0 = base + blockIdx.y * copy_bytes + (i / Vh) * Layout<R, 4>::LINK_BYTES * Vh;
    Quat<R> q;
    global_get_q(p0, Vh, i % Vh, q);
    const double a = q.v[0], b = q.v[1], c = q.v[2], e = q.v[3];
    const double n = 1.0 / sqrt(a * a + b * b + c * c + e * e);
    q.v[0] = (R)(a * n); q.v[1] = (R)(b * n); q.v[2] = (R)(c * n); q.v[3] = (R)(e * n);
    global_put_q(p0, Vh, i % Vh, q);
}

// F and theta, N_c = 2: grid (ceil(Vsh/block), ncopies*Nt, 2) as measure_kernel; double throughout
template <class R, int GAUGE>
__global__ void measure2_kernel(const char* links, Dims d, double* partial, int64_t copy_bytes) {
    typedef Layout<R, 4> L;
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
        const int64_t cb = (int64_t)t * Vsh + i;
        int rem = i;
        const int zh = rem % Nzh; rem /= Nzh;
        const int y = rem % d.Ny;
        const int x = rem / d.Ny;
        const int r = (t + x + y + par) & 1;
        const int sy = Nzh, sx = Nzh * d.Ny, st = Vsh;
        int64_t cbn[4];
        cbn[0] = cb + (t ? -st : (int64_t)(d.Nt - 1) * st);
        cbn[1] = cb + (x ? -sx : (d.Nx - 1) * sx);
        cbn[2] = cb + (y ? -sy : (d.Ny - 1) * sy);
        cbn[3] = r ? cb : (zh ? cb - 1 : cb + Nzh - 1);
        double a[4] = {0.0, 0.0, 0.0, 0.0}, D = 0.0, E = 0.0, F = 0.0;
#pragma unroll
        for (int mu = MU0; mu < 4; ++mu) {
            Quat<R> u, w;
            global_get_q(links + L::link_offset(par, mu, Vh), Vh, cb, u);
            global_get_q(links + L::link_offset(1 - par, mu, Vh), Vh, cbn[mu], w);
            if (GAUGE == GAUGE_MAG) {
                f_term += su2_diag2<double>(u);
                su2_acc_mag<double>(D, E, F, u, w);
            } else {
                f_term += 2.0 * (double)u.v[0];          // Re tr U_mu(x)
                su2_acc_landau<double>(a, u, w);
            }
        }
        th_term = (GAUGE == GAUGE_MAG) ? E * E + F * F : 0.5 * (a[1] * a[1] + a[2] * a[2] + a[3] * a[3]);
    }
    block_sum2(f_term, th_term);
    if (threadIdx.x == 0) {
        const int64_t b = ((int64_t)(blockIdx.y * 2 + par)) * gx + bx;
        partial[2 * b] = f_term;
        partial[2 * b + 1] = th_term;
    }
}

// U_0(x) <- R(x) U_0(x) R(x+t)^dag, R = g_tot g_applied^dag
template <class R>
__global__ void coulomb_finalize2_kernel(char* links, const char* gtot, const char* gapp, Dims d,
                                         int64_t copy_links_bytes, int64_t copy_field_bytes) {
    typedef Layout<R, 4> L;
    links += blockIdx.y * copy_links_bytes;
    gtot += blockIdx.y * copy_field_bytes;
    if (gapp) gapp += blockIdx.y * copy_field_bytes;
    const int Vsh = d.Nx * d.Ny * (d.Nz >> 1);
    const int64_t Vh = (int64_t)d.Nt * Vsh;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 2 * Vh) return;
    const int par = (int)(i / Vh);
    const int64_t cb = i % Vh;
    const int t = (int)(cb / Vsh);
    const int64_t cbf = cb + ((t == d.Nt - 1) ? -(int64_t)(d.Nt - 1) * Vsh : (int64_t)Vsh);
    Quat<R> U, Ga, Gb, P;
    global_get_q(gtot + L::site_offset(par, Vh), Vh, cb, Ga);
    global_get_q(gtot + L::site_offset(1 - par, Vh), Vh, cbf, Gb);
    if (gapp) {
        global_get_q(gapp + L::site_offset(par, Vh), Vh, cb, P);
        Ga = qmul_dagger(Ga, P);
        global_get_q(gapp + L::site_offset(1 - par, Vh), Vh, cbf, P);
        Gb = qmul_dagger(Gb, P);
    }
    char* p0 = links + L::link_offset(par, 0, Vh);
    global_get_q(p0, Vh, cb, U);
    global_put_q(p0, Vh, cb, qmul_dagger(qmul(Ga, U), Gb));
}

// h(x) Haar on SU(2) = uniform on S^3: four standard normals (Box-Muller on the Philox uniforms of counter
// (site, 0, 0 | 3 << 8, 0), key seed + copy) normalised; in double (R27 for N_c = 2)
template <class R>
__global__ void haar_field2_kernel(char* field, Dims d, uint64_t seed, int64_t copy_bytes) {
    const int64_t V = 2 * Vh_of(d);
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= V) return;
    const int copy = blockIdx.y;
    int par, cb;
    site_to_cb(d, s, par, cb);
    const u32x4 w = rng_draw(seed + (uint64_t)copy, (uint32_t)s, 0u, 0, 3, 0u);
    const double r0 = sqrt(-2.0 * log(uniform01(w.x))), r1 = sqrt(-2.0 * log(uniform01(w.z)));
    double s0, c0, s1, c1;
    sincos(6.283185307179586477 * uniform01(w.y), &s0, &c0);
    sincos(6.283185307179586477 * uniform01(w.w), &s1, &c1);
    // first row (a, b) = (r0 c0 + i r0 s0, r1 c1 + i r1 s1) = (u0 + i u3, u2 + i u1)
    const double u0 = r0 * c0, u3 = r0 * s0, u2 = r1 * c1, u1 = r1 * s1;
    const double n = 1.0 / sqrt(u0 * u0 + u1 * u1 + u2 * u2 + u3 * u3);
    Quat<R> q;
    q.v[0] = (R)(u0 * n); q.v[1] = (R)(u1 * n); q.v[2] = (R)(u2 * n); q.v[3] = (R)(u3 * n);
    global_put_q(field + copy * copy_bytes + Layout<R, 4>::site_offset(par, Vh_of(d)), Vh_of(d), cb, q);
}

// U_mu(x) <- h(x) U_mu(x) h(x+mu)^dagger (Eq. (1)); g(x) <- h(x) g(x) when tracked
template <class R>
__global__ void gauge_apply2_kernel(char* links, char* gtot, const char* hfield, Dims d, int64_t copy_links_bytes,
                                    int64_t copy_field_bytes) {
    typedef Layout<R, 4> L;
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
    const int r = (t + x + y + par) & 1;
    int64_t cbf[4];
    cbf[0] = cb + ((t == d.Nt - 1) ? -(int64_t)(d.Nt - 1) * Vsh : (int64_t)Vsh);
    cbf[1] = cb + ((x == d.Nx - 1) ? -(d.Nx - 1) * Nzh * d.Ny : Nzh * d.Ny);
    cbf[2] = cb + ((y == d.Ny - 1) ? -(d.Ny - 1) * Nzh : Nzh);
    cbf[3] = r ? ((zh == Nzh - 1) ? cb - (Nzh - 1) : cb + 1) : cb;
    Quat<R> h, hf, U;
    global_get_q(hfield + L::site_offset(par, Vh), Vh, cb, h);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        global_get_q(hfield + L::site_offset(1 - par, Vh), Vh, cbf[mu], hf);
        char* p0 = links + L::link_offset(par, mu, Vh);
        global_get_q(p0, Vh, cb, U);
        global_put_q(p0, Vh, cb, qmul_dagger(qmul(h, U), hf));
    }
    if (gtot) {
        char* g0 = gtot + blockIdx.y * copy_field_bytes + L::site_offset(par, Vh);
        global_get_q(g0, Vh, cb, U);
        global_put_q(g0, Vh, cb, qmul(h, U));
    }
}

// Eq. (33) for N_c = 2: det U = u0^2 + u1^2 + u2^2 + u3^2 for a matrix of the form of Eq. (15); same partials
// as unitarity_kernel (aux_kernels.cuh)
template <class R>
__global__ void unitarity2_kernel(const char* base, int64_t Vh, int64_t copy_bytes, double* partial) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double dev = 0.0;
    if (i < 8 * Vh) {
        Quat<R> q;
        global_get_q(base + blockIdx.y * copy_bytes + (i / Vh) * Layout<R, 4>::LINK_BYTES * Vh, Vh, i % Vh, q);
        const double a = q.v[0], b = q.v[1], c = q.v[2], e = q.v[3];
        dev = fabs(1.0 - (a * a + b * b + c * c + e * e));
    }
    __shared__ double smax[32];
    double mx = dev;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o));
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) smax[w] = mx;
    double zero = 0.0;
    block_sum2(dev, zero);
    if (threadIdx.x == 0) {
        double m2 = 0.0;
        for (int k = 0; k < nw; ++k) m2 = fmax(m2, smax[k]);
        double* p = partial + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 2;
        p[0] = dev; p[1] = m2;
    }
}

}  // namespace gf
