// sweep_su2.cuh — the half-sweep kernel for the gauge group SU(2).
//
// Alg. 1 with N_c = 2: there is one SU(2) "subgroup", the group itself, so Step 1
// is Eq. (20) resp. Eq. (29) applied once.  One thread per site; the 2d
// links are 2d quaternions = 32 (SP) or 64 (DP) registers, so they are loaded straight into registers
// with 16-byte loads (no shared-memory staging as in the SU(3) kernel), rotated (Step 2: two quaternion
// products per direction) and stored in place.  Algorithmic traffic: 2 * 2d * 4 * s bytes per site update
// (Landau SP 256 B, DP 512 B).  Grid, batching, frozen slices and the fused F / theta partials are those of
// sweep.cuh.
#pragma once
#include <atomic>

#include "su2.cuh"
#include "sweep.cuh"

namespace gf {

// per-site terms of the reductions, N_c = 2:
//   Landau/Coulomb: Re tr K(x) = a0;  tr[Delta Delta^dag] = 2 |k_vec|^2 = |a_vec|^2 / 2  (Eqs. (6)-(7), Delta = k_vec . sigma)
//   MAG: sum over the 2d links of sum_i |U_ii|^2 (Eq. (11));  |X_12|^2 = E^2 + F^2 (Eqs. (12)-(13): X_12 = F + i E)
template <class A>
GF_DEV A su2_theta_landau(const A a[4]) { return (a[1] * a[1] + a[2] * a[2] + a[3] * a[3]) * (A)0.5; }

template <class R, class A, int GAUGE, bool STOCH, bool TRACK, bool RED>
__global__ void __launch_bounds__(128, sizeof(R) == 8 ? 3 : 4) sweep_su2_kernel(const SweepArgs args) {
    typedef Layout<R, 4> L;
    constexpr int MU0 = (GAUGE == GAUGE_COULOMB) ? 1 : 0;
    constexpr int ND = 4 - MU0;
    // (CTAs of at most 128 threads: red_s below holds the partial sums of four warps; sweep_su2_block)
    pdl_launch_dependents();
    const int Nzh = args.Nz >> 1;
    const int Vsh = args.Nx * args.Ny * Nzh;
    const int64_t Vh = (int64_t)args.Nt * Vsh;
    if (args.slice_skip && args.slice_skip[blockIdx.y]) return;   // block-uniform
    const int copy = (args.ncopies == 1) ? 0 : blockIdx.y / args.Nt;
    const int t = blockIdx.y - copy * args.Nt;
    char* const links = args.links + copy * args.copy_links_bytes;
    char* const gtot = TRACK ? args.gtot + copy * args.copy_gtot_bytes : nullptr;
    const uint64_t seed = args.seed + (uint64_t)copy;
    const int i_raw = blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = i_raw < Vsh;
    const int i_s = active ? i_raw : Vsh - 1;
    const int64_t cb = (int64_t)t * Vsh + i_s;

    // a1: decode, neighbours (as in sweep.cuh)
    int zh, y;
    const int xy = fast_div(i_s, Nzh, args.rcp_nzh, zh);
    const int x = fast_div(xy, args.Ny, args.rcp_ny, y);
    const int par = (GAUGE == GAUGE_COULOMB) ? ((args.parity + t) & 1) : args.parity;
    const int r = (t + x + y + par) & 1;
    const int z = 2 * zh + r;
    const uint32_t site = (uint32_t)((((uint32_t)t * (uint32_t)args.Nx + (uint32_t)x) * (uint32_t)args.Ny + (uint32_t)y) *
                                     (uint32_t)args.Nz + (uint32_t)z);   // unsigned: V may exceed 2^31
    const int sy = Nzh, sx = Nzh * args.Ny;
    const int64_t st = Vsh;
    int64_t cbn[4];
    cbn[0] = cb + (t ? -st : (int64_t)(args.Nt - 1) * st);
    cbn[1] = cb + (x ? -sx : (args.Nx - 1) * sx);
    cbn[2] = cb + (y ? -sy : (args.Ny - 1) * sy);
    cbn[3] = r ? cb : (zh ? cb - 1 : cb + Nzh - 1);

    // a2: gather
    const int64_t lstride = (int64_t)L::LINK_BYTES * Vh;
    char* const up0 = links + L::link_offset(par, MU0, Vh);
    char* const dn0 = links + L::link_offset(1 - par, MU0, Vh);
    Quat<R> up[ND], dn[ND];
    pdl_wait();   // nothing of the previous kernel's output is read above this line
#pragma unroll
    for (int m = 0; m < ND; ++m) {
        global_get_q(up0 + m * lstride, Vh, cb, up[m]);
        global_get_q(dn0 + m * lstride, Vh, cbn[MU0 + m], dn[m]);
    }
    Quat<R> gt;
    if (TRACK) global_get_q(gtot + L::site_offset(par, Vh), Vh, cb, gt);
    HbDraw<A> pre;   // heatbath: the link-independent part, while the loads are in flight
    if (STOCH && args.algo == ALGO_SA) hb_draws<A>(GAUGE == GAUGE_MAG, seed, site, args.sweep_index, 0, pre);

    // a3: neighbourhood summary
    A a[4] = {A(0), A(0), A(0), A(0)};
    A Dm = A(0), Em = A(0), Fm = A(0);
#pragma unroll
    for (int m = 0; m < ND; ++m) {
        if (GAUGE == GAUGE_MAG) su2_acc_mag<A>(Dm, Em, Fm, up[m], dn[m]);
        else su2_acc_landau<A>(a, up[m], dn[m]);
    }
    A th_pre = A(0);
    if (RED) th_pre = (GAUGE == GAUGE_MAG) ? Em * Em + Fm * Fm : su2_theta_landau<A>(a);
    if (GAUGE == GAUGE_MAG) {
        const A lam = sqrt_t(Dm * Dm + Em * Em + Fm * Fm);   // Eq. (29)
        a[0] = Dm + lam; a[1] = -Em; a[2] = -Fm; a[3] = A(0);
    }

    // a4/a5: Step 1
    A g[4];
    choose_rule<STOCH, A>(a, g, GAUGE == GAUGE_MAG, Dm, Em, Fm, args, seed, site, 0, pre);
    Quat<R> gr;
#pragma unroll
    for (int k = 0; k < 4; ++k) gr.v[k] = (R)g[k];

    // a6: Step 2
#pragma unroll
    for (int m = 0; m < ND; ++m) {
        up[m] = qmul(gr, up[m]);
        dn[m] = qmul_dagger(dn[m], gr);
    }

    // a9 fused: terms of the updated site, from the rotated links
    double red_f = 0.0, red_th = 0.0, red_pre = 0.0;
    if (RED) {
        A b[4] = {A(0), A(0), A(0), A(0)};
        A D2 = A(0), E2 = A(0), F2 = A(0), fd = A(0);
#pragma unroll
        for (int m = 0; m < ND; ++m) {
            if (GAUGE == GAUGE_MAG) {
                su2_acc_mag<A>(D2, E2, F2, up[m], dn[m]);
                fd += su2_diag2<A>(up[m]) + su2_diag2<A>(dn[m]);
            } else {
                su2_acc_landau<A>(b, up[m], dn[m]);
            }
        }
        if (active) {
            red_f = (double)((GAUGE == GAUGE_MAG) ? fd : b[0]);
            red_th = (double)((GAUGE == GAUGE_MAG) ? E2 * E2 + F2 * F2 : su2_theta_landau<A>(b));
            red_pre = (double)th_pre;
        }
    }

    // a7: scatter
    if (active) {
#pragma unroll
        for (int m = 0; m < ND; ++m) {
            global_put_q(up0 + m * lstride, Vh, cb, up[m]);
            global_put_q(dn0 + m * lstride, Vh, cbn[MU0 + m], dn[m]);
        }
        if (TRACK) global_put_q(gtot + L::site_offset(par, Vh), Vh, cb, qmul(gr, gt));
    }

    if (RED) {   // block-uniform
        __shared__ double red_s[3][4];
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        red_f = warp_sum_d(red_f);
        red_th = warp_sum_d(red_th);
        red_pre = warp_sum_d(red_pre);
        if (lane == 0) { red_s[0][w] = red_f; red_s[1][w] = red_th; red_s[2][w] = red_pre; }
        __syncthreads();
        if (threadIdx.x == 0) {
            const int nw = (blockDim.x + 31) >> 5;
            double s0 = 0.0, s1 = 0.0, s2 = 0.0;
            for (int k = 0; k < nw; ++k) { s0 += red_s[0][k]; s1 += red_s[1][k]; s2 += red_s[2][k]; }
            double* p = args.red + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 3;
            p[0] = s0; p[1] = s1; p[2] = s2;
        }
    }
}

inline int sweep_su2_block(int Vsh, int block_override) {
    int block = block_override;
    if (block <= 0 || block > 128) block = 128;
    const int need = ((Vsh + 31) / 32) * 32;
    return block < need ? block : need;
}

template <class R, class A, int GAUGE, bool STOCH, bool TRACK, bool RED>
static cudaError_t launch_su2_one(const SweepArgs& args, int block, cudaStream_t stream) {
    const int Vsh = args.Nx * args.Ny * (args.Nz / 2);
    block = sweep_su2_block(Vsh, block);
    const dim3 grid((unsigned)((Vsh + block - 1) / block), (unsigned)(args.ncopies * args.Nt));
    // the kernel uses no dynamic shared memory; a small grid asks for some so that its CTAs spread over all SMs
    // (sweep_inst.cuh, launch_one)
    auto kern = sweep_su2_kernel<R, A, GAUGE, STOCH, TRACK, RED>;
    size_t smem_launch = 0;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    DevLimits lim;
    e = dev_limits(dev, lim);   // SM count and shared-memory limits of this device (cached)
    if (e != cudaSuccess) return e;
    const long long ctas = (long long)grid.x * grid.y, per_sm = (ctas + lim.sms - 1) / lim.sms;
    if (per_sm <= 8 && lim.smem_per_sm / (size_t)per_sm > 2048) {
        smem_launch = (lim.smem_per_sm / (size_t)per_sm - 1024) / 1024 * 1024;
        if (smem_launch > lim.smem_cta_cap) smem_launch = lim.smem_cta_cap;
        static std::atomic<int> attr_set[64];
        if (dev < 0 || dev >= 64 || !attr_set[dev].load(std::memory_order_acquire)) {
            e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)lim.smem_cta_cap);
            if (e != cudaSuccess) return e;
            // (no carveout preference: the kernel loads through L1, which large grids want as large as it gets)
            if (dev >= 0 && dev < 64) attr_set[dev].store(1, std::memory_order_release);
        }
    }
    return launch_with_pdl(kern, grid, dim3((unsigned)block), smem_launch, stream, args);
}
template <class R, class A, int GAUGE>
static cudaError_t launch_su2_gauge(const SweepArgs& args, bool track, int block, cudaStream_t stream) {
    const bool stoch = (args.algo == ALGO_SR || args.algo == ALGO_SA);
    const int which = (stoch ? 4 : 0) | (track ? 2 : 0) | (args.red ? 1 : 0);
    switch (which) {
        case 0: return launch_su2_one<R, A, GAUGE, false, false, false>(args, block, stream);
        case 1: return launch_su2_one<R, A, GAUGE, false, false, true>(args, block, stream);
        case 2: return launch_su2_one<R, A, GAUGE, false, true, false>(args, block, stream);
        case 3: return launch_su2_one<R, A, GAUGE, false, true, true>(args, block, stream);
        case 4: return launch_su2_one<R, A, GAUGE, true, false, false>(args, block, stream);
        case 5: return launch_su2_one<R, A, GAUGE, true, false, true>(args, block, stream);
        case 6: return launch_su2_one<R, A, GAUGE, true, true, false>(args, block, stream);
        default: return launch_su2_one<R, A, GAUGE, true, true, true>(args, block, stream);
    }
}

// host-side launcher of one (R, A) family; instantiated in sweep_su2.cu
template <class R, class A>
cudaError_t launch_sweep_su2(const SweepArgs& args, int gauge, bool track, int block, cudaStream_t stream) {
    switch (gauge) {
        case GAUGE_LANDAU: return launch_su2_gauge<R, A, GAUGE_LANDAU>(args, track, block, stream);
        case GAUGE_COULOMB: return launch_su2_gauge<R, A, GAUGE_COULOMB>(args, track, block, stream);
        case GAUGE_MAG: return launch_su2_gauge<R, A, GAUGE_MAG>(args, track, block, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace gf
