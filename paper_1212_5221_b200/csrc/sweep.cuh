// sweep.cuh — the half-sweep kernel: Alg. 1's "for all x of sublattice" for
// one parity, one thread per site (BASELINE.json north_star), sm_100a.
//
// Design: the 2d links of a site are streamed once from HBM into the thread's
// private slice of shared memory with 16-byte cp.async (no register staging, 2d*R*s bytes in flight
// per thread), then
//   pass 1  builds the neighbourhood summary in registers: K(x) of Eq. (19) for
//           Landau/Coulomb, the three Hermitian M_k for MAG;
//   Step 1  runs the three Cabibbo-Marinari subgroup updates on the summary
//           alone (K -> g K, M_k -> g M_k g^dagger), accumulating G = g3 g2 g1;
//   pass 2  re-reads each link from shared memory, rotates it once with the SU(3) matrix G
//           (Step 2: U_mu(x) <- G U_mu(x), U_mu(x-mu) <- U_mu(x-mu) G^dagger)
//           and writes it back in place with 16-byte stores.
// Every link is read once and written once per half-sweep; nothing is re-read from HBM.  No
// __syncthreads: a thread only ever touches its own shared-memory slice.
#pragma once
#include <atomic>
#include <cstdint>
#include <cuda_runtime.h>

#include "layout.cuh"
#include "step1.cuh"
#include "su3.cuh"

namespace gf {

enum { GAUGE_LANDAU = 0, GAUGE_COULOMB = 1, GAUGE_MAG = 2 };

struct SweepArgs {
    char* links;   // device link store (layout.cuh)
    char* gtot;    // tracked transform store or nullptr
    int Nt, Nx, Ny, Nz;
    int parity;          // active parity of this half-sweep
    int algo;            // ALGO_*
    double param;        // omega | p | T
    uint64_t seed;
    uint32_t sweep_index;
    // nullptr, or per-block partial sums [gridDim.y = Nt][gridDim.x][3] of
    //   (F term after the update, theta term after the update, theta term before the update)
    // of the sites this launch updates (fused reductions)
    double* red;
    const unsigned char* slice_skip;   // nullptr, or [ncopies*Nt]: 1 = leave this time-slice alone (frozen)
    // batched gauge copies: blockIdx.y = copy*Nt + t; copy c lives at links + c*copy_links_bytes
    // (gtot + c*copy_gtot_bytes) and draws its random numbers with the Philox key seed + c
    int ncopies;
    int64_t copy_links_bytes, copy_gtot_bytes;
    uint32_t rcp_nzh, rcp_ny;   // floor(2^32 / (Nz/2)), floor(2^32 / Ny): site decode without integer division
    int pdl;                    // launch with programmatic stream serialization (host side only)
    // t-sharding: this store holds the time-slices [t_off, t_off + Nt) of a
    // lattice split over several link stores.  The only links a half-sweep touches outside its own store are
    // U_0(x - t_hat) of its first slice: they are the last slice (Nt_dn - 1) of the store links_dn (Vh_dn sites per
    // parity), which the kernel reads and writes in place (the same device, a peer mapping or an IPC mapping).
    // Not sharded: links_dn = links, Vh_dn = Vh, Nt_dn = Nt, t_off = 0 (the periodic wrap in t).
    char* links_dn;
    int64_t Vh_dn, copy_links_bytes_dn;
    int Nt_dn, t_off;
};

// Programmatic dependent launch (sm_90+): a half-sweep lets the next kernel in the stream be scheduled as soon as
// all of its own CTAs have started (launch_dependents), and touches no link before the previous kernel has
// completed and flushed (wait).  The next half-sweep's CTAs thus fill the SMs that the tail of this one leaves
// idle and have their site decode done when the data dependency resolves: the inter-kernel bubble that
// dominates small lattices shrinks.  Without the launch attribute both instructions are no-ops.
GF_DEV void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
GF_DEV void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// n / d for 0 <= n < 2^31 with rcp = floor(2^32 / d) (d >= 2): __umulhi underestimates the quotient by at most one
GF_DEV int fast_div(int n, int d, uint32_t rcp, int& rem) {
    int q = (int)__umulhi((uint32_t)n, rcp);
    rem = n - q * d;
    if (rem >= d) { ++q; rem -= d; }
    return q;
}
inline uint32_t fast_div_rcp(int d) { return d > 1 ? (uint32_t)(4294967296ull / (uint64_t)d) : 0xffffffffu; }

// ---- asynchronous global -> shared copies -------------------------------------------------
GF_DEV void cp_async16(uint32_t saddr, const void* g) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(saddr), "l"(g) : "memory");
}
GF_DEV void cp_async8(uint32_t saddr, const void* g) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(saddr), "l"(g) : "memory");
}
GF_DEV void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

// ---- 16-byte vector moves between shared/global memory and a register matrix ------------------
template <class R>
struct Vec16;
template <>
struct Vec16<float> {
    typedef float4 type;
    GF_DEV static void unpack(const float4& q, float* v) { v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w; }
    GF_DEV static float4 pack(const float* v) { return make_float4(v[0], v[1], v[2], v[3]); }
};
template <>
struct Vec16<double> {
    typedef double2 type;
    GF_DEV static void unpack(const double2& q, double* v) { v[0] = q.x; v[1] = q.y; }
    GF_DEV static double2 pack(const double* v) { return make_double2(v[0], v[1]); }
};

// read link slot l of this thread from shared memory (and rebuild row 2 when RECON = 12).
// The slice stride NTHR is the compile-time maximal CTA size, whatever blockDim.x is, so that every
// shared-memory address is tid*16 + an immediate (+ one multiply-add for a run-time l).
template <class R, int RECON, int NTHR>
GF_DEV void smem_get(const unsigned char* smem, int nlinks, int l, Mat<R>& m) {
    typedef Layout<R, RECON> L;
    typedef typename Vec16<R>::type V;
    const int tid = threadIdx.x;
    const unsigned char* base = smem + tid * 16 + l * (L::NV16 * NTHR * 16);
#pragma unroll
    for (int c = 0; c < L::NV16; ++c) {
        const V q = *reinterpret_cast<const V*>(base + c * NTHR * 16);
        Vec16<R>::unpack(q, &m.v[c * L::PER16]);
    }
    if (L::TAIL8) {
        const float2 q = *reinterpret_cast<const float2*>(smem + nlinks * L::NV16 * NTHR * 16 +
                                                          (l * NTHR + tid) * 8);
        m.v[L::NV16 * L::PER16] = (R)q.x;
        m.v[L::NV16 * L::PER16 + 1] = (R)q.y;
    }
    if (RECON == 12) reconstruct_row2(m);
}

// store the first RECON reals of a matrix to its place in HBM
template <class R, int RECON>
GF_DEV void global_put(char* plane0, int64_t Vh, int64_t cb, const Mat<R>& m) {
    typedef Layout<R, RECON> L;
    typedef typename Vec16<R>::type V;
    const int64_t plane = 16 * Vh;
    char* q = plane0 + cb * 16;
#pragma unroll
    for (int c = 0; c < L::NV16; ++c, q += plane)
        *reinterpret_cast<V*>(q) = Vec16<R>::pack(&m.v[c * L::PER16]);
    if (L::TAIL8)
        *reinterpret_cast<float2*>(q - cb * 8) =
            make_float2((float)m.v[L::NV16 * L::PER16], (float)m.v[L::NV16 * L::PER16 + 1]);
}
template <class R, int RECON>
GF_DEV void global_get(const char* plane0, int64_t Vh, int64_t cb, Mat<R>& m) {
    typedef Layout<R, RECON> L;
    typedef typename Vec16<R>::type V;
#pragma unroll
    for (int c = 0; c < L::NV16; ++c) {
        const V q = *reinterpret_cast<const V*>(plane0 + (int64_t)c * 16 * Vh + cb * 16);
        Vec16<R>::unpack(q, &m.v[c * L::PER16]);
    }
    if (L::TAIL8) {
        const float2 q = *reinterpret_cast<const float2*>(plane0 + (int64_t)L::NV16 * 16 * Vh + cb * 8);
        m.v[L::NV16 * L::PER16] = (R)q.x;
        m.v[L::NV16 * L::PER16 + 1] = (R)q.y;
    }
    if (RECON == 12) reconstruct_row2(m);
}

// ---- Step 1 for one subgroup (I,J), index S in the Cabibbo-Marinari order (0,1),(0,2),(1,2) ----
// d: what hb_draws (below) prepared for this subgroup while the gather was in flight (heatbath only).  The heatbath
// runs in the Step-1 type A: float on SP contexts, double on MP and DP contexts (step1.cuh).
template <bool STOCH, class A>
GF_DEV void choose_rule(const A a[4], A g[4], bool mag, A Dm, A Em, A Fm, const SweepArgs& args, uint64_t seed,
                        uint32_t site, int sub, const HbDraw<A>& d) {
    if (!STOCH) {
        if (args.algo == ALGO_MICRO) rule_micro<A>(a, g);
        else rule_or<A>(a, (A)args.param, g);
    } else {
        if (args.algo == ALGO_SR) {
            // stochastic relaxation: g^2 with probability p, else g
            const double u = uniform01(rng_draw(seed, site, args.sweep_index, sub, 0, 0).x);
            if (u < args.param) rule_micro<A>(a, g);
            else rule_or<A>(a, A(1), g);
        } else if (mag) {
            hb_finish_mag<A>(Dm, Em, Fm, (A)args.param, d, g);
        } else {
            hb_finish_landau<A>(a, (A)args.param, d, seed, site, args.sweep_index, sub, g);
        }
    }
}

// the link-independent part of the heatbath for subgroup `sub` (step1.cuh): Philox draws and what follows from them
// alone.  The half-sweep kernels call it between issuing their loads and waiting for them.
template <class A>
GF_DEV void hb_draws(bool mag, uint64_t seed, uint32_t site, uint32_t sweep, int sub, HbDraw<A>& d) {
    if (mag) hb_draws_mag<A>(seed, site, sweep, sub, d);
    else hb_draws_landau<A>(seed, site, sweep, sub, d);
}

template <int I, int J, int S, bool STOCH, class A>
GF_DEV void subgroup_landau(Mat<A>& K, Mat<A>& G, const SweepArgs& args, uint64_t seed, uint32_t site, const HbDraw<A>& d) {
    // Fig. A.10 on K, signs per Eq. (15)
    A a[4], g[4];
    a[0] = K.v[RE(I, I)] + K.v[RE(J, J)];
    a[3] = K.v[IM(I, I)] - K.v[IM(J, J)];
    a[2] = K.v[RE(I, J)] - K.v[RE(J, I)];
    a[1] = K.v[IM(I, J)] + K.v[IM(J, I)];
    choose_rule<STOCH, A>(a, g, false, A(0), A(0), A(0), args, seed, site, S, d);
    sub_left<I, J>(K, g);   // applying g at x maps K(x) -> g K(x)
    sub_left<I, J>(G, g);
}

template <int I, int J, int S, bool STOCH, class A>
GF_DEV void subgroup_mag(Herm<A> (&M)[3], Mat<A>& G, const SweepArgs& args, uint64_t seed, uint32_t site, const HbDraw<A>& d) {
    // f(g) = const + g^T [[D,E,F],[E,-D,0],[F,0,-D]] g  (Eqs. (25)-(28), SU(3) form)
    // (I,J) with I < J: off-diagonal element (I,J) of a Herm is o[2*OFF], o[2*OFF+1]
    constexpr int OFF = (I == 0) ? (J - 1) : 2;
    const A aa = M[I].d[I] + M[J].d[J];
    const A bb = M[I].d[J] + M[J].d[I];
    const A Dm = (aa - bb) / A(2);
    const A Em = M[I].o[2 * OFF + 1] - M[J].o[2 * OFF + 1];
    const A Fm = M[I].o[2 * OFF] - M[J].o[2 * OFF];
    const A lam = sqrt_t(Dm * Dm + Em * Em + Fm * Fm);   // Eq. (29)
    A a[4] = {Dm + lam, -Em, -Fm, A(0)}, g[4];
    choose_rule<STOCH, A>(a, g, true, Dm, Em, Fm, args, seed, site, S, d);
#pragma unroll
    for (int k = 0; k < 3; ++k) {   // M_k -> g M_k g^dagger
        Mat<A> F;
        herm_expand(M[k], F);
        sub_left<I, J>(F, g);
        sub_right_dagger<I, J>(F, g);
        herm_compress(F, M[k]);
    }
    sub_left<I, J>(G, g);
}

// ---- per-site terms of the fused reductions (a9 inside the sweep) -------------
// Landau/Coulomb: Delta(x) = traceless[(K - K^dag)/2i] (Eq. (6)), term = tr[Delta Delta^dag]
// (Eq. (7)); Re tr K(x) is the sum of Re tr over the 2d links that touch x (Eq. (17)).
template <class A>
GF_DEV A theta_term_landau(const Mat<A>& K) {
    A sum = A(0), tr = A(0);
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const A xr = K.v[RE(a, b)] - K.v[RE(b, a)];
            const A xi = K.v[IM(a, b)] + K.v[IM(b, a)];
            sum += A(0.25) * (xr * xr + xi * xi);
            if (a == b) tr += A(0.5) * xi;
        }
    const A th = sum - tr * tr / A(3);   // = tr[Delta Delta^dag] >= 0; rounding can leave -1e-23 at a fixed point
    return th > A(0) ? th : A(0);
}
template <class A>
GF_DEV A f_term_landau(const Mat<A>& K) { return K.v[RE(0, 0)] + K.v[RE(1, 1)] + K.v[RE(2, 2)]; }
// MAG: sum over the subgroups of |X^s_12|^2 = E_s^2 + F_s^2 (R11); local value of Eq. (11)
template <class A>
GF_DEV A theta_term_mag(const Herm<A> (&M)[3]) {
    A th = A(0);
    {   const A E = M[0].o[1] - M[1].o[1], F = M[0].o[0] - M[1].o[0]; th += E * E + F * F; }
    {   const A E = M[0].o[3] - M[2].o[3], F = M[0].o[2] - M[2].o[2]; th += E * E + F * F; }
    {   const A E = M[1].o[5] - M[2].o[5], F = M[1].o[4] - M[2].o[4]; th += E * E + F * F; }
    return th;
}
template <class A>
GF_DEV A f_term_mag(const Herm<A> (&M)[3]) { return M[0].d[0] + M[1].d[1] + M[2].d[2]; }

GF_DEV double warp_sum_d(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// ---- the kernel ----------------------------------------------------------------------------
#ifndef GF_SP_BLOCK
#define GF_SP_BLOCK 128     // CTA size of the float-storage kernels
#endif
#ifndef GF_SP_MIN_CTAS
#define GF_SP_MIN_CTAS 3
#endif
#ifndef GF_MIN_CTAS_MP
#define GF_MIN_CTAS_MP 4
#endif
#ifndef GF_SP_STOCH_BLOCK
#define GF_SP_STOCH_BLOCK 64    // CTA size of the float kernels with a stochastic rule
#endif
#ifndef GF_SP_STOCH_MIN_CTAS
#define GF_SP_STOCH_MIN_CTAS 9
#endif
template <class R, class A = R>
struct SweepLaunch {   // CTA shape per storage type
    static constexpr int MAX_BLOCK = sizeof(R) == 4 ? GF_SP_BLOCK : 64;
    static constexpr int MIN_CTAS = (sizeof(R) == 4 && sizeof(A) == 8) ? GF_MIN_CTAS_MP : (sizeof(R) == 4 ? GF_SP_MIN_CTAS : 3);
    // The float kernels with a stochastic rule are bound by arithmetic latency, not by HBM: more warps in flight pay.
    // The shared-memory slice is laid out for the largest CTA of the instantiation, so a 64-thread maximum halves it
    // (SP-12 Landau: 24.6 KB) and 9 CTAs = 18 warps fit an SM where four 128-thread CTAs gave 16.
    __host__ __device__ static constexpr bool small_cta(bool stoch) { return stoch && sizeof(R) == 4 && sizeof(A) == 4; }
    __host__ __device__ static constexpr int max_block(bool stoch) { return small_cta(stoch) ? GF_SP_STOCH_BLOCK : MAX_BLOCK; }
    __host__ __device__ static constexpr int min_ctas(bool stoch) { return small_cta(stoch) ? GF_SP_STOCH_MIN_CTAS : MIN_CTAS; }
};

template <class R, class A, int RECON, int GAUGE, bool STOCH, bool TRACK, bool RED>
__global__ void __launch_bounds__(SweepLaunch<R, A>::max_block(STOCH), SweepLaunch<R, A>::min_ctas(STOCH))
sweep_kernel(const SweepArgs args) {
    typedef Layout<R, RECON> L;
    constexpr int MU0 = (GAUGE == GAUGE_COULOMB) ? 1 : 0;
    constexpr int ND = 4 - MU0;
    constexpr int NL = 2 * ND;
    static_assert(SweepLaunch<R, A>::MAX_BLOCK <= 128, "red_s below holds the partial sums of at most four warps");
    extern __shared__ __align__(16) unsigned char smem[];

    // grid = (ceil(Vsh / block), ncopies*Nt): blockIdx.y is (gauge copy, time-slice), so a CTA never
    // straddles slices (per-slice reductions, frozen slices).  Threads past the end of the slice redo
    // the last site without storing, so that every thread reaches the block reduction.
    pdl_launch_dependents();
    const int Nzh = args.Nz >> 1;
    const int Vsh = args.Nx * args.Ny * Nzh;
    const int64_t Vh = (int64_t)args.Nt * Vsh;
    if (args.slice_skip && args.slice_skip[blockIdx.y]) return;   // block-uniform (flags are set by the host between runs of kernels)
    const int copy = (args.ncopies == 1) ? 0 : blockIdx.y / args.Nt;
    const int t = blockIdx.y - copy * args.Nt;
    char* const links = args.links + copy * args.copy_links_bytes;
    char* const gtot = TRACK ? args.gtot + copy * args.copy_gtot_bytes : nullptr;
    const uint64_t seed = args.seed + (uint64_t)copy;
    const int i_raw = blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = i_raw < Vsh;
    const int i_s = active ? i_raw : Vsh - 1;
    const int64_t cb = (int64_t)t * Vsh + i_s;

    // ---- a1: decode the checkerboard index, neighbours with periodic wrap ----
    int zh, y;
    const int xy = fast_div(i_s, Nzh, args.rcp_nzh, zh);
    const int x = fast_div(xy, args.Ny, args.rcp_ny, y);
    // own parity in the 4-d colouring; Coulomb's 3-d colouring p3 maps to (p3 + t) & 1
    const int par = (GAUGE == GAUGE_COULOMB) ? ((args.parity + t) & 1) : args.parity;
    const int r = (t + x + y + par) & 1;   // z = 2 zh + r
    const int z = 2 * zh + r;
    // Philox site index: lexicographic in the whole lattice (t_off = first slice of this store; an even number,
    // so the colouring above is the global one)
    const uint32_t site = (uint32_t)((((uint32_t)(t + args.t_off) * (uint32_t)args.Nx + (uint32_t)x) * (uint32_t)args.Ny +
                                      (uint32_t)y) * (uint32_t)args.Nz + (uint32_t)z);

    // checkerboard index of x - mu (lives in the other parity's arrays)
    const int sy = Nzh, sx = Nzh * args.Ny;
    const int64_t st = Vsh;
    // x - t_hat of the first slice: the last slice of the store links_dn (block-uniform)
    const int64_t Vh_t = t ? Vh : args.Vh_dn;
    const int64_t cbn0 = t ? cb - st : (int64_t)(args.Nt_dn - 1) * st + i_s;
    const int64_t cbn1 = cb + (x ? -sx : (args.Nx - 1) * sx);
    const int64_t cbn2 = cb + (y ? -sy : (args.Ny - 1) * sy);
    const int64_t cbn3 = r ? cb : (zh ? cb - 1 : cb + Nzh - 1);

    // ---- a2: stream the 2d links into this thread's shared-memory slice ----
    // slice layout [link][chunk][NTHR] x 16 bytes (+ [link][NTHR] x 8 bytes of SP-18 tails); pointers step
    // by one chunk plane (16 Vh bytes) and one link array (LINK_BYTES Vh bytes)
    constexpr int NTHR = SweepLaunch<R, A>::max_block(STOCH);
    const int tid = threadIdx.x;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem) + (uint32_t)tid * 16;
    const int64_t plane = 16 * Vh;
    const int64_t lstride = (int64_t)L::LINK_BYTES * Vh;
    char* const up0 = links + L::link_offset(par, MU0, Vh);        // U_mu(x): own parity
    char* const dn0 = links + L::link_offset(1 - par, MU0, Vh);    // U_mu(x - mu): other parity
    char* const dnt = (t ? links : args.links_dn + copy * args.copy_links_bytes_dn) + L::link_offset(1 - par, 0, Vh_t);   // U_0(x - t_hat)
    pdl_wait();   // nothing of the previous kernel's output is read above this line
    {
        const char* pu = up0;
        const char* pd = dn0;
#pragma unroll
        for (int m = 0; m < ND; ++m, pu += lstride, pd += lstride) {
            const int mu = MU0 + m;
            const int64_t cdn = (mu == 0) ? cbn0 : (mu == 1) ? cbn1 : (mu == 2) ? cbn2 : cbn3;
            const int64_t plane_d = (mu == 0) ? 16 * Vh_t : plane;
            const char* qu = pu + cb * 16;
            const char* qd = ((mu == 0) ? dnt : pd) + cdn * 16;
#pragma unroll
            for (int c = 0; c < L::NV16; ++c, qu += plane, qd += plane_d) {
                cp_async16(sbase + (uint32_t)(((2 * m) * L::NV16 + c) * NTHR * 16), qu);
                cp_async16(sbase + (uint32_t)(((2 * m + 1) * L::NV16 + c) * NTHR * 16), qd);
            }
            if (L::TAIL8) {
                cp_async8(sbase - (uint32_t)tid * 8 + (uint32_t)(NL * L::NV16 * NTHR * 16 + (2 * m) * NTHR * 8),
                          qu - cb * 8);
                cp_async8(sbase - (uint32_t)tid * 8 + (uint32_t)(NL * L::NV16 * NTHR * 16 + (2 * m + 1) * NTHR * 8),
                          qd - cdn * 8);
            }
        }
    }
    Mat<R> Gt;
    if (TRACK) global_get<R, 18>(gtot + Layout<R, 18>::site_offset(par, Vh), Vh, cb, Gt);
    // stochastic rules: draws, logarithms and trigonometric functions of the three subgroups while the gather is in
    // flight (a rolled loop and a local array: one copy of the code, nothing held in registers over pass 1)
    HbDraw<A> pre[STOCH ? 3 : 1];
    if (STOCH && args.algo == ALGO_SA) {
#pragma unroll 1
        for (int s = 0; s < 3; ++s) hb_draws<A>(GAUGE == GAUGE_MAG, seed, site, args.sweep_index, s, pre[s]);
    }
    cp_async_wait_all();

    // ---- a3: neighbourhood summary, pass 1 over the links ----
    // (loops over mu are deliberately not unrolled: one link pair in registers at a time)
    Mat<A> G;
    set_identity(G);
    Mat<A> K;             // Landau/Coulomb: Eq. (19)
    Herm<A> M[3];         // MAG: Hermitian M_k
    if (GAUGE == GAUGE_MAG) {
        set_zero(M[0]); set_zero(M[1]); set_zero(M[2]);
    } else {
        set_zero(K);
    }
#pragma unroll 1
    for (int m = 0; m < ND; ++m) {
        Mat<R> U;
        smem_get<R, RECON, NTHR>(smem, NL, 2 * m, U);       // U_mu(x)
        if (GAUGE == GAUGE_MAG) { mag_acc_up<0>(M[0], U); mag_acc_up<1>(M[1], U); mag_acc_up<2>(M[2], U); }
        else acc_plain(K, U);
        smem_get<R, RECON, NTHR>(smem, NL, 2 * m + 1, U);   // U_mu(x - mu)
        if (GAUGE == GAUGE_MAG) { mag_acc_down<0>(M[0], U); mag_acc_down<1>(M[1], U); mag_acc_down<2>(M[2], U); }
        else acc_dagger(K, U);
    }

    // fused reductions: theta term of this site before its update (completes theta of the previous sweep)
    constexpr bool red = RED;   // args.red is non-null exactly when RED
    A th_pre = A(0);
    if (red) th_pre = (GAUGE == GAUGE_MAG) ? theta_term_mag<A>(M) : theta_term_landau<A>(K);

    // ---- a4/a5: Step 1 through the three SU(2) subgroups, G = g3 g2 g1 ----
    if (GAUGE == GAUGE_MAG) {
        subgroup_mag<0, 1, 0, STOCH, A>(M, G, args, seed, site, pre[0]);
        subgroup_mag<0, 2, 1, STOCH, A>(M, G, args, seed, site, pre[STOCH ? 1 : 0]);
        subgroup_mag<1, 2, 2, STOCH, A>(M, G, args, seed, site, pre[STOCH ? 2 : 0]);
    } else {
        subgroup_landau<0, 1, 0, STOCH, A>(K, G, args, seed, site, pre[0]);
        subgroup_landau<0, 2, 1, STOCH, A>(K, G, args, seed, site, pre[STOCH ? 1 : 0]);
        subgroup_landau<1, 2, 2, STOCH, A>(K, G, args, seed, site, pre[STOCH ? 2 : 0]);
    }

    // the summary now is that of the updated site (K -> G K, M_k -> G M_k G^dag): its F and theta terms
    double red_f = 0.0, red_th = 0.0, red_pre = 0.0;
    if (red && active) {
        red_f = (double)((GAUGE == GAUGE_MAG) ? f_term_mag<A>(M) : f_term_landau<A>(K));
        red_th = (double)((GAUGE == GAUGE_MAG) ? theta_term_mag<A>(M) : theta_term_landau<A>(K));
        red_pre = (double)th_pre;
    }

    // ---- a6/a7: Step 2, pass 2 over the links: rotate and write back in place ----
    constexpr int NR = (RECON == 12) ? 2 : 3;
    Mat<R> Gr;   // G in the storage type (MP: Step 2 in SP)
#pragma unroll
    for (int k = 0; k < 18; ++k) Gr.v[k] = (R)G.v[k];
    {
        char* pu = up0;
        char* pd = dn0;
#pragma unroll 1
        for (int m = 0; m < ND; ++m, pu += lstride, pd += lstride) {
            const int mu = MU0 + m;
            const int64_t cdn = (mu == 0) ? cbn0 : (mu == 1) ? cbn1 : (mu == 2) ? cbn2 : cbn3;
            Mat<R> U, O;
            smem_get<R, RECON, NTHR>(smem, NL, 2 * m, U);
            mul_left<NR>(Gr, U, O);
            if (active) global_put<R, RECON>(pu, Vh, cb, O);
            smem_get<R, RECON, NTHR>(smem, NL, 2 * m + 1, U);
            mul_right_dagger<NR>(U, Gr, O);
            if (active) global_put<R, RECON>((mu == 0) ? dnt : pd, (mu == 0) ? Vh_t : Vh, cdn, O);
        }
    }

    // ---- a8: accumulate the transform, g_tot(x) <- G g_tot(x) ----
    if (TRACK) {
        Mat<R> O;
        mul_left<3>(G, Gt, O);
        if (active) global_put<R, 18>(gtot + Layout<R, 18>::site_offset(par, Vh), Vh, cb, O);
    }

    // ---- a9 fused: block partials of (F, theta after, theta before), double, fixed order ----
    if (red) {   // block-uniform
        __shared__ double red_s[3][4];
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        red_f = warp_sum_d(red_f);
        red_th = warp_sum_d(red_th);
        red_pre = warp_sum_d(red_pre);
        if (lane == 0) { red_s[0][w] = red_f; red_s[1][w] = red_th; red_s[2][w] = red_pre; }
        __syncthreads();
        if (threadIdx.x == 0) {
            const int nw = (blockDim.x + 31) >> 5;
            double a = 0.0, b = 0.0, c = 0.0;
            for (int k = 0; k < nw; ++k) { a += red_s[0][k]; b += red_s[1][k]; c += red_s[2][k]; }
            double* p = args.red + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 3;
            p[0] = a; p[1] = b; p[2] = c;
        }
    }
}

// CTA size actually used for a slice of Vsh sites per parity (block_override = 0: default)
template <class R, class A = R>
inline int sweep_block(int Vsh, int block_override, bool stoch = false) {
    int block = block_override;
    const int maxb = SweepLaunch<R, A>::max_block(stoch);
    if (block <= 0 || block > maxb) block = maxb;
    const int need = ((Vsh + 31) / 32) * 32;
    return block < need ? block : need;
}

// What the launchers need to know about a device, asked once per device: the SM count, the shared memory of an SM and
// the most dynamic shared memory one CTA may opt into (a B200: 148, 228 KB, 227 KB).  smem_cta_cap leaves 1 KB of the
// opt-in limit to the kernels' static shared memory (226 KB on a B200).
struct DevLimits {
    int sms;
    size_t smem_per_sm, smem_cta_cap;
};
inline cudaError_t dev_limits(int dev, DevLimits& out) {
    struct Slot {
        std::atomic<int> ready;
        DevLimits v;
    };
    static Slot cache[64];
    const bool cached = dev >= 0 && dev < 64;
    if (cached && cache[dev].ready.load(std::memory_order_acquire)) { out = cache[dev].v; return cudaSuccess; }
    int sms = 0, per_sm = 0, optin = 0;
    cudaError_t e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&per_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return e;
    if (sms <= 0 || per_sm <= 0 || optin <= 1024) return cudaErrorInvalidDevice;
    out.sms = sms;
    out.smem_per_sm = (size_t)per_sm;
    out.smem_cta_cap = (size_t)optin - 1024;
    if (cached) {   // several threads may get here together: they write the same values
        cache[dev].v = out;
        cache[dev].ready.store(1, std::memory_order_release);
    }
    return cudaSuccess;
}

// launch a half-sweep kernel, with the programmatic-stream-serialization attribute when args.pdl is set
template <class K>
inline cudaError_t launch_with_pdl(K kern, dim3 grid, dim3 block, size_t smem, cudaStream_t stream, const SweepArgs& args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = args.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, args);
}

// host-side launcher of one (R, A, RECON) family; defined in sweep_inst.cuh
template <class R, class A, int RECON>
cudaError_t launch_sweep(const SweepArgs& args, int gauge, bool track, int block, cudaStream_t stream);

}  // namespace gf
