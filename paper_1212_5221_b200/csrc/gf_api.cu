// gf_api.cu — the C ABI of include/gf.h: context, dispatch and the run loops.
// Host code only orchestrates; every step of the path runs in the kernels of sweep.cuh /
// aux_kernels.cuh.  There is no CPU fallback.
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/gf.h"
#include "aux_kernels.cuh"
#include "sweep.cuh"

using namespace gf;

namespace gf {
// one explicit instantiation per translation unit sweep_<prec><recon>.cu
extern template cudaError_t launch_sweep<float, float, 18>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep<float, float, 12>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep<float, double, 18>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep<float, double, 12>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep<double, double, 18>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep<double, double, 12>(const SweepArgs&, int, bool, int, cudaStream_t);
}  // namespace gf

struct gf_ctx {
    int Nx, Ny, Nz, Nt;
    int precision, recon;
    unsigned flags;
    cudaStream_t stream;
    int64_t V, Vh;
    size_t real_bytes;      // 4 | 8
    char* links;            // device link store
    char* gtot;             // tracked transform (18 reals/site) or nullptr
    char* gapplied;         // part of gtot already applied to the temporal links (Coulomb) or nullptr
    bool have_links;
    bool temporal_stale;    // Coulomb sweeps ran since the temporal links were last finalised
    // reductions
    double* partial;        // per-block partial sums
    int meas_block, meas_gx;
    double* slice_dev;      // [2*Nt]
    double* slice_host;     // pinned [2*Nt]
    // fused reductions of the half-sweep kernels
    double* red_part[2];    // per-block partials of the even / odd half-sweep, [Nt][gx_max][3]
    double* red_dev;        // [2][Nt][3] slice sums
    double* red_host;       // pinned copy
    int fused;              // gf_run uses the fused reductions (default 1)
    // per-slice Coulomb fixing (GF_FLAG_FREEZE_SLICES)
    unsigned char* skip_dev;    // [Nt] 1 = slice stopped, its CTAs exit at once
    unsigned char* skip_host;   // pinned copy
    std::vector<int> slice_sweeps;   // sweeps applied to every slice by the last gf_run
    bool have_slice_sweeps;
    // host<->device staging for gf_set_links / gf_get_*
    void* staging;
    size_t staging_bytes;
    int64_t device_bytes;
    int block_override;     // 0 = default CTA size
    // kernel timing (gf_kernel_timing)
    bool timing;
    std::vector<cudaEvent_t> ev;   // pairs (start, stop)
    size_t ev_used;
    int64_t launches;       // kernels enqueued by this context (gf_launch_count)
    char err[512];
};

static int fail(gf_ctx* c, int code, const char* fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}
#define CU(call)                                                                                     \
    do {                                                                                             \
        cudaError_t e_ = (call);                                                                     \
        if (e_ != cudaSuccess)                                                                       \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? GF_ENOMEM : GF_ECUDA, "%s: %s (%s:%d)", #call, \
                        cudaGetErrorString(e_), __FILE__, __LINE__);                                 \
    } while (0)

static Dims dims_of(const gf_ctx* c) {
    Dims d = {c->Nt, c->Nx, c->Ny, c->Nz};
    return d;
}
static int64_t link_store_bytes(const gf_ctx* c) { return (int64_t)8 * c->recon * c->real_bytes * c->Vh; }
static int64_t field_store_bytes(const gf_ctx* c) { return (int64_t)2 * 18 * c->real_bytes * c->Vh; }

// dispatch on (storage type, RECON)
#define DISPATCH_RR(ctx, FN, ...)                                                  \
    do {                                                                           \
        if ((ctx)->real_bytes == 4) {                                              \
            if ((ctx)->recon == 18) { FN(float, 18, __VA_ARGS__); }                \
            else { FN(float, 12, __VA_ARGS__); }                                   \
        } else {                                                                   \
            if ((ctx)->recon == 18) { FN(double, 18, __VA_ARGS__); }               \
            else { FN(double, 12, __VA_ARGS__); }                                  \
        }                                                                          \
    } while (0)

extern "C" {

const char* gf_version(void) { return "gf 0.1 (sm_100a)"; }

const char* gf_last_error(const gf_ctx* ctx) { return ctx ? ctx->err : "null context"; }

int64_t gf_device_bytes(const gf_ctx* ctx) { return ctx ? ctx->device_bytes : 0; }

int64_t gf_volume(const gf_ctx* ctx) { return ctx ? ctx->V : 0; }

int gf_create(gf_ctx** out, int Nx, int Ny, int Nz, int Nt, int precision, int recon, unsigned flags,
              void* cuda_stream) {
    if (!out) return GF_EINVAL;
    *out = nullptr;
    const int n[4] = {Nx, Ny, Nz, Nt};
    for (int k = 0; k < 4; ++k)
        if (n[k] < 2 || (n[k] & 1)) return GF_EINVAL;
    const double vol = (double)Nx * Ny * Nz * Nt;
    if (vol >= 4294967296.0) return GF_EINVAL;
    if (precision != GF_SP && precision != GF_DP && precision != GF_MP) return GF_EINVAL;
    if (recon != 18 && recon != 12) return GF_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) return GF_ECUDA;   // no CPU fallback
    gf_ctx* ctx = new (std::nothrow) gf_ctx();
    if (!ctx) return GF_ENOMEM;
    ctx->Nx = Nx; ctx->Ny = Ny; ctx->Nz = Nz; ctx->Nt = Nt;
    ctx->precision = precision; ctx->recon = recon; ctx->flags = flags;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->V = (int64_t)Nx * Ny * Nz * Nt;
    ctx->Vh = ctx->V / 2;
    ctx->real_bytes = (precision == GF_DP) ? 8 : 4;
    ctx->links = ctx->gtot = ctx->gapplied = nullptr;
    ctx->have_links = false; ctx->temporal_stale = false;
    ctx->partial = nullptr; ctx->slice_dev = nullptr; ctx->slice_host = nullptr;
    ctx->red_part[0] = ctx->red_part[1] = nullptr; ctx->red_dev = nullptr; ctx->red_host = nullptr;
    ctx->fused = 1;
    ctx->skip_dev = nullptr; ctx->skip_host = nullptr; ctx->have_slice_sweeps = false;
    ctx->staging = nullptr; ctx->staging_bytes = 0;
    ctx->device_bytes = 0; ctx->block_override = 0;
    ctx->timing = false; ctx->ev_used = 0; ctx->launches = 0;
    ctx->err[0] = 0;

    cudaError_t e = cudaMalloc((void**)&ctx->links, (size_t)link_store_bytes(ctx));
    if (e == cudaSuccess) ctx->device_bytes += link_store_bytes(ctx);
    if (e == cudaSuccess && (flags & GF_FLAG_TRACK_TRANSFORM)) {
        e = cudaMalloc((void**)&ctx->gtot, (size_t)field_store_bytes(ctx));
        if (e == cudaSuccess) ctx->device_bytes += field_store_bytes(ctx);
    }
    ctx->meas_block = 128;
    const int Vsh = Nx * Ny * (Nz / 2);
    ctx->meas_gx = (Vsh + ctx->meas_block - 1) / ctx->meas_block;
    const size_t npart = (size_t)ctx->meas_gx * Nt * 2;
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->partial, npart * 2 * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->slice_dev, (size_t)2 * Nt * sizeof(double));
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->slice_host, (size_t)2 * Nt * sizeof(double));
    const size_t nred = (size_t)((Vsh + 31) / 32) * Nt * 3;   // smallest CTA = 32 sites
    for (int k = 0; k < 2; ++k)
        if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->red_part[k], nred * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->red_dev, (size_t)6 * Nt * sizeof(double));
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->red_host, (size_t)6 * Nt * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->skip_dev, (size_t)Nt);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->skip_host, (size_t)Nt);
    if (e != cudaSuccess) {
        const int code = (e == cudaErrorMemoryAllocation) ? GF_ENOMEM : GF_ECUDA;
        gf_destroy(ctx);
        cudaGetLastError();
        return code;
    }
    ctx->device_bytes += (int64_t)(npart * 2 + 2 * Nt + 2 * nred + 6 * Nt) * sizeof(double);
    *out = ctx;
    return GF_OK;
}

int gf_destroy(gf_ctx* ctx) {
    if (!ctx) return GF_OK;
    cudaStreamSynchronize(ctx->stream);
    cudaFree(ctx->links);
    cudaFree(ctx->gtot);
    cudaFree(ctx->gapplied);
    cudaFree(ctx->partial);
    cudaFree(ctx->slice_dev);
    cudaFree(ctx->staging);
    cudaFree(ctx->red_part[0]);
    cudaFree(ctx->red_part[1]);
    cudaFree(ctx->red_dev);
    cudaFree(ctx->skip_dev);
    if (ctx->skip_host) cudaFreeHost(ctx->skip_host);
    if (ctx->red_host) cudaFreeHost(ctx->red_host);
    if (ctx->slice_host) cudaFreeHost(ctx->slice_host);
    for (cudaEvent_t ev : ctx->ev) cudaEventDestroy(ev);
    delete ctx;
    return GF_OK;
}

int gf_sync(gf_ctx* ctx) {
    if (!ctx) return GF_EINVAL;
    CU(cudaStreamSynchronize(ctx->stream));
    return GF_OK;
}

static int ensure_staging(gf_ctx* ctx, size_t bytes) {
    if (ctx->staging_bytes >= bytes) return GF_OK;
    if (ctx->staging) {
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->staging);
        ctx->device_bytes -= (int64_t)ctx->staging_bytes;
        ctx->staging = nullptr; ctx->staging_bytes = 0;
    }
    CU(cudaMalloc(&ctx->staging, bytes));
    ctx->staging_bytes = bytes;
    ctx->device_bytes += (int64_t)bytes;
    return GF_OK;
}

static const int64_t STAGE_SITES = 1 << 18;   // sites per host<->device staging chunk

#define CONVERT_IN(R, RECON, E, src, s0, ns)                                                            \
    convert_in_kernel<E, R, RECON><<<(unsigned)(((ns) * 4 + 255) / 256), 256, 0, ctx->stream>>>(        \
        (const E*)(src), ctx->links, dims_of(ctx), (s0), (ns))
#define CONVERT_OUT(R, RECON, E, dst, s0, ns)                                                           \
    convert_out_kernel<E, R, RECON><<<(unsigned)(((ns) * 4 + 255) / 256), 256, 0, ctx->stream>>>(       \
        (E*)(dst), ctx->links, dims_of(ctx), (s0), (ns))

static int reset_transform(gf_ctx* ctx) {
    if (ctx->gtot) {
        const unsigned g = (unsigned)((2 * ctx->Vh + 255) / 256);
        if (ctx->real_bytes == 4) field_identity_kernel<float><<<g, 256, 0, ctx->stream>>>(ctx->gtot, ctx->Vh);
        else field_identity_kernel<double><<<g, 256, 0, ctx->stream>>>(ctx->gtot, ctx->Vh);
        CU(cudaGetLastError());
        ++ctx->launches;
    }
    if (ctx->gapplied) {
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->gapplied);
        ctx->gapplied = nullptr;
        ctx->device_bytes -= field_store_bytes(ctx);
    }
    ctx->temporal_stale = false;
    return GF_OK;
}

int gf_set_links(gf_ctx* ctx, const void* links, int elem_bytes, int is_device) {
    if (!ctx) return GF_EINVAL;
    if (!links || (elem_bytes != 4 && elem_bytes != 8)) return fail(ctx, GF_EINVAL, "gf_set_links: bad arguments");
    const int64_t link_elems = 4 * 18;
    if (is_device) {
        if (elem_bytes == 4) DISPATCH_RR(ctx, CONVERT_IN, float, links, (int64_t)0, ctx->V);
        else DISPATCH_RR(ctx, CONVERT_IN, double, links, (int64_t)0, ctx->V);
        CU(cudaGetLastError());
        ++ctx->launches;
    } else {
        const int64_t chunk = ctx->V < STAGE_SITES ? ctx->V : STAGE_SITES;
        int rc = ensure_staging(ctx, (size_t)(chunk * link_elems * elem_bytes));
        if (rc) return rc;
        for (int64_t s0 = 0; s0 < ctx->V; s0 += chunk) {
            const int64_t ns = (ctx->V - s0 < chunk) ? ctx->V - s0 : chunk;
            const char* src = (const char*)links + s0 * link_elems * elem_bytes;
            CU(cudaMemcpyAsync(ctx->staging, src, (size_t)(ns * link_elems * elem_bytes), cudaMemcpyHostToDevice,
                               ctx->stream));
            if (elem_bytes == 4) DISPATCH_RR(ctx, CONVERT_IN, float, ctx->staging, s0, ns);
            else DISPATCH_RR(ctx, CONVERT_IN, double, ctx->staging, s0, ns);
            CU(cudaGetLastError());
            ++ctx->launches;
        }
    }
    int rc = reset_transform(ctx);
    if (rc) return rc;
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->have_links = true;
    return GF_OK;
}

int gf_get_links(gf_ctx* ctx, void* links, int elem_bytes, int is_device) {
    if (!ctx) return GF_EINVAL;
    if (!links || (elem_bytes != 4 && elem_bytes != 8)) return fail(ctx, GF_EINVAL, "gf_get_links: bad arguments");
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_get_links: no links set");
    if (ctx->temporal_stale && ctx->gtot) {
        int rc = gf_coulomb_finalize(ctx);
        if (rc) return rc;
    }
    const int64_t link_elems = 4 * 18;
    if (is_device) {
        if (elem_bytes == 4) DISPATCH_RR(ctx, CONVERT_OUT, float, links, (int64_t)0, ctx->V);
        else DISPATCH_RR(ctx, CONVERT_OUT, double, links, (int64_t)0, ctx->V);
        CU(cudaGetLastError());
        ++ctx->launches;
    } else {
        const int64_t chunk = ctx->V < STAGE_SITES ? ctx->V : STAGE_SITES;
        int rc = ensure_staging(ctx, (size_t)(chunk * link_elems * elem_bytes));
        if (rc) return rc;
        for (int64_t s0 = 0; s0 < ctx->V; s0 += chunk) {
            const int64_t ns = (ctx->V - s0 < chunk) ? ctx->V - s0 : chunk;
            char* dst = (char*)links + s0 * link_elems * elem_bytes;
            if (elem_bytes == 4) DISPATCH_RR(ctx, CONVERT_OUT, float, ctx->staging, s0, ns);
            else DISPATCH_RR(ctx, CONVERT_OUT, double, ctx->staging, s0, ns);
            CU(cudaGetLastError());
            ++ctx->launches;
            CU(cudaMemcpyAsync(dst, ctx->staging, (size_t)(ns * link_elems * elem_bytes), cudaMemcpyDeviceToHost,
                               ctx->stream));
        }
    }
    CU(cudaStreamSynchronize(ctx->stream));
    return GF_OK;
}

int gf_get_gauge_transform(gf_ctx* ctx, void* g, int elem_bytes, int is_device) {
    if (!ctx) return GF_EINVAL;
    if (!g || (elem_bytes != 4 && elem_bytes != 8)) return fail(ctx, GF_EINVAL, "gf_get_gauge_transform: bad arguments");
    if (!ctx->gtot) return fail(ctx, GF_ESTATE, "gf_get_gauge_transform: context created without GF_FLAG_TRACK_TRANSFORM");
    const int64_t chunk = is_device ? ctx->V : (ctx->V < 4 * STAGE_SITES ? ctx->V : 4 * STAGE_SITES);
    if (!is_device) {
        int rc = ensure_staging(ctx, (size_t)(chunk * 18 * elem_bytes));
        if (rc) return rc;
    }
    for (int64_t s0 = 0; s0 < ctx->V; s0 += chunk) {
        const int64_t ns = (ctx->V - s0 < chunk) ? ctx->V - s0 : chunk;
        void* dst = is_device ? (void*)((char*)g + s0 * 18 * elem_bytes) : ctx->staging;
        const unsigned grid = (unsigned)((ns + 255) / 256);
        if (ctx->real_bytes == 4) {
            if (elem_bytes == 4) field_out_kernel<float, float><<<grid, 256, 0, ctx->stream>>>((float*)dst, ctx->gtot, dims_of(ctx), s0, ns);
            else field_out_kernel<double, float><<<grid, 256, 0, ctx->stream>>>((double*)dst, ctx->gtot, dims_of(ctx), s0, ns);
        } else {
            if (elem_bytes == 4) field_out_kernel<float, double><<<grid, 256, 0, ctx->stream>>>((float*)dst, ctx->gtot, dims_of(ctx), s0, ns);
            else field_out_kernel<double, double><<<grid, 256, 0, ctx->stream>>>((double*)dst, ctx->gtot, dims_of(ctx), s0, ns);
        }
        CU(cudaGetLastError());
        ++ctx->launches;
        if (!is_device)
            CU(cudaMemcpyAsync((char*)g + s0 * 18 * elem_bytes, ctx->staging, (size_t)(ns * 18 * elem_bytes),
                               cudaMemcpyDeviceToHost, ctx->stream));
    }
    CU(cudaStreamSynchronize(ctx->stream));
    return GF_OK;
}

// ---- sweeps ----------------------------------------------------------------------------------
static int check_sweep_args(gf_ctx* ctx, int gauge, int algo, double param) {
    if (!ctx) return GF_EINVAL;
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "no links set (call gf_set_links first)");
    if (gauge < GF_LANDAU || gauge > GF_MAG) return fail(ctx, GF_EINVAL, "unknown gauge %d", gauge);
    if (algo < GF_OR || algo > GF_MICRO) return fail(ctx, GF_EINVAL, "unknown algorithm %d", algo);
    if (algo == GF_OR && !(param >= 1.0 && param < 2.0)) return fail(ctx, GF_EINVAL, "omega = %g not in [1,2)", param);
    if (algo == GF_SR && !(param >= 0.0 && param <= 1.0)) return fail(ctx, GF_EINVAL, "p = %g not in [0,1]", param);
    if (algo == GF_SA && !(param > 0.0)) return fail(ctx, GF_EINVAL, "T = %g not positive", param);
    return GF_OK;
}

static int launch_half(gf_ctx* ctx, int gauge, int algo, double param, uint64_t seed, uint32_t sweep_index,
                       int parity, double* red = nullptr, const unsigned char* skip = nullptr) {
    SweepArgs a;
    a.links = ctx->links; a.gtot = ctx->gtot;
    a.Nt = ctx->Nt; a.Nx = ctx->Nx; a.Ny = ctx->Ny; a.Nz = ctx->Nz;
    a.parity = parity; a.algo = algo; a.param = param; a.seed = seed; a.sweep_index = sweep_index;
    a.red = red;
    a.slice_skip = skip;
    const bool track = ctx->gtot != nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (ctx->timing) {
        if (ctx->ev_used + 2 > ctx->ev.size()) {
            cudaEvent_t a0, a1;
            CU(cudaEventCreate(&a0));
            CU(cudaEventCreate(&a1));
            ctx->ev.push_back(a0);
            ctx->ev.push_back(a1);
        }
        e0 = ctx->ev[ctx->ev_used]; e1 = ctx->ev[ctx->ev_used + 1];
        ctx->ev_used += 2;
        CU(cudaEventRecord(e0, ctx->stream));
    }
    cudaError_t e;
    const int blk = ctx->block_override;
    if (ctx->precision == GF_DP) {
        e = (ctx->recon == 18) ? launch_sweep<double, double, 18>(a, gauge, track, blk, ctx->stream)
                               : launch_sweep<double, double, 12>(a, gauge, track, blk, ctx->stream);
    } else if (ctx->precision == GF_MP) {
        e = (ctx->recon == 18) ? launch_sweep<float, double, 18>(a, gauge, track, blk, ctx->stream)
                               : launch_sweep<float, double, 12>(a, gauge, track, blk, ctx->stream);
    } else {
        e = (ctx->recon == 18) ? launch_sweep<float, float, 18>(a, gauge, track, blk, ctx->stream)
                               : launch_sweep<float, float, 12>(a, gauge, track, blk, ctx->stream);
    }
    CU(e);
    ++ctx->launches;
    if (ctx->timing) CU(cudaEventRecord(e1, ctx->stream));
    return GF_OK;
}

static int pre_sweep(gf_ctx* ctx, int gauge) {
    if (gauge == GF_COULOMB) {
        if (ctx->gtot) ctx->temporal_stale = true;
    } else if (ctx->temporal_stale) {
        return gf_coulomb_finalize(ctx);
    }
    return GF_OK;
}

int gf_half_sweep(gf_ctx* ctx, int gauge, int algo, double param, uint64_t seed, uint32_t sweep_index,
                  int parity) {
    int rc = check_sweep_args(ctx, gauge, algo, param);
    if (rc) return rc;
    if (parity != 0 && parity != 1) return fail(ctx, GF_EINVAL, "parity %d", parity);
    rc = pre_sweep(ctx, gauge);
    if (rc) return rc;
    return launch_half(ctx, gauge, algo, param, seed, sweep_index, parity);
}

int gf_sweep(gf_ctx* ctx, int gauge, int algo, double param, uint64_t seed, uint32_t sweep_index) {
    int rc = check_sweep_args(ctx, gauge, algo, param);
    if (rc) return rc;
    rc = pre_sweep(ctx, gauge);
    if (rc) return rc;
    rc = launch_half(ctx, gauge, algo, param, seed, sweep_index, 0);   // even first (Alg. 1)
    if (rc) return rc;
    return launch_half(ctx, gauge, algo, param, seed, sweep_index, 1);
}

// ---- reductions --------------------------------------------------------------------------------
#define MEASURE(R, RECON, gauge_)                                                                          \
    do {                                                                                                   \
        dim3 grid((unsigned)ctx->meas_gx, (unsigned)ctx->Nt, 2);                                           \
        if ((gauge_) == GF_LANDAU)                                                                         \
            measure_kernel<R, RECON, GAUGE_LANDAU><<<grid, ctx->meas_block, 0, ctx->stream>>>(ctx->links, dims_of(ctx), ctx->partial); \
        else if ((gauge_) == GF_COULOMB)                                                                   \
            measure_kernel<R, RECON, GAUGE_COULOMB><<<grid, ctx->meas_block, 0, ctx->stream>>>(ctx->links, dims_of(ctx), ctx->partial); \
        else                                                                                               \
            measure_kernel<R, RECON, GAUGE_MAG><<<grid, ctx->meas_block, 0, ctx->stream>>>(ctx->links, dims_of(ctx), ctx->partial); \
    } while (0)

// enqueue the reduction and the copy of the 2*Nt slice sums to pinned host memory
static int enqueue_measure(gf_ctx* ctx, int gauge) {
    DISPATCH_RR(ctx, MEASURE, gauge);
    CU(cudaGetLastError());
    slice_reduce_kernel<<<ctx->Nt, 128, 0, ctx->stream>>>(ctx->partial, 2 * ctx->meas_gx, ctx->Nt, ctx->slice_dev);
    CU(cudaGetLastError());
    ctx->launches += 2;
    CU(cudaMemcpyAsync(ctx->slice_host, ctx->slice_dev, (size_t)2 * ctx->Nt * sizeof(double), cudaMemcpyDeviceToHost,
                       ctx->stream));
    return GF_OK;
}

// after a stream sync: normalise (Eqs. (4), (7), (11)) in a fixed order
static void finish_measure(const gf_ctx* ctx, int gauge, double* F, double* theta, double* theta_slice,
                           double* theta_max) {
    const int nd = (gauge == GF_COULOMB) ? 3 : 4;
    const double Vs = (double)ctx->Nx * ctx->Ny * ctx->Nz;
    double fs = 0.0, ths = 0.0, tmax = 0.0;
    for (int t = 0; t < ctx->Nt; ++t) {
        fs += ctx->slice_host[t];
        ths += ctx->slice_host[ctx->Nt + t];
        const double th_t = ctx->slice_host[ctx->Nt + t] / (3.0 * Vs);
        if (theta_slice) theta_slice[t] = th_t;
        if (th_t > tmax) tmax = th_t;
    }
    if (F) *F = fs / (3.0 * nd * (double)ctx->V);
    if (theta) *theta = ths / (3.0 * (double)ctx->V);
    if (theta_max) *theta_max = tmax;
}

int gf_measure(gf_ctx* ctx, int gauge, double* F, double* theta, double* theta_slice) {
    if (!ctx) return GF_EINVAL;
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_measure: no links set");
    if (gauge < GF_LANDAU || gauge > GF_MAG) return fail(ctx, GF_EINVAL, "unknown gauge %d", gauge);
    if (gauge != GF_COULOMB && ctx->temporal_stale) {
        int rc = gf_coulomb_finalize(ctx);
        if (rc) return rc;
    }
    int rc = enqueue_measure(ctx, gauge);
    if (rc) return rc;
    CU(cudaStreamSynchronize(ctx->stream));
    finish_measure(ctx, gauge, F, theta, theta_slice, nullptr);
    return GF_OK;
}

// ---- reunitarisation -----------------------------------------------------------------------------
#define REUNIT_LINKS(R, RECON, dummy)                                                                       \
    reunit_kernel<R, RECON><<<(unsigned)((8 * ctx->Vh + 255) / 256), 256, 0, ctx->stream>>>(ctx->links, ctx->Vh, 8)

int gf_reunitarize(gf_ctx* ctx) {
    if (!ctx) return GF_EINVAL;
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_reunitarize: no links set");
    DISPATCH_RR(ctx, REUNIT_LINKS, 0);
    CU(cudaGetLastError());
    ++ctx->launches;
    if (ctx->gtot) {
        const unsigned g = (unsigned)((2 * ctx->Vh + 255) / 256);
        if (ctx->real_bytes == 4) reunit_kernel<float, 18><<<g, 256, 0, ctx->stream>>>(ctx->gtot, ctx->Vh, 2);
        else reunit_kernel<double, 18><<<g, 256, 0, ctx->stream>>>(ctx->gtot, ctx->Vh, 2);
        CU(cudaGetLastError());
        ++ctx->launches;
    }
    return GF_OK;
}

// ---- Coulomb finalisation ------------------------------------------------------------------------
#define FINALIZE(R, RECON, dummy)                                                                           \
    coulomb_finalize_kernel<R, RECON><<<(unsigned)((2 * ctx->Vh + 127) / 128), 128, 0, ctx->stream>>>(       \
        ctx->links, ctx->gtot, ctx->gapplied, dims_of(ctx))

int gf_coulomb_finalize(gf_ctx* ctx) {
    if (!ctx) return GF_EINVAL;
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_coulomb_finalize: no links set");
    if (!ctx->gtot) return fail(ctx, GF_ESTATE, "gf_coulomb_finalize: context created without GF_FLAG_TRACK_TRANSFORM");
    if (!ctx->temporal_stale) return GF_OK;
    DISPATCH_RR(ctx, FINALIZE, 0);
    CU(cudaGetLastError());
    ++ctx->launches;
    if (!ctx->gapplied) {
        CU(cudaMalloc((void**)&ctx->gapplied, (size_t)field_store_bytes(ctx)));
        ctx->device_bytes += field_store_bytes(ctx);
    }
    CU(cudaMemcpyAsync(ctx->gapplied, ctx->gtot, (size_t)field_store_bytes(ctx), cudaMemcpyDeviceToDevice, ctx->stream));
    ctx->temporal_stale = false;
    return GF_OK;
}

// ---- run loops -----------------------------------------------------------------------------------
static int sweep_gx(const gf_ctx* ctx) {
    const int Vsh = ctx->Nx * ctx->Ny * (ctx->Nz / 2);
    const int block = (ctx->real_bytes == 4) ? sweep_block<float>(Vsh, ctx->block_override)
                                             : sweep_block<double>(Vsh, ctx->block_override);
    return (Vsh + block - 1) / block;
}

// exact F / theta of the current links (measure kernels: double, both parities) -> host scalars
static int exact_measure(gf_ctx* ctx, int gauge, double* F, double* stop) {
    int rc = enqueue_measure(ctx, gauge);
    if (rc) return rc;
    CU(cudaStreamSynchronize(ctx->stream));
    double theta = 0.0, tmax = 0.0;
    finish_measure(ctx, gauge, F, &theta, nullptr, &tmax);
    *stop = (gauge == GF_COULOMB) ? tmax : theta;
    return GF_OK;
}

/*
 * gf_run.  With the fused reductions (default) the odd half-sweep of a check sweep s
 * leaves, at no extra traffic, F(s) (every link touches exactly one odd site) and theta_odd(s), the odd
 * sites' share of theta(s); the even sites' share is what the even half-sweep of sweep s+1 sees before
 * it updates.  theta(s) >= theta_odd(s), so a check with theta_odd(s) >= eps cannot have converged and
 * costs nothing; only when theta_odd(s) < eps is the exact reduction (measure kernels) run, so the
 * stopping decision is the one a reduction after every check would take.  History entries carry
 * theta(s) = theta_odd(s) + theta_even(s), completed at the following check (or by the exact
 * reduction); the values returned in *out always come from the exact reduction of the final links.
 *
 * Per-slice Coulomb fixing (GF_FLAG_FREEZE_SLICES): the same bound is used slice by
 * slice.  A slice whose theta_odd,t(s) < eps triggers the exact reduction; every not yet stopped slice
 * with exact theta_t(s) < eps is stopped at sweep s: its flag in skip_dev makes its CTAs exit at once
 * in all later half-sweeps, and its exact slice sums stand in for the (no longer written) partials.
 */
int gf_run(gf_ctx* ctx, int gauge, int algo, double param, uint64_t seed, uint32_t first_sweep_index,
           int max_sweeps, double eps, int check_every, int reunit_every, gf_result* out, double* hist) {
    int rc = check_sweep_args(ctx, gauge, algo, param);
    if (rc) return rc;
    if (max_sweeps < 0 || check_every < 1 || reunit_every < 0) return fail(ctx, GF_EINVAL, "gf_run: bad loop arguments");
    rc = pre_sweep(ctx, gauge);
    if (rc) return rc;
    const bool fused = ctx->fused != 0;
    const bool coulomb = gauge == GF_COULOMB;
    const bool freeze = coulomb && (ctx->flags & GF_FLAG_FREEZE_SLICES);
    const int nd = coulomb ? 3 : 4;
    const int Nt = ctx->Nt;
    const int gx = sweep_gx(ctx);
    const double Vs = (double)ctx->Nx * ctx->Ny * ctx->Nz;
    double F = 0.0, stop = 0.0;
    bool have_exact = false, converged = false;

    // slices already stopped, with the exact slice sums (F terms, theta terms) they were stopped at
    std::vector<unsigned char> frozen((size_t)Nt, 0);
    std::vector<double> fz_F((size_t)Nt, 0.0), fz_th((size_t)Nt, 0.0);
    int n_frozen = 0;
    ctx->slice_sweeps.assign((size_t)Nt, 0);
    ctx->have_slice_sweeps = true;
    const unsigned char* skip = nullptr;
    if (freeze) {
        memset(ctx->skip_host, 0, (size_t)Nt);
        CU(cudaMemcpyAsync(ctx->skip_dev, ctx->skip_host, (size_t)Nt, cudaMemcpyHostToDevice, ctx->stream));
        skip = ctx->skip_dev;
    }
    // stopping quantity from per-slice sums of theta terms a[t] (+ b[t]): theta (Eq. (7)), or max_t theta_t
    auto stop_of = [&](const double* a, int sa, const double* b, int sb) {
        double tot = 0.0, tmax = 0.0;
        for (int t = 0; t < Nt; ++t) {
            const double v = frozen[(size_t)t] ? fz_th[(size_t)t]
                                               : a[(size_t)t * sa] + (b ? b[(size_t)t * sb] : 0.0);
            tot += v;
            if (v / (3.0 * Vs) > tmax) tmax = v / (3.0 * Vs);
        }
        return coulomb ? tmax : tot / (3.0 * (double)ctx->V);
    };
    // stop every running slice whose exact theta_t (slice_host, just reduced) is below eps
    auto apply_freeze = [&](int s_now) -> int {
        bool changed = false;
        for (int t = 0; t < Nt; ++t) {
            if (frozen[(size_t)t]) continue;
            if (ctx->slice_host[Nt + t] / (3.0 * Vs) < eps) {
                frozen[(size_t)t] = 1;
                fz_F[(size_t)t] = ctx->slice_host[t];
                fz_th[(size_t)t] = ctx->slice_host[Nt + t];
                ctx->slice_sweeps[(size_t)t] = s_now;
                ctx->skip_host[t] = 1;
                ++n_frozen;
                changed = true;
            }
        }
        if (changed)
            CU(cudaMemcpyAsync(ctx->skip_dev, ctx->skip_host, (size_t)Nt, cudaMemcpyHostToDevice, ctx->stream));
        return GF_OK;
    };

    // history entry still waiting for the even sites' share of theta:
    //   stage 1 = the next even half-sweep must produce it, stage 2 = produced, reduced at the next check
    int pend_stage = 0, pend_entry = -1;
    std::vector<double> pend_odd((size_t)Nt, 0.0);
    int s = 0, nh = 0, last_entry_sweep = -1;
    while (s < max_sweeps) {
        const bool check_now = ((s + 1) % check_every == 0) || (s + 1 == max_sweeps);
        const bool red_even = fused && pend_stage == 1;
        const uint32_t idx = first_sweep_index + (uint32_t)s;
        rc = launch_half(ctx, gauge, algo, param, seed, idx, 0, red_even ? ctx->red_part[0] : nullptr, skip);
        if (rc) return rc;
        if (red_even) pend_stage = 2;
        const bool reunit_now = reunit_every && (s + 1) % reunit_every == 0;
        rc = launch_half(ctx, gauge, algo, param, seed, idx, 1,
                         (fused && check_now && !reunit_now) ? ctx->red_part[1] : nullptr, skip);
        if (rc) return rc;
        ++s;
        if (reunit_now) {
            rc = gf_reunitarize(ctx);
            if (rc) return rc;
        }
        have_exact = false;
        if (!check_now) continue;
        if (!fused || reunit_now) {   // links were just reprojected: reduce what is stored now
            if (pend_stage == 2) {
                red_reduce_kernel<<<Nt, 128, 0, ctx->stream>>>(ctx->red_part[0], gx, ctx->red_dev);
                CU(cudaGetLastError());
                ++ctx->launches;
                CU(cudaMemcpyAsync(ctx->red_host, ctx->red_dev, (size_t)3 * Nt * sizeof(double),
                                   cudaMemcpyDeviceToHost, ctx->stream));
            }
            rc = exact_measure(ctx, gauge, &F, &stop);
            if (rc) return rc;
            if (pend_stage == 2 && hist)
                hist[3 * pend_entry + 2] = stop_of(pend_odd.data(), 1, ctx->red_host + 2, 3);
            pend_stage = 0;
            have_exact = true;
            if (freeze) {
                rc = apply_freeze(s);
                if (rc) return rc;
            }
        } else {
            red_reduce_kernel<<<Nt, 128, 0, ctx->stream>>>(ctx->red_part[1], gx, ctx->red_dev + 3 * Nt);
            CU(cudaGetLastError());
            ++ctx->launches;
            if (pend_stage == 2) {
                red_reduce_kernel<<<Nt, 128, 0, ctx->stream>>>(ctx->red_part[0], gx, ctx->red_dev);
                CU(cudaGetLastError());
                ++ctx->launches;
            }
            CU(cudaMemcpyAsync(ctx->red_host, ctx->red_dev, (size_t)6 * Nt * sizeof(double), cudaMemcpyDeviceToHost,
                               ctx->stream));
            CU(cudaStreamSynchronize(ctx->stream));
            const double* ev = ctx->red_host;            // [t][3]: even half-sweep of this or an earlier sweep
            const double* od = ctx->red_host + 3 * Nt;   // [t][3]: odd half-sweep of sweep s
            if (pend_stage == 2) {
                if (hist) hist[3 * pend_entry + 2] = stop_of(pend_odd.data(), 1, ev + 2, 3);
                pend_stage = 0;
            }
            double fs = 0.0;
            for (int t = 0; t < Nt; ++t) fs += frozen[(size_t)t] ? fz_F[(size_t)t] : od[3 * t];
            F = fs / (3.0 * nd * (double)ctx->V);
            stop = stop_of(od + 1, 3, nullptr, 0);   // lower bound of theta(s)
            bool need_exact = stop < eps;
            if (freeze)   // a running slice may have converged on its own
                for (int t = 0; t < Nt && !need_exact; ++t)
                    need_exact = !frozen[(size_t)t] && od[3 * t + 1] / (3.0 * Vs) < eps;
            if (need_exact) {
                rc = exact_measure(ctx, gauge, &F, &stop);
                if (rc) return rc;
                have_exact = true;
                if (freeze) {
                    rc = apply_freeze(s);
                    if (rc) return rc;
                }
            } else {
                for (int t = 0; t < Nt; ++t) pend_odd[(size_t)t] = od[3 * t + 1];
                pend_stage = 1;
                pend_entry = nh;
            }
        }
        if (hist) { hist[3 * nh] = (double)s; hist[3 * nh + 1] = F; hist[3 * nh + 2] = stop; }
        last_entry_sweep = s;
        ++nh;
        if (freeze ? (n_frozen == Nt) : (have_exact && stop < eps)) { converged = true; break; }
    }
    if (!have_exact) {
        rc = exact_measure(ctx, gauge, &F, &stop);
        if (rc) return rc;
        converged = freeze ? (n_frozen == Nt) : (stop < eps);
        if (hist && nh > 0 && last_entry_sweep == s) { hist[3 * (nh - 1) + 1] = F; hist[3 * (nh - 1) + 2] = stop; }
    }
    for (int t = 0; t < Nt; ++t)
        if (!frozen[(size_t)t]) ctx->slice_sweeps[(size_t)t] = s;
    if (coulomb && ctx->gtot) {
        rc = gf_coulomb_finalize(ctx);
        if (rc) return rc;
        CU(cudaStreamSynchronize(ctx->stream));
    }
    if (out) { out->sweeps = s; out->F = F; out->theta = stop; }
    return converged ? GF_OK : GF_NOT_CONVERGED;
}

int gf_get_slice_sweeps(gf_ctx* ctx, int* sweeps) {
    if (!ctx) return GF_EINVAL;
    if (!sweeps) return fail(ctx, GF_EINVAL, "gf_get_slice_sweeps: NULL pointer");
    if (!ctx->have_slice_sweeps) return fail(ctx, GF_ESTATE, "gf_get_slice_sweeps: no gf_run yet");
    for (int t = 0; t < ctx->Nt; ++t) sweeps[t] = ctx->slice_sweeps[(size_t)t];
    return GF_OK;
}

int gf_anneal(gf_ctx* ctx, int gauge, double T_hi, double T_lo, int n_steps, int n_micro, uint64_t seed,
              uint32_t first_sweep_index, uint32_t* next_sweep_index) {
    int rc = check_sweep_args(ctx, gauge, GF_SA, T_hi);
    if (rc) return rc;
    if (!(T_lo > 0.0) || n_steps < 0 || n_micro < 0) return fail(ctx, GF_EINVAL, "gf_anneal: bad schedule");
    rc = pre_sweep(ctx, gauge);
    if (rc) return rc;
    uint32_t idx = first_sweep_index;
    for (int k = 0; k < n_steps; ++k) {
        const double T = (n_steps <= 1) ? T_hi : T_hi - k * (T_hi - T_lo) / (n_steps - 1);
        for (int p = 0; p < 2; ++p) {
            rc = launch_half(ctx, gauge, GF_SA, T, seed, idx, p);
            if (rc) return rc;
        }
        ++idx;
        for (int m = 0; m < n_micro; ++m) {
            for (int p = 0; p < 2; ++p) {
                rc = launch_half(ctx, gauge, GF_MICRO, 0.0, seed, idx, p);
                if (rc) return rc;
            }
            ++idx;
        }
    }
    if (next_sweep_index) *next_sweep_index = idx;
    return GF_OK;
}

// ---- instrumentation -----------------------------------------------------------------------------
int gf_kernel_timing(gf_ctx* ctx, int enable) {
    if (!ctx) return GF_EINVAL;
    ctx->timing = enable != 0;
    return GF_OK;
}

int gf_kernel_time_ms(gf_ctx* ctx, double* total_ms, int* launches, int reset) {
    if (!ctx) return GF_EINVAL;
    CU(cudaStreamSynchronize(ctx->stream));
    double tot = 0.0;
    for (size_t k = 0; k + 1 < ctx->ev_used; k += 2) {
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, ctx->ev[k], ctx->ev[k + 1]));
        tot += ms;
    }
    if (total_ms) *total_ms = tot;
    if (launches) *launches = (int)(ctx->ev_used / 2);
    if (reset) ctx->ev_used = 0;
    return GF_OK;
}

int gf_launch_count(gf_ctx* ctx, int64_t* launches, int reset) {
    if (!ctx) return GF_EINVAL;
    if (launches) *launches = ctx->launches;
    if (reset) ctx->launches = 0;
    return GF_OK;
}

// tuning hook (not declared in gf.h): 0 = gf_run measures after every check with the measure kernels
int gf_debug_set_fused(gf_ctx* ctx, int fused) {
    if (!ctx) return GF_EINVAL;
    ctx->fused = fused != 0;
    return GF_OK;
}

// tuning hook (not declared in gf.h): CTA size of the half-sweep kernel, 0 = default
int gf_debug_set_block(gf_ctx* ctx, int block) {
    if (!ctx || block < 0 || (block & 31)) return GF_EINVAL;
    ctx->block_override = block;
    return GF_OK;
}

}  // extern "C"
