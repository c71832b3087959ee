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
#include "aux_su2.cuh"
#include "sweep.cuh"
#include "sweep_su2.cuh"
#include "wilson.cuh"

using namespace gf;

namespace gf {
// one explicit instantiation per translation unit sweep_<prec><recon>.cu
extern template cudaError_t launch_sweep<float, float, 18>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep<float, float, 12>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep<float, double, 18>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep<float, double, 12>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep<double, double, 18>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep<double, double, 12>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep_su2<float, float>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep_su2<float, double>(const SweepArgs&, int, bool, int, cudaStream_t);
extern template cudaError_t launch_sweep_su2<double, double>(const SweepArgs&, int, bool, int, cudaStream_t);
}  // namespace gf

struct gf_ctx {
    int Nx, Ny, Nz, Nt;
    int B;                  // gauge copies held by this context (gf_create_batch), 1 for gf_create
    int NS;                 // B * Nt: (copy, time-slice) pairs = grid.y of the per-site kernels
    int precision, recon;   // recon = reals stored per link: 18 | 12 (SU(3)), 4 (SU(2))
    int nc;                 // gauge group SU(nc): 3, or 2 with GF_FLAG_SU2
    unsigned flags;
    cudaStream_t stream;
    int64_t V, Vh;
    size_t real_bytes;      // 4 | 8
    char* links;            // device link store
    char* gtot;             // tracked transform (18 reals/site) or nullptr
    char* gapplied;         // snapshot of gtot taken when Coulomb sweeps start: the part already applied to the temporal links
    bool gapp_valid;        // the pending finalisation uses R = gtot gapplied^dag (false: gtot was the identity, R = gtot)
    std::vector<unsigned char> gtot_ident;   // per copy: gtot is still the identity set by reset_transform
    bool have_links;        // every copy has received links
    std::vector<unsigned char> copies_set;
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
    std::vector<unsigned char> slice_frozen;   // slices of the units the last run stopped (converged)
    bool have_slice_sweeps;
    // host<->device staging for gf_set_links / gf_get_*
    void* staging;
    size_t staging_bytes;
    int64_t device_bytes;
    int block_override;     // 0 = default CTA size
    int block_auto;         // the default: the largest CTA size that still gives every SM a few CTAs (auto_block)
    int pdl;                // half-sweeps launched with programmatic stream serialization (default 1)
    // kernel timing (gf_kernel_timing)
    bool timing;
    std::vector<cudaEvent_t> ev;   // pairs (start, stop)
    size_t ev_used;
    int64_t launches;       // kernels enqueued by this context (gf_launch_count)
    // t-sharding (gf_create_shard): this store holds the slices [t0, t0 + Nt) of a lattice of NtG
    // slices.  Host-side reduction arrays and the run loop's bookkeeping are indexed by GLOBAL slice (NSG = B * NtG
    // entries; a shard fills its own part, the comm's allreduce completes it); not sharded: NtG = Nt, t0 = 0.
    bool sharded;
    int NtG, t0, NSG;
    int64_t VG;
    char* links_dn;         // store holding slice t0 - 1 as its last slice (not sharded: links)
    int64_t Vh_dn;
    int Nt_dn;
    char* links_up;         // link store holding slice t0 + Nt as its first slice (not sharded: links)
    char* gtot_up;          // transform stores holding slice t0 + Nt as their first slice (not sharded: gtot / gapplied)
    char* gapp_up;
    int64_t Vh_up;
    bool attached;
    bool have_comm;
    gf_comm comm;
    std::vector<void*> ipc_opened;   // mappings opened by gf_shard_attach_ipc
    char err[512];
};

// CTA size of the half-sweep kernels when the caller sets none: the largest (128 threads for float storage and SU(2),
// 64 for double), except on lattices so small that a half-sweep of such CTAs would not give every SM one (float) or
// two (double) of them — then 32 threads.  Measured with the launches spread over all SMs (sweep_inst.cuh), us per
// half-sweep, largest CTA / 32 threads: 8^4 SP-12 3.5 / 3.3, DP-18 4.7 / 4.4; 12^4 SP-12 3.8 / 3.6, DP-18 7.5 / 6.4;
// 16^4 SP-12 5.3 / 6.4, SP-18 6.6 / 10.0, DP-18 11.4 / 13.8; larger lattices: the largest CTA by a growing margin.
// Counted on the WHOLE lattice (all copies, all time-slices of all t-shards), so a shard makes the choice of the
// unsharded context and its fused partial sums keep their order.
static int auto_block(const gf_ctx* c) {
    const bool dbl = c->nc == 3 && c->real_bytes == 8;
    const int maxb = dbl ? 64 : 128;
    const int64_t Vsh = (int64_t)c->Nx * c->Ny * (c->Nz / 2), units = (int64_t)c->B * c->NtG;
    const int64_t ctas = ((Vsh + maxb - 1) / maxb) * units;
    // thresholds calibrated on the 148 SMs of a B200 (one CTA per SM in float, 300 CTAs in double), scaled with the SM
    // count of the device the context lives on; the t-shards of one lattice must sit on devices of one kind for their
    // fused partial sums to keep the unsharded order (gf.h, "t-shards")
    int dev = 0, sms = 148;
    DevLimits lim;
    if (cudaGetDevice(&dev) == cudaSuccess && dev_limits(dev, lim) == cudaSuccess) sms = lim.sms;
    return ctas < (dbl ? (int64_t)300 * sms / 148 : (int64_t)sms) ? 32 : maxb;
}

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
// bytes of ONE gauge copy; the B copies of a context are contiguous
static int64_t link_store_bytes(const gf_ctx* c) { return (int64_t)8 * c->recon * c->real_bytes * c->Vh; }
static int64_t field_store_bytes(const gf_ctx* c) { return (int64_t)2 * (c->nc == 2 ? 4 : 18) * c->real_bytes * c->Vh; }
// reals per matrix in the host layout
static int64_t host_mat_elems(const gf_ctx* c) { return c->nc == 2 ? 8 : 18; }

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

int gf_num_colors(const gf_ctx* ctx) { return ctx ? ctx->nc : 0; }

int gf_create(gf_ctx** out, int Nx, int Ny, int Nz, int Nt, int precision, int recon, unsigned flags,
              void* cuda_stream) {
    return gf_create_batch(out, Nx, Ny, Nz, Nt, 1, precision, recon, flags, cuda_stream);
}

static int create_impl(gf_ctx** out, int Nx, int Ny, int Nz, int Nt, int n_copies, int precision, int recon,
                       unsigned flags, void* cuda_stream, int t0, int NtG);

int gf_create_batch(gf_ctx** out, int Nx, int Ny, int Nz, int Nt, int n_copies, int precision, int recon,
                    unsigned flags, void* cuda_stream) {
    return create_impl(out, Nx, Ny, Nz, Nt, n_copies, precision, recon, flags, cuda_stream, 0, Nt);
}

int gf_create_shard(gf_ctx** out, int Nx, int Ny, int Nz, int Nt_local, int t0, int Nt_global, int precision, int recon,
                    unsigned flags, void* cuda_stream) {
    if (!out) return GF_EINVAL;
    *out = nullptr;
    // even first slice and even extents: the 4-d colouring of the store is the global one
    if (t0 < 0 || (t0 & 1) || Nt_global < 2 || (Nt_global & 1) || Nt_local < 2 || t0 + Nt_local > Nt_global) return GF_EINVAL;
    if (flags & GF_FLAG_SU2) return GF_EINVAL;   // SU(3) only
    return create_impl(out, Nx, Ny, Nz, Nt_local, 1, precision, recon, flags, cuda_stream, t0, Nt_global);
}

static int create_impl(gf_ctx** out, int Nx, int Ny, int Nz, int Nt, int n_copies, int precision, int recon,
                       unsigned flags, void* cuda_stream, int t0, int NtG) {
    if (!out) return GF_EINVAL;
    *out = nullptr;
    if (n_copies < 1 || (int64_t)n_copies * Nt > 65535) return GF_EINVAL;   // grid.y = n_copies * Nt
    const int n[4] = {Nx, Ny, Nz, Nt};
    for (int k = 0; k < 4; ++k)
        if (n[k] < 2 || (n[k] & 1)) return GF_EINVAL;
    const double vol = (double)Nx * Ny * Nz * NtG;
    if (vol >= 4294967296.0) return GF_EINVAL;
    if (precision != GF_SP && precision != GF_DP && precision != GF_MP) return GF_EINVAL;
    if (recon != 18 && recon != 12) return GF_EINVAL;
    const int nc = (flags & GF_FLAG_SU2) ? 2 : 3;
    if (nc == 2) recon = 4;   // first row of the 2x2 matrix (csrc/su2.cuh)
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) return GF_ECUDA;   // no CPU fallback
    gf_ctx* ctx = new (std::nothrow) gf_ctx();
    if (!ctx) return GF_ENOMEM;
    ctx->Nx = Nx; ctx->Ny = Ny; ctx->Nz = Nz; ctx->Nt = Nt;
    ctx->B = n_copies; ctx->NS = n_copies * Nt;
    ctx->copies_set.assign((size_t)n_copies, 0);
    ctx->precision = precision; ctx->recon = recon; ctx->nc = nc; ctx->flags = flags;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->V = (int64_t)Nx * Ny * Nz * Nt;
    ctx->Vh = ctx->V / 2;
    ctx->real_bytes = (precision == GF_DP) ? 8 : 4;
    ctx->links = ctx->gtot = ctx->gapplied = nullptr;
    ctx->have_links = false; ctx->temporal_stale = false;
    ctx->gapp_valid = false;
    ctx->gtot_ident.assign((size_t)n_copies, 1);
    ctx->partial = nullptr; ctx->slice_dev = nullptr; ctx->slice_host = nullptr;
    ctx->red_part[0] = ctx->red_part[1] = nullptr; ctx->red_dev = nullptr; ctx->red_host = nullptr;
    ctx->fused = 1;
    ctx->skip_dev = nullptr; ctx->skip_host = nullptr; ctx->have_slice_sweeps = false;
    ctx->staging = nullptr; ctx->staging_bytes = 0;
    ctx->device_bytes = 0; ctx->block_override = 0; ctx->pdl = 1;
    ctx->timing = false; ctx->ev_used = 0; ctx->launches = 0;
    ctx->err[0] = 0;
    ctx->sharded = (NtG != Nt);
    ctx->NtG = NtG; ctx->t0 = t0; ctx->NSG = n_copies * NtG;
    ctx->VG = (int64_t)Nx * Ny * Nz * NtG;
    ctx->links_dn = nullptr; ctx->Vh_dn = ctx->Vh; ctx->Nt_dn = Nt;
    ctx->gtot_up = ctx->gapp_up = nullptr; ctx->links_up = nullptr; ctx->Vh_up = ctx->Vh;
    ctx->attached = !ctx->sharded;
    ctx->block_auto = auto_block(ctx);
    ctx->have_comm = false;
    memset(&ctx->comm, 0, sizeof(ctx->comm));

    const int B = n_copies, NS = n_copies * Nt, NSG = ctx->NSG;
    cudaError_t e = cudaMalloc((void**)&ctx->links, (size_t)(B * link_store_bytes(ctx)));
    if (e == cudaSuccess) ctx->device_bytes += B * link_store_bytes(ctx);
    if (e == cudaSuccess && (flags & GF_FLAG_TRACK_TRANSFORM)) {
        e = cudaMalloc((void**)&ctx->gtot, (size_t)(B * field_store_bytes(ctx)));
        if (e == cudaSuccess) ctx->device_bytes += B * field_store_bytes(ctx);
    }
    ctx->meas_block = 128;
    const int Vsh = Nx * Ny * (Nz / 2);
    ctx->meas_gx = (Vsh + ctx->meas_block - 1) / ctx->meas_block;
    const size_t npart = (size_t)ctx->meas_gx * NS * 2;
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->partial, npart * 2 * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->slice_dev, (size_t)2 * NS * sizeof(double));
    if (e == cudaSuccess && ctx->sharded && ctx->gtot) {   // a shard's neighbours map it: allocated once, never moved
        e = cudaMalloc((void**)&ctx->gapplied, (size_t)(B * field_store_bytes(ctx)));
        if (e == cudaSuccess) ctx->device_bytes += B * field_store_bytes(ctx);
    }
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->slice_host, (size_t)2 * NSG * sizeof(double));
    const size_t nred = (size_t)((Vsh + 31) / 32) * NS * 3;   // smallest CTA = 32 sites
    for (int k = 0; k < 2; ++k)
        if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->red_part[k], nred * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->red_dev, (size_t)6 * NS * sizeof(double));
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->red_host, (size_t)6 * NSG * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->skip_dev, (size_t)NS);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->skip_host, (size_t)NS);
    if (e != cudaSuccess) {
        const int code = (e == cudaErrorMemoryAllocation) ? GF_ENOMEM : GF_ECUDA;
        gf_destroy(ctx);
        cudaGetLastError();
        return code;
    }
    ctx->device_bytes += (int64_t)(npart * 2 + 2 * NS + 2 * nred + 6 * NS) * sizeof(double);
    if (!ctx->sharded) {   // the periodic wrap in t: the store is its own neighbour
        ctx->links_dn = ctx->links;
        ctx->links_up = ctx->links;
        ctx->gtot_up = ctx->gtot;
    }
    *out = ctx;
    return GF_OK;
}

int gf_destroy(gf_ctx* ctx) {
    if (!ctx) return GF_OK;
    cudaStreamSynchronize(ctx->stream);
    for (void* p : ctx->ipc_opened) cudaIpcCloseMemHandle(p);
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
        (const E*)(src), lbase, dims_of(ctx), (s0), (ns))
#define CONVERT_OUT(R, RECON, E, dst, s0, ns)                                                           \
    convert_out_kernel<E, R, RECON><<<(unsigned)(((ns) * 4 + 255) / 256), 256, 0, ctx->stream>>>(       \
        (E*)(dst), lbase, dims_of(ctx), (s0), (ns))

// the same for SU(2) contexts: E = host element type, storage type from the context
#define CONVERT2(KERN, E, hostp, s0, ns)                                                                  \
    do {                                                                                                  \
        const unsigned g_ = (unsigned)(((ns) * 4 + 255) / 256);                                           \
        if (ctx->real_bytes == 4) KERN<E, float><<<g_, 256, 0, ctx->stream>>>((hostp), lbase, dims_of(ctx), (s0), (ns)); \
        else KERN<E, double><<<g_, 256, 0, ctx->stream>>>((hostp), lbase, dims_of(ctx), (s0), (ns));      \
    } while (0)

static void convert_in_any(gf_ctx* ctx, char* lbase, const void* src, int elem_bytes, int64_t s0, int64_t ns) {
    if (ctx->nc == 2) {
        if (elem_bytes == 4) CONVERT2(convert_in2_kernel, float, (const float*)src, s0, ns);
        else CONVERT2(convert_in2_kernel, double, (const double*)src, s0, ns);
    } else {
        if (elem_bytes == 4) DISPATCH_RR(ctx, CONVERT_IN, float, src, s0, ns);
        else DISPATCH_RR(ctx, CONVERT_IN, double, src, s0, ns);
    }
}
static void convert_out_any(gf_ctx* ctx, const char* lbase, void* dst, int elem_bytes, int64_t s0, int64_t ns) {
    if (ctx->nc == 2) {
        if (elem_bytes == 4) CONVERT2(convert_out2_kernel, float, (float*)dst, s0, ns);
        else CONVERT2(convert_out2_kernel, double, (double*)dst, s0, ns);
    } else {
        if (elem_bytes == 4) DISPATCH_RR(ctx, CONVERT_OUT, float, dst, s0, ns);
        else DISPATCH_RR(ctx, CONVERT_OUT, double, dst, s0, ns);
    }
}

static int field_identity(gf_ctx* ctx, char* field) {
    const unsigned g = (unsigned)((2 * ctx->Vh + 255) / 256);
    if (ctx->nc == 2) {
        if (ctx->real_bytes == 4) field_identity2_kernel<float><<<g, 256, 0, ctx->stream>>>(field, ctx->Vh);
        else field_identity2_kernel<double><<<g, 256, 0, ctx->stream>>>(field, ctx->Vh);
    } else if (ctx->real_bytes == 4) field_identity_kernel<float><<<g, 256, 0, ctx->stream>>>(field, ctx->Vh);
    else field_identity_kernel<double><<<g, 256, 0, ctx->stream>>>(field, ctx->Vh);
    CU(cudaGetLastError());
    ++ctx->launches;
    return GF_OK;
}

// the accumulated transform of `copy` restarts at the identity (new links were just stored)
static int reset_transform(gf_ctx* ctx, int copy) {
    if (ctx->gtot) {
        int rc = field_identity(ctx, ctx->gtot + copy * field_store_bytes(ctx));
        if (rc) return rc;
    }
    ctx->gtot_ident[(size_t)copy] = 1;
    // gapplied is a snapshot taken at the next start of Coulomb sweeps (coulomb_begin); nothing to reset here.
    // A single lattice gives the memory back (a transform field is 1/4 of an 18-real link store).
    if (ctx->gapplied && ctx->B == 1 && !ctx->sharded) {
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->gapplied);
        ctx->gapplied = nullptr;
        ctx->gapp_valid = false;
        ctx->device_bytes -= field_store_bytes(ctx);
    }
    if (ctx->B == 1) ctx->temporal_stale = false;
    return GF_OK;
}

static int check_copy(gf_ctx* ctx, int copy, const char* who) {
    if (copy < 0 || copy >= ctx->B) return fail(ctx, GF_EINVAL, "%s: copy %d not in [0, %d)", who, copy, ctx->B);
    return GF_OK;
}
static int single_only(gf_ctx* ctx, const char* who) {
    if (ctx->B != 1) return fail(ctx, GF_ESTATE, "%s: context holds %d gauge copies, use the _copy / _batch call", who, ctx->B);
    return GF_OK;
}

int gf_num_copies(const gf_ctx* ctx) { return ctx ? ctx->B : 0; }

// ---- t-shards: neighbours and the caller's communicator ---------------------------
// stream-ordered barrier over all shards: everything enqueued so far on every shard's stream completes before
// anything enqueued afterwards on any of them starts (the caller's callback; nothing to do for one store)
static void shard_barrier(gf_ctx* ctx) {
    if (ctx->have_comm && ctx->comm.barrier) ctx->comm.barrier(ctx->comm.user);
}
// complete a host array indexed by global slice: every shard has filled its own entries and zeroed the others
static void shard_allreduce(gf_ctx* ctx, double* buf, int n) {
    if (ctx->have_comm && ctx->comm.allreduce_sum) ctx->comm.allreduce_sum(ctx->comm.user, buf, n);
}
static int need_attached(gf_ctx* ctx, const char* who) {
    if (!ctx->attached) return fail(ctx, GF_ESTATE, "%s: shard has no neighbours yet (gf_shard_attach)", who);
    return GF_OK;
}
static int not_on_shards(gf_ctx* ctx, const char* who) {
    if (ctx->sharded) return fail(ctx, GF_ESTATE, "%s: not available on a t-shard", who);
    return GF_OK;
}
static ShardDn shard_dn(const gf_ctx* ctx) {
    ShardDn sh;
    sh.links_dn = ctx->links_dn; sh.Vh_dn = ctx->Vh_dn; sh.Nt_dn = ctx->Nt_dn;
    sh.copy_bytes_dn = ctx->sharded ? 0 : (int64_t)8 * ctx->recon * ctx->real_bytes * ctx->Vh;
    return sh;
}

int gf_shard_set_comm(gf_ctx* ctx, const gf_comm* comm) {
    if (!ctx) return GF_EINVAL;
    ctx->have_comm = comm != nullptr;
    if (comm) ctx->comm = *comm;
    return GF_OK;
}

int gf_shard_info(const gf_ctx* ctx, int* t0, int* Nt_local, int* Nt_global) {
    if (!ctx) return GF_EINVAL;
    if (t0) *t0 = ctx->t0;
    if (Nt_local) *Nt_local = ctx->Nt;
    if (Nt_global) *Nt_global = ctx->NtG;
    return GF_OK;
}

// make a pointer of another device of this process usable from the current one
static int enable_peer_for(gf_ctx* ctx, const void* ptr) {
    cudaPointerAttributes at;
    CU(cudaPointerGetAttributes(&at, ptr));
    int dev = 0;
    CU(cudaGetDevice(&dev));
    if (at.type == cudaMemoryTypeDevice && at.device != dev) {
        int can = 0;
        CU(cudaDeviceCanAccessPeer(&can, dev, at.device));
        if (!can) return fail(ctx, GF_ECUDA, "gf_shard_attach: device %d cannot map device %d", dev, at.device);
        cudaError_t e = cudaDeviceEnablePeerAccess(at.device, 0);
        if (e == cudaErrorPeerAccessAlreadyEnabled) cudaGetLastError();
        else CU(e);
    }
    return GF_OK;
}

static int check_neighbour(gf_ctx* ctx, const gf_ctx* nb, int want_t0, const char* what) {
    if (!nb) return fail(ctx, GF_EINVAL, "gf_shard_attach: NULL %s", what);
    if (nb->Nx != ctx->Nx || nb->Ny != ctx->Ny || nb->Nz != ctx->Nz || nb->NtG != ctx->NtG || nb->precision != ctx->precision ||
        nb->recon != ctx->recon || nb->nc != ctx->nc || nb->B != ctx->B || (nb->gtot != nullptr) != (ctx->gtot != nullptr))
        return fail(ctx, GF_EINVAL, "gf_shard_attach: the %s does not match this shard (extents, precision, recon, flags)", what);
    if (nb->t0 != want_t0) return fail(ctx, GF_EINVAL, "gf_shard_attach: the %s starts at slice %d, expected %d", what, nb->t0, want_t0);
    return GF_OK;
}

int gf_shard_attach(gf_ctx* ctx, gf_ctx* below, gf_ctx* above) {
    if (!ctx) return GF_EINVAL;
    // below holds slice t0 - 1 as its last one, above holds slice t0 + Nt as its first one (periodic in NtG)
    int rc = check_neighbour(ctx, above, (ctx->t0 + ctx->Nt) % ctx->NtG, "shard above");
    if (rc) return rc;
    if (!below) return fail(ctx, GF_EINVAL, "gf_shard_attach: NULL shard below");
    rc = check_neighbour(ctx, below, below->t0, "shard below");
    if (rc) return rc;
    if ((below->t0 + below->Nt) % ctx->NtG != ctx->t0)
        return fail(ctx, GF_EINVAL, "gf_shard_attach: the shard below ends at slice %d, this one starts at %d", below->t0 + below->Nt, ctx->t0);
    // shards of one device are ordered by sharing a stream (a host-only barrier orders nothing between two streams)
    for (const gf_ctx* nb : {below, above}) {
        if (nb == ctx || nb->stream == ctx->stream || (ctx->have_comm && ctx->comm.barrier)) continue;
        cudaPointerAttributes at;
        int dev = 0;
        CU(cudaPointerGetAttributes(&at, nb->links));
        CU(cudaGetDevice(&dev));
        if (at.type == cudaMemoryTypeDevice && at.device == dev)
            return fail(ctx, GF_EINVAL, "gf_shard_attach: a neighbour on this device uses another stream and no communicator "
                                        "barrier is set (share one stream, or call gf_shard_set_comm first)");
    }
    rc = enable_peer_for(ctx, below->links);
    if (rc) return rc;
    ctx->links_dn = below->links; ctx->Vh_dn = below->Vh; ctx->Nt_dn = below->Nt;
    rc = enable_peer_for(ctx, above->links);
    if (rc) return rc;
    ctx->links_up = above->links; ctx->Vh_up = above->Vh;
    if (ctx->gtot) {
        rc = enable_peer_for(ctx, above->gtot);
        if (rc) return rc;
        ctx->gtot_up = above->gtot; ctx->gapp_up = above->gapplied; ctx->Vh_up = above->Vh;
    }
    ctx->attached = true;
    return GF_OK;
}

int gf_shard_export(gf_ctx* ctx, gf_shard_handle* h) {
    if (!ctx || !h) return GF_EINVAL;
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "gf_shard_handle holds 64-byte CUDA IPC handles");
    memset(h, 0, sizeof(*h));
    CU(cudaIpcGetMemHandle((cudaIpcMemHandle_t*)h->links, ctx->links));
    if (ctx->gtot) {
        CU(cudaIpcGetMemHandle((cudaIpcMemHandle_t*)h->gtot, ctx->gtot));
        if (ctx->gapplied) CU(cudaIpcGetMemHandle((cudaIpcMemHandle_t*)h->gapplied, ctx->gapplied));
        h->has_transform = 1;
    }
    h->t0 = ctx->t0; h->Nt_local = ctx->Nt;
    h->Nx = ctx->Nx; h->Ny = ctx->Ny; h->Nz = ctx->Nz; h->Nt_global = ctx->NtG;
    h->precision = ctx->precision; h->recon = ctx->recon;
    return GF_OK;
}

// mappings opened by gf_shard_attach_ipc are closed before a re-attach and when an attach fails part-way
static void close_ipc_mappings(gf_ctx* ctx) {
    for (void* q : ctx->ipc_opened) cudaIpcCloseMemHandle(q);
    ctx->ipc_opened.clear();
    if (ctx->sharded) {
        ctx->links_dn = ctx->links_up = nullptr;
        ctx->gtot_up = ctx->gapp_up = nullptr;
        ctx->attached = false;
    }
}
static int check_handle(gf_ctx* ctx, const gf_shard_handle* h, const char* what) {
    if (h->Nx != ctx->Nx || h->Ny != ctx->Ny || h->Nz != ctx->Nz || h->Nt_global != ctx->NtG || h->precision != ctx->precision ||
        h->recon != ctx->recon)
        return fail(ctx, GF_EINVAL, "gf_shard_attach_ipc: the %s (%dx%dx%d, Nt_global %d, precision %d, recon %d) does not match this "
                                    "shard (%dx%dx%d, Nt_global %d, precision %d, recon %d)", what, h->Nx, h->Ny, h->Nz, h->Nt_global,
                    h->precision, h->recon, ctx->Nx, ctx->Ny, ctx->Nz, ctx->NtG, ctx->precision, ctx->recon);
    if (h->Nt_local < 2 || h->t0 < 0 || h->t0 + h->Nt_local > ctx->NtG)
        return fail(ctx, GF_EINVAL, "gf_shard_attach_ipc: the %s holds slices [%d, %d) of %d", what, h->t0, h->t0 + h->Nt_local, ctx->NtG);
    if ((ctx->gtot != nullptr) != (h->has_transform != 0))
        return fail(ctx, GF_EINVAL, "gf_shard_attach_ipc: GF_FLAG_TRACK_TRANSFORM differs between this shard and the %s", what);
    static const unsigned char zero[64] = {0};
    if (memcmp(h->links, zero, 64) == 0 ||
        (h->has_transform && (memcmp(h->gtot, zero, 64) == 0 || memcmp(h->gapplied, zero, 64) == 0)))
        return fail(ctx, GF_EINVAL, "gf_shard_attach_ipc: the %s carries an empty store handle (not filled by gf_shard_export)", what);
    return GF_OK;
}

int gf_shard_attach_ipc(gf_ctx* ctx, const gf_shard_handle* below, const gf_shard_handle* above) {
    if (!ctx || !below || !above) return GF_EINVAL;
    if (!ctx->sharded) return fail(ctx, GF_ESTATE, "gf_shard_attach_ipc: not a t-shard (gf_create_shard)");
    // everything is checked before anything is mapped: a mismatched neighbour would be indexed with this shard's layout
    int rc = check_handle(ctx, below, "shard below");
    if (rc) return rc;
    rc = check_handle(ctx, above, "shard above");
    if (rc) return rc;
    if ((below->t0 + below->Nt_local) % ctx->NtG != ctx->t0 || above->t0 != (ctx->t0 + ctx->Nt) % ctx->NtG)
        return fail(ctx, GF_EINVAL, "gf_shard_attach_ipc: neighbours do not adjoin slices [%d, %d)", ctx->t0, ctx->t0 + ctx->Nt);
    CU(cudaStreamSynchronize(ctx->stream));
    close_ipc_mappings(ctx);   // a repeated attach starts from nothing (an open handle cannot be opened twice)
    const int64_t Vs2 = (int64_t)ctx->Nx * ctx->Ny * ctx->Nz / 2;
    auto open = [&](const unsigned char* h, char** out) -> cudaError_t {
        void* p = nullptr;
        cudaError_t e = cudaIpcOpenMemHandle(&p, *(const cudaIpcMemHandle_t*)h, cudaIpcMemLazyEnablePeerAccess);
        if (e == cudaSuccess) { ctx->ipc_opened.push_back(p); *out = (char*)p; }
        return e;
    };
    cudaError_t e = open(below->links, &ctx->links_dn);
    ctx->Nt_dn = below->Nt_local; ctx->Vh_dn = Vs2 * below->Nt_local;
    if (e == cudaSuccess) {
        if (memcmp(below->links, above->links, sizeof(below->links)) == 0)
            ctx->links_up = ctx->links_dn;   // two shards: the same store on both sides, mapped once
        else
            e = open(above->links, &ctx->links_up);
    }
    ctx->Vh_up = Vs2 * above->Nt_local;
    if (e == cudaSuccess && ctx->gtot) e = open(above->gtot, &ctx->gtot_up);
    if (e == cudaSuccess && ctx->gtot) e = open(above->gapplied, &ctx->gapp_up);
    if (e != cudaSuccess) {
        close_ipc_mappings(ctx);
        cudaGetLastError();
        return fail(ctx, GF_ECUDA, "gf_shard_attach_ipc: cudaIpcOpenMemHandle: %s (mappings opened so far were closed)", cudaGetErrorString(e));
    }
    ctx->attached = true;
    return GF_OK;
}

int gf_set_links_copy(gf_ctx* ctx, int copy, const void* links, int elem_bytes, int is_device) {
    if (!ctx) return GF_EINVAL;
    if (!links || (elem_bytes != 4 && elem_bytes != 8)) return fail(ctx, GF_EINVAL, "gf_set_links: bad arguments");
    int rc = check_copy(ctx, copy, "gf_set_links_copy");
    if (rc) return rc;
    if (ctx->B > 1 && ctx->temporal_stale && ctx->gtot) {   // the other copies keep their pending finalisation
        rc = gf_coulomb_finalize(ctx);
        if (rc) return rc;
    }
    char* lbase = ctx->links + copy * link_store_bytes(ctx);
    const int64_t link_elems = 4 * host_mat_elems(ctx);
    if (is_device) {
        convert_in_any(ctx, lbase, links, elem_bytes, 0, ctx->V);
        CU(cudaGetLastError());
        ++ctx->launches;
    } else {
        const int64_t chunk = ctx->V < STAGE_SITES ? ctx->V : STAGE_SITES;
        rc = ensure_staging(ctx, (size_t)(chunk * link_elems * elem_bytes));
        if (rc) return rc;
        for (int64_t s0 = 0; s0 < ctx->V; s0 += chunk) {
            const int64_t ns = (ctx->V - s0 < chunk) ? ctx->V - s0 : chunk;
            const char* src = (const char*)links + s0 * link_elems * elem_bytes;
            CU(cudaMemcpyAsync(ctx->staging, src, (size_t)(ns * link_elems * elem_bytes), cudaMemcpyHostToDevice,
                               ctx->stream));
            convert_in_any(ctx, lbase, ctx->staging, elem_bytes, s0, ns);
            CU(cudaGetLastError());
            ++ctx->launches;
        }
    }
    rc = reset_transform(ctx, copy);
    if (rc) return rc;
    CU(cudaStreamSynchronize(ctx->stream));
    shard_barrier(ctx);
    ctx->copies_set[(size_t)copy] = 1;
    ctx->have_links = true;
    for (int c = 0; c < ctx->B; ++c) ctx->have_links = ctx->have_links && ctx->copies_set[(size_t)c];
    return GF_OK;
}

// every copy of the context receives the same configuration
int gf_set_links(gf_ctx* ctx, const void* links, int elem_bytes, int is_device) {
    if (!ctx) return GF_EINVAL;
    int rc = gf_set_links_copy(ctx, 0, links, elem_bytes, is_device);
    if (rc) return rc;
    for (int c = 1; c < ctx->B; ++c) {
        CU(cudaMemcpyAsync(ctx->links + c * link_store_bytes(ctx), ctx->links, (size_t)link_store_bytes(ctx),
                           cudaMemcpyDeviceToDevice, ctx->stream));
        rc = reset_transform(ctx, c);
        if (rc) return rc;
        ctx->copies_set[(size_t)c] = 1;
    }
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->have_links = true;
    return GF_OK;
}

int gf_get_links_copy(gf_ctx* ctx, int copy, void* links, int elem_bytes, int is_device) {
    if (!ctx) return GF_EINVAL;
    if (!links || (elem_bytes != 4 && elem_bytes != 8)) return fail(ctx, GF_EINVAL, "gf_get_links: bad arguments");
    int rc = check_copy(ctx, copy, "gf_get_links_copy");
    if (rc) return rc;
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_get_links: no links set");
    if (ctx->temporal_stale && ctx->gtot) {
        rc = gf_coulomb_finalize(ctx);
        if (rc) return rc;
    }
    const char* lbase = ctx->links + copy * link_store_bytes(ctx);
    const int64_t link_elems = 4 * host_mat_elems(ctx);
    if (is_device) {
        convert_out_any(ctx, lbase, links, elem_bytes, 0, ctx->V);
        CU(cudaGetLastError());
        ++ctx->launches;
    } else {
        const int64_t chunk = ctx->V < STAGE_SITES ? ctx->V : STAGE_SITES;
        rc = ensure_staging(ctx, (size_t)(chunk * link_elems * elem_bytes));
        if (rc) return rc;
        for (int64_t s0 = 0; s0 < ctx->V; s0 += chunk) {
            const int64_t ns = (ctx->V - s0 < chunk) ? ctx->V - s0 : chunk;
            char* dst = (char*)links + s0 * link_elems * elem_bytes;
            convert_out_any(ctx, lbase, ctx->staging, elem_bytes, s0, ns);
            CU(cudaGetLastError());
            ++ctx->launches;
            CU(cudaMemcpyAsync(dst, ctx->staging, (size_t)(ns * link_elems * elem_bytes), cudaMemcpyDeviceToHost,
                               ctx->stream));
        }
    }
    CU(cudaStreamSynchronize(ctx->stream));
    return GF_OK;
}

int gf_get_links(gf_ctx* ctx, void* links, int elem_bytes, int is_device) {
    if (!ctx) return GF_EINVAL;
    int rc = single_only(ctx, "gf_get_links");
    if (rc) return rc;
    return gf_get_links_copy(ctx, 0, links, elem_bytes, is_device);
}

int gf_get_gauge_transform_copy(gf_ctx* ctx, int copy, void* g, int elem_bytes, int is_device) {
    if (!ctx) return GF_EINVAL;
    if (!g || (elem_bytes != 4 && elem_bytes != 8)) return fail(ctx, GF_EINVAL, "gf_get_gauge_transform: bad arguments");
    int rc = check_copy(ctx, copy, "gf_get_gauge_transform_copy");
    if (rc) return rc;
    if (!ctx->gtot) return fail(ctx, GF_ESTATE, "gf_get_gauge_transform: context created without GF_FLAG_TRACK_TRANSFORM");
    const char* fbase = ctx->gtot + copy * field_store_bytes(ctx);
    const int64_t me = host_mat_elems(ctx);
    const int64_t chunk = is_device ? ctx->V : (ctx->V < 4 * STAGE_SITES ? ctx->V : 4 * STAGE_SITES);
    if (!is_device) {
        rc = ensure_staging(ctx, (size_t)(chunk * me * elem_bytes));
        if (rc) return rc;
    }
    for (int64_t s0 = 0; s0 < ctx->V; s0 += chunk) {
        const int64_t ns = (ctx->V - s0 < chunk) ? ctx->V - s0 : chunk;
        void* dst = is_device ? (void*)((char*)g + s0 * me * elem_bytes) : ctx->staging;
        const unsigned grid = (unsigned)((ns + 255) / 256);
#define FIELD_OUT(KERN)                                                                                              \
        if (ctx->real_bytes == 4) {                                                                                  \
            if (elem_bytes == 4) KERN<float, float><<<grid, 256, 0, ctx->stream>>>((float*)dst, fbase, dims_of(ctx), s0, ns);   \
            else KERN<double, float><<<grid, 256, 0, ctx->stream>>>((double*)dst, fbase, dims_of(ctx), s0, ns);       \
        } else {                                                                                                     \
            if (elem_bytes == 4) KERN<float, double><<<grid, 256, 0, ctx->stream>>>((float*)dst, fbase, dims_of(ctx), s0, ns);  \
            else KERN<double, double><<<grid, 256, 0, ctx->stream>>>((double*)dst, fbase, dims_of(ctx), s0, ns);      \
        }
        if (ctx->nc == 2) { FIELD_OUT(field_out2_kernel) } else { FIELD_OUT(field_out_kernel) }
#undef FIELD_OUT
        CU(cudaGetLastError());
        ++ctx->launches;
        if (!is_device)
            CU(cudaMemcpyAsync((char*)g + s0 * me * elem_bytes, ctx->staging, (size_t)(ns * me * elem_bytes),
                               cudaMemcpyDeviceToHost, ctx->stream));
    }
    CU(cudaStreamSynchronize(ctx->stream));
    return GF_OK;
}

int gf_get_gauge_transform(gf_ctx* ctx, void* g, int elem_bytes, int is_device) {
    if (!ctx) return GF_EINVAL;
    int rc = single_only(ctx, "gf_get_gauge_transform");
    if (rc) return rc;
    return gf_get_gauge_transform_copy(ctx, 0, g, elem_bytes, is_device);
}

// ---- sweeps ----------------------------------------------------------------------------------
static int check_sweep_args(gf_ctx* ctx, int gauge, int algo, double param) {
    if (!ctx) return GF_EINVAL;
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "no links set (call gf_set_links first)");
    if (!ctx->attached) return fail(ctx, GF_ESTATE, "shard has no neighbours yet (gf_shard_attach)");
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
    a.ncopies = ctx->B;
    a.copy_links_bytes = link_store_bytes(ctx);
    a.copy_gtot_bytes = field_store_bytes(ctx);
    a.rcp_nzh = fast_div_rcp(ctx->Nz / 2);
    a.rcp_ny = fast_div_rcp(ctx->Ny);
    a.pdl = ctx->pdl;
    a.links_dn = ctx->links_dn; a.Vh_dn = ctx->Vh_dn; a.Nt_dn = ctx->Nt_dn; a.t_off = ctx->t0;
    a.copy_links_bytes_dn = ctx->sharded ? 0 : link_store_bytes(ctx);
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
    const int blk = ctx->block_override ? ctx->block_override : ctx->block_auto;
    if (ctx->nc == 2) {
        e = (ctx->precision == GF_DP)   ? launch_sweep_su2<double, double>(a, gauge, track, blk, ctx->stream)
            : (ctx->precision == GF_MP) ? launch_sweep_su2<float, double>(a, gauge, track, blk, ctx->stream)
                                        : launch_sweep_su2<float, float>(a, gauge, track, blk, ctx->stream);
    } else if (ctx->precision == GF_DP) {
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
    // t-shards: the next half-sweep of a neighbour touches the boundary links this one wrote;
    // Coulomb sweeps touch spatial links only and need nothing
    if (gauge != GF_COULOMB) shard_barrier(ctx);
    return GF_OK;
}

// Coulomb sweeps are about to start on temporal links that are up to date: whatever g(x) has accumulated so far
// (Landau / MAG sweeps, gf_random_gauge) has been applied to U_0 already, so the finalisation that follows must
// apply only what the Coulomb sweeps add, R = g_now g_start^dag.  Snapshot g_start (nothing to do while every
// copy's g is still the identity of gf_set_links).
static int coulomb_begin(gf_ctx* ctx) {
    bool all_ident = true;
    for (unsigned char f : ctx->gtot_ident) all_ident = all_ident && f;
    if (all_ident) {
        ctx->gapp_valid = false;
    } else {
        if (!ctx->gapplied) {
            CU(cudaMalloc((void**)&ctx->gapplied, (size_t)(ctx->B * field_store_bytes(ctx))));
            ctx->device_bytes += ctx->B * field_store_bytes(ctx);
        }
        CU(cudaMemcpyAsync(ctx->gapplied, ctx->gtot, (size_t)(ctx->B * field_store_bytes(ctx)), cudaMemcpyDeviceToDevice,
                           ctx->stream));
        ctx->gapp_valid = true;
    }
    ctx->temporal_stale = true;
    return GF_OK;
}

static void transform_changed(gf_ctx* ctx) {
    if (ctx->gtot) ctx->gtot_ident.assign((size_t)ctx->B, 0);
}

static int pre_sweep(gf_ctx* ctx, int gauge) {
    int rc = GF_OK;
    if (gauge == GF_COULOMB) {
        if (ctx->gtot && !ctx->temporal_stale) rc = coulomb_begin(ctx);
    } else if (ctx->temporal_stale) {
        rc = gf_coulomb_finalize(ctx);
    }
    transform_changed(ctx);
    return rc;
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
        dim3 grid((unsigned)(2 * ctx->meas_gx), (unsigned)ctx->NS);                                        \
        const int64_t cb_ = link_store_bytes(ctx);                                                         \
        if ((gauge_) == GF_LANDAU)                                                                         \
            measure_kernel<R, RECON, GAUGE_LANDAU><<<grid, ctx->meas_block, 0, ctx->stream>>>(ctx->links, dims_of(ctx), ctx->partial, cb_, shard_dn(ctx), eq16_); \
        else if ((gauge_) == GF_COULOMB)                                                                   \
            measure_kernel<R, RECON, GAUGE_COULOMB><<<grid, ctx->meas_block, 0, ctx->stream>>>(ctx->links, dims_of(ctx), ctx->partial, cb_, shard_dn(ctx), eq16_); \
        else                                                                                               \
            measure_kernel<R, RECON, GAUGE_MAG><<<grid, ctx->meas_block, 0, ctx->stream>>>(ctx->links, dims_of(ctx), ctx->partial, cb_, shard_dn(ctx), eq16_); \
    } while (0)

// enqueue the reduction and the copy of the 2*Nt slice sums to pinned host memory
#define MEASURE2(R, gauge_)                                                                                \
    do {                                                                                                   \
        dim3 grid((unsigned)(2 * ctx->meas_gx), (unsigned)ctx->NS);                                        \
        const int64_t cb_ = link_store_bytes(ctx);                                                         \
        if ((gauge_) == GF_LANDAU)                                                                         \
            measure2_kernel<R, GAUGE_LANDAU><<<grid, ctx->meas_block, 0, ctx->stream>>>(ctx->links, dims_of(ctx), ctx->partial, cb_); \
        else if ((gauge_) == GF_COULOMB)                                                                   \
            measure2_kernel<R, GAUGE_COULOMB><<<grid, ctx->meas_block, 0, ctx->stream>>>(ctx->links, dims_of(ctx), ctx->partial, cb_); \
        else                                                                                               \
            measure2_kernel<R, GAUGE_MAG><<<grid, ctx->meas_block, 0, ctx->stream>>>(ctx->links, dims_of(ctx), ctx->partial, cb_); \
    } while (0)

static int enqueue_measure(gf_ctx* ctx, int gauge, int eq16_ = 0) {
    shard_barrier(ctx);   // the first slice reads the neighbour's last one
    if (ctx->nc == 2) {
        if (ctx->real_bytes == 4) MEASURE2(float, gauge);
        else MEASURE2(double, gauge);
    } else
        DISPATCH_RR(ctx, MEASURE, gauge);
    CU(cudaGetLastError());
    slice_reduce_kernel<<<ctx->NS, 128, 0, ctx->stream>>>(ctx->partial, 2 * ctx->meas_gx, ctx->NS, ctx->slice_dev);
    CU(cudaGetLastError());
    ctx->launches += 2;
    // slice_host = [F terms of the NSG global slices][theta terms of the NSG global slices]
    if (ctx->sharded) {
        memset(ctx->slice_host, 0, (size_t)2 * ctx->NSG * sizeof(double));
        CU(cudaMemcpyAsync(ctx->slice_host + ctx->t0, ctx->slice_dev, (size_t)ctx->NS * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaMemcpyAsync(ctx->slice_host + ctx->NSG + ctx->t0, ctx->slice_dev + ctx->NS, (size_t)ctx->NS * sizeof(double),
                           cudaMemcpyDeviceToHost, ctx->stream));
    } else {
        CU(cudaMemcpyAsync(ctx->slice_host, ctx->slice_dev, (size_t)2 * ctx->NS * sizeof(double), cudaMemcpyDeviceToHost,
                           ctx->stream));
    }
    return GF_OK;
}
// wait for enqueue_measure's copies; t-shards: complete the global slice sums (every shard holds all of them and sums
// them in slice order, so F, theta and every stopping decision are those of the unsharded lattice, bit for bit)
static int finish_enqueued_measure(gf_ctx* ctx) {
    CU(cudaStreamSynchronize(ctx->stream));
    if (ctx->sharded) shard_allreduce(ctx, ctx->slice_host, 2 * ctx->NSG);
    return GF_OK;
}

// after a stream sync: normalise (Eqs. (4), (7), (11)) the slice sums of gauge copy c in a fixed order
static void finish_measure(const gf_ctx* ctx, int gauge, int c, double* F, double* theta, double* theta_slice,
                           double* theta_max) {
    const int nd = (gauge == GF_COULOMB) ? 3 : 4;
    const double ncd = (double)ctx->nc;   // N_c of Eqs. (4), (7), (11)
    const double Vs = (double)ctx->Nx * ctx->Ny * ctx->Nz;
    const double* fs_ = ctx->slice_host + (size_t)c * ctx->NtG;
    const double* th_ = ctx->slice_host + (size_t)ctx->NSG + (size_t)c * ctx->NtG;
    double fs = 0.0, ths = 0.0, tmax = 0.0;
    for (int t = 0; t < ctx->NtG; ++t) {
        fs += fs_[t];
        ths += th_[t];
        const double th_t = th_[t] / (ncd * Vs);
        if (theta_slice) theta_slice[t] = th_t;
        if (th_t > tmax) tmax = th_t;
    }
    if (F) *F = fs / (ncd * nd * (double)ctx->VG);
    if (theta) *theta = ths / (ncd * (double)ctx->VG);
    if (theta_max) *theta_max = tmax;
}

int gf_measure_batch(gf_ctx* ctx, int gauge, double* F, double* theta, double* theta_slice) {
    if (!ctx) return GF_EINVAL;
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_measure: no links set");
    if (gauge < GF_LANDAU || gauge > GF_MAG) return fail(ctx, GF_EINVAL, "unknown gauge %d", gauge);
    if (gauge != GF_COULOMB && ctx->temporal_stale) {
        int rc = gf_coulomb_finalize(ctx);
        if (rc) return rc;
    }
    int rc = need_attached(ctx, "gf_measure");
    if (rc) return rc;
    rc = enqueue_measure(ctx, gauge);
    if (rc) return rc;
    rc = finish_enqueued_measure(ctx);
    if (rc) return rc;
    for (int c = 0; c < ctx->B; ++c)
        finish_measure(ctx, gauge, c, F ? F + c : nullptr, theta ? theta + c : nullptr,
                       theta_slice ? theta_slice + (size_t)c * ctx->NtG : nullptr, nullptr);
    return GF_OK;
}

int gf_measure_mag_eq16(gf_ctx* ctx, double* theta_eq16) {
    if (!ctx) return GF_EINVAL;
    if (!theta_eq16) return fail(ctx, GF_EINVAL, "gf_measure_mag_eq16: NULL pointer");
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_measure_mag_eq16: no links set");
    if (ctx->nc != 3) return fail(ctx, GF_ESTATE, "gf_measure_mag_eq16: N_c = 2 has one subgroup, gf_measure's theta is Eq. (13)");
    int rc = need_attached(ctx, "gf_measure_mag_eq16");
    if (rc) return rc;
    if (ctx->temporal_stale) {
        rc = gf_coulomb_finalize(ctx);
        if (rc) return rc;
    }
    rc = enqueue_measure(ctx, GF_MAG, 1);
    if (rc) return rc;
    rc = finish_enqueued_measure(ctx);
    if (rc) return rc;
    for (int c = 0; c < ctx->B; ++c) finish_measure(ctx, GF_MAG, c, nullptr, theta_eq16 + c, nullptr, nullptr);
    return GF_OK;
}

int gf_measure(gf_ctx* ctx, int gauge, double* F, double* theta, double* theta_slice) {
    if (!ctx) return GF_EINVAL;
    int rc = single_only(ctx, "gf_measure");
    if (rc) return rc;
    return gf_measure_batch(ctx, gauge, F, theta, theta_slice);
}

// ---- reunitarisation -----------------------------------------------------------------------------
#define REUNIT_LINKS(R, RECON, dummy)                                                                       \
    reunit_kernel<R, RECON><<<dim3((unsigned)((8 * ctx->Vh + 255) / 256), (unsigned)ctx->B), 256, 0, ctx->stream>>>( \
        ctx->links, ctx->Vh, 8, link_store_bytes(ctx))

int gf_reunitarize(gf_ctx* ctx) {
    if (!ctx) return GF_EINVAL;
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_reunitarize: no links set");
    if (ctx->nc == 2) {
        const dim3 g8((unsigned)((8 * ctx->Vh + 255) / 256), (unsigned)ctx->B), g2((unsigned)((2 * ctx->Vh + 255) / 256), (unsigned)ctx->B);
        if (ctx->real_bytes == 4) reunit2_kernel<float><<<g8, 256, 0, ctx->stream>>>(ctx->links, ctx->Vh, 8, link_store_bytes(ctx));
        else reunit2_kernel<double><<<g8, 256, 0, ctx->stream>>>(ctx->links, ctx->Vh, 8, link_store_bytes(ctx));
        CU(cudaGetLastError());
        ++ctx->launches;
        if (ctx->gtot) {
            if (ctx->real_bytes == 4) reunit2_kernel<float><<<g2, 256, 0, ctx->stream>>>(ctx->gtot, ctx->Vh, 2, field_store_bytes(ctx));
            else reunit2_kernel<double><<<g2, 256, 0, ctx->stream>>>(ctx->gtot, ctx->Vh, 2, field_store_bytes(ctx));
            CU(cudaGetLastError());
            ++ctx->launches;
        }
        return GF_OK;
    }
    DISPATCH_RR(ctx, REUNIT_LINKS, 0);
    CU(cudaGetLastError());
    ++ctx->launches;
    if (ctx->gtot) {
        const dim3 g((unsigned)((2 * ctx->Vh + 255) / 256), (unsigned)ctx->B);
        if (ctx->real_bytes == 4) reunit_kernel<float, 18><<<g, 256, 0, ctx->stream>>>(ctx->gtot, ctx->Vh, 2, field_store_bytes(ctx));
        else reunit_kernel<double, 18><<<g, 256, 0, ctx->stream>>>(ctx->gtot, ctx->Vh, 2, field_store_bytes(ctx));
        CU(cudaGetLastError());
        ++ctx->launches;
    }
    shard_barrier(ctx);   // the neighbour above reads this store's last slice in its next half-sweep
    return GF_OK;
}

// ---- Coulomb finalisation ------------------------------------------------------------------------
#define FINALIZE(R, RECON, dummy)                                                                           \
    coulomb_finalize_kernel<R, RECON><<<dim3((unsigned)((2 * ctx->Vh + 127) / 128), (unsigned)ctx->B), 128, 0, ctx->stream>>>( \
        ctx->links, ctx->gtot, gapp, dims_of(ctx), link_store_bytes(ctx), field_store_bytes(ctx), up)

int gf_coulomb_finalize(gf_ctx* ctx) {
    if (!ctx) return GF_EINVAL;
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_coulomb_finalize: no links set");
    if (!ctx->gtot) return fail(ctx, GF_ESTATE, "gf_coulomb_finalize: context created without GF_FLAG_TRACK_TRANSFORM");
    if (!ctx->temporal_stale) return GF_OK;
    const char* gapp = ctx->gapp_valid ? ctx->gapplied : nullptr;   // the g(x) the Coulomb sweeps started from
    int rc_att = need_attached(ctx, "gf_coulomb_finalize");
    if (rc_att) return rc_att;
    // g(x + t_hat) of the last slice: the first slice of the store above (t-shards; every shard makes the same calls,
    // so gapp_valid agrees between them), else this store (periodic wrap)
    ShardUp up;
    up.gtot_up = ctx->sharded ? ctx->gtot_up : ctx->gtot;
    up.gapp_up = ctx->sharded ? (ctx->gapp_valid ? ctx->gapp_up : nullptr) : gapp;
    up.Vh_up = ctx->sharded ? ctx->Vh_up : ctx->Vh;
    up.copy_bytes_up = ctx->sharded ? 0 : field_store_bytes(ctx);
    shard_barrier(ctx);   // the sweeps of the shard above are complete
    if (ctx->nc == 2) {
        const dim3 g((unsigned)((2 * ctx->Vh + 127) / 128), (unsigned)ctx->B);
        if (ctx->real_bytes == 4)
            coulomb_finalize2_kernel<float><<<g, 128, 0, ctx->stream>>>(ctx->links, ctx->gtot, gapp, dims_of(ctx),
                                                                        link_store_bytes(ctx), field_store_bytes(ctx));
        else
            coulomb_finalize2_kernel<double><<<g, 128, 0, ctx->stream>>>(ctx->links, ctx->gtot, gapp, dims_of(ctx),
                                                                         link_store_bytes(ctx), field_store_bytes(ctx));
    } else
        DISPATCH_RR(ctx, FINALIZE, 0);
    CU(cudaGetLastError());
    ++ctx->launches;
    ctx->temporal_stale = false;   // the next start of Coulomb sweeps takes a new snapshot (coulomb_begin)
    shard_barrier(ctx);            // the shard below reads g(x) of this store's first slice: not to be changed before it has
    return GF_OK;
}

// ---- run loops -----------------------------------------------------------------------------------
// sweeps of heatbath / microcanonical / stochastic-relaxation type on 12-real contexts are reprojected at least this
// often (see the comment above anneal_impl and DESIGN.md §7)
static const int GF_RECON12_REUNIT = 16;

// CTAs per (copy, time-slice) of a half-sweep with the rule `algo` (the stochastic float kernels use smaller CTAs)
static int sweep_gx(const gf_ctx* ctx, int algo) {
    const int Vsh = ctx->Nx * ctx->Ny * (ctx->Nz / 2);
    const int blk = ctx->block_override ? ctx->block_override : ctx->block_auto;
    const bool stoch = (algo == GF_SR || algo == GF_SA);
    const int block = (ctx->nc == 2)              ? sweep_su2_block(Vsh, blk)
                      : (ctx->precision == GF_SP) ? sweep_block<float, float>(Vsh, blk, stoch)
                      : (ctx->precision == GF_MP) ? sweep_block<float, double>(Vsh, blk, stoch)
                                                  : sweep_block<double, double>(Vsh, blk, stoch);
    return (Vsh + block - 1) / block;
}

// exact F / theta terms of the current links (measure kernels: double, both parities) -> slice_host
static int exact_measure(gf_ctx* ctx, int gauge) {
    int rc = enqueue_measure(ctx, gauge);
    if (rc) return rc;
    return finish_enqueued_measure(ctx);
}

/*
 * run_impl — Alg. 1's outer loop for every gauge copy of the context at once.
 *
 * Units.  The lattice sites are grouped into independent optimisation problems ("units"), each with
 * its own stopping quantity: a gauge copy (Landau, MAG: theta of Eq. (7)/(16); Coulomb: max_t theta_t),
 * or, for Coulomb with GF_FLAG_FREEZE_SLICES, a single time-slice of a copy.  A
 * unit is stopped ("frozen") at the first check at which its exact stopping quantity is < eps: the
 * flags of its slices in skip_dev make its CTAs exit at once in all later half-sweeps, and its exact
 * slice sums stand in for the partials those CTAs no longer write.  The loop ends when every unit is
 * frozen or after max_sweeps.  With one copy and one unit this is the plain "sweep until theta < eps".
 *
 * Fused reductions (default).  The odd half-sweep of a check sweep s leaves, at no
 * extra traffic, F(s) (every link touches exactly one odd site) and theta_odd(s), the odd sites' share
 * of theta(s); the even sites' share is what the even half-sweep of sweep s+1 sees before it updates.
 * theta(s) >= theta_odd(s), so a unit with theta_odd(s) >= eps cannot have converged and its check
 * costs nothing; only when some running unit has theta_odd(s) < eps is the exact reduction (measure
 * kernels) run, so every stopping decision is the one a reduction after every check would take.
 * History entries carry theta(s) = theta_odd(s) + theta_even(s), completed at the following check (or
 * by the exact reduction); the values returned in out[] always come from the exact reduction of the
 * final links.
 *
 * skip_slice: NULL, or [B*Nt] flags of slices that are not to be touched by this run (gf_fix: units that
 * converged in an earlier stage; a unit is left alone when all of its slices are flagged); they are
 * reported with sweeps = 0.  ctx->slice_frozen receives the slices of the units stopped by this run.
 * hist: NULL or [checks][B][3] = (sweep, F, stopping quantity).
 */
static int run_impl(gf_ctx* ctx, int gauge, int algo, double param, uint64_t seed, uint32_t first_sweep_index,
                    int max_sweeps, double eps, int check_every, int reunit_every, const unsigned char* skip_slice,
                    gf_result* out, double* hist, bool* all_converged) {
    int rc = check_sweep_args(ctx, gauge, algo, param);
    if (rc) return rc;
    if (max_sweeps < 0 || check_every < 1 || reunit_every < 0) return fail(ctx, GF_EINVAL, "gf_run: bad loop arguments");
    rc = pre_sweep(ctx, gauge);
    if (rc) return rc;
    if (algo != GF_OR && ctx->recon == 12 && (reunit_every == 0 || reunit_every > GF_RECON12_REUNIT))
        reunit_every = GF_RECON12_REUNIT;
    const bool fused = ctx->fused != 0;
    const bool coulomb = gauge == GF_COULOMB;
    const bool per_slice = coulomb && (ctx->flags & GF_FLAG_FREEZE_SLICES);
    const int nd = coulomb ? 3 : 4;
    // host-side bookkeeping is per GLOBAL slice (t-shards: NSG = NtG slices of which this store holds [t0, t0 + Nt);
    // otherwise NSG = NS = B * Nt); kernels and device arrays are per local slice
    const int Nt = ctx->NtG, B = ctx->B, NS = ctx->NSG, NSloc = ctx->NS, goff = ctx->t0;
    const int nunits = per_slice ? NS : B, uspan = per_slice ? 1 : Nt;   // unit u = slices [u*uspan, (u+1)*uspan)
    const int gx = sweep_gx(ctx, algo);
    const double Vs = (double)ctx->Nx * ctx->Ny * ctx->Nz;
    const double ncd = (double)ctx->nc;
    bool have_exact = false;

    // frozen slices, with the exact slice sums (F terms, theta terms) they were stopped at
    std::vector<unsigned char> frozen((size_t)NS, 0), unit_frozen((size_t)nunits, 0);
    std::vector<double> fz_F((size_t)NS, 0.0), fz_th((size_t)NS, 0.0);
    std::vector<double> Fc((size_t)B, 0.0), stopc((size_t)B, 0.0);
    int n_frozen = 0;
    ctx->slice_sweeps.assign((size_t)NS, 0);
    ctx->have_slice_sweeps = true;
    const bool use_skip = nunits > 1 || skip_slice;
    const unsigned char* skip = use_skip ? ctx->skip_dev : nullptr;
    if (use_skip) memset(ctx->skip_host, 0, (size_t)NSloc);
    auto skip_set = [&](int sl) {   // global slice -> this store's flag array
        if (sl - goff >= 0 && sl - goff < NSloc) ctx->skip_host[sl - goff] = 1;
    };

    // stopping quantity of slices [lo, hi) from per-slice sums of theta terms val(s): Eq. (7) over the
    // slices' sites, or max_t theta_t for Coulomb
    auto stop_range = [&](int lo, int hi, auto val) {
        double tot = 0.0, tmax = 0.0;
        for (int sl = lo; sl < hi; ++sl) {
            const double v = frozen[(size_t)sl] ? fz_th[(size_t)sl] : val(sl);
            tot += v;
            if (v / (ncd * Vs) > tmax) tmax = v / (ncd * Vs);
        }
        return coulomb ? tmax : tot / (ncd * (double)ctx->VG);
    };
    auto freeze_unit = [&](int u, int s_now) {
        unit_frozen[(size_t)u] = 1;
        ++n_frozen;
        for (int sl = u * uspan; sl < (u + 1) * uspan; ++sl) {
            frozen[(size_t)sl] = 1;
            fz_F[(size_t)sl] = ctx->slice_host[sl];
            fz_th[(size_t)sl] = ctx->slice_host[NS + sl];
            ctx->slice_sweeps[(size_t)sl] = s_now;
            if (use_skip) skip_set(sl);
        }
    };
    // after an exact reduction (slice_host): stop every running unit whose exact stopping quantity is
    // below eps, then fill F and the stopping quantity of every copy from the exact sums
    auto after_exact = [&](int s_now) -> int {
        bool changed = false;
        for (int u = 0; u < nunits; ++u) {
            if (unit_frozen[(size_t)u]) continue;
            const double st = stop_range(u * uspan, (u + 1) * uspan, [&](int sl) { return ctx->slice_host[NS + sl]; });
            if (st < eps) { freeze_unit(u, s_now); changed = true; }
        }
        if (changed && use_skip)
            CU(cudaMemcpyAsync(ctx->skip_dev, ctx->skip_host, (size_t)NSloc, cudaMemcpyHostToDevice, ctx->stream));
        for (int c = 0; c < B; ++c) {
            double fs = 0.0;
            for (int sl = c * Nt; sl < (c + 1) * Nt; ++sl) fs += frozen[(size_t)sl] ? fz_F[(size_t)sl] : ctx->slice_host[sl];
            Fc[(size_t)c] = fs / (ncd * nd * (double)ctx->VG);
            stopc[(size_t)c] = stop_range(c * Nt, (c + 1) * Nt, [&](int sl) { return ctx->slice_host[NS + sl]; });
        }
        have_exact = true;
        return GF_OK;
    };

    if (skip_slice) {   // units left alone: frozen from the start with their exact sums
        rc = exact_measure(ctx, gauge);
        if (rc) return rc;
        for (int u = 0; u < nunits; ++u) {
            bool all = true;
            for (int sl = u * uspan; sl < (u + 1) * uspan; ++sl) all = all && skip_slice[sl];
            if (all) freeze_unit(u, 0);
        }
    }
    if (use_skip) CU(cudaMemcpyAsync(ctx->skip_dev, ctx->skip_host, (size_t)NSloc, cudaMemcpyHostToDevice, ctx->stream));

    // fused partials of the even (and odd) half-sweep -> red_host = [NS][3] even, then [NS][3] odd, per global slice
    auto fetch_red = [&](bool even, bool odd) -> int {
        if (ctx->sharded) memset(ctx->red_host, 0, (size_t)6 * NS * sizeof(double));
        for (int k = 0; k < 2; ++k) {
            if (!(k ? odd : even)) continue;
            red_reduce_kernel<<<NSloc, 128, 0, ctx->stream>>>(ctx->red_part[k], gx, ctx->red_dev + 3 * NSloc * k);
            CU(cudaGetLastError());
            ++ctx->launches;
            CU(cudaMemcpyAsync(ctx->red_host + 3 * NS * k + 3 * goff, ctx->red_dev + 3 * NSloc * k, (size_t)3 * NSloc * sizeof(double),
                               cudaMemcpyDeviceToHost, ctx->stream));
        }
        return GF_OK;
    };
    auto finish_red = [&]() -> int {   // after the copies of fetch_red have been waited for
        if (ctx->sharded) shard_allreduce(ctx, ctx->red_host, 6 * NS);
        return GF_OK;
    };

    // history entry still waiting for the even sites' share of theta:
    //   stage 1 = the next even half-sweep must produce it, stage 2 = produced, reduced at the next check
    int pend_stage = 0, pend_entry = -1;
    std::vector<double> pend_odd((size_t)NS, 0.0);
    auto complete_pending = [&](const double* ev) {   // ev = [NS][3] partial sums of the even half-sweep
        if (hist)
            for (int c = 0; c < B; ++c)
                hist[3 * ((size_t)pend_entry * B + c) + 2] =
                    stop_range(c * Nt, (c + 1) * Nt, [&](int sl) { return pend_odd[(size_t)sl] + ev[3 * sl + 2]; });
        pend_stage = 0;
    };
    // GF_FLAG_LAGGED_STOP (one unit): a check whose lower bound theta_odd(s) falls below eps is not decided by the
    // stand-alone reduction but half a sweep later, from the even sites' share that the even half-sweep of sweep s + 1
    // sees before it updates: exact and free; if theta(s) < eps the run stops there (gf.h)
    // Not on GF_SP contexts: there the fused terms are formed from float sums (noise ~1e-12 in theta, see `trig`), a
    // decision at theta ~ eps could differ from the exact one, and by the time it is taken the links have moved on, so
    // the exact reduction can no longer settle it.  SP runs keep the margin + exact reduction of the plain path.
    const bool lagged = fused && (ctx->flags & GF_FLAG_LAGGED_STOP) && nunits == 1 && !skip_slice && ctx->precision != GF_SP;
    bool lag_decide = false, lag_stopped = false;
    // float Step 1 (GF_SP): the fused terms are formed from float sums and carry their rounding noise (~1e-12 in
    // theta); the exact reduction is called for a little earlier so that the bound stays one
    const double trig = eps + ((ctx->precision == GF_SP && eps > 0.0) ? (2e-12 > 1e-2 * eps ? 2e-12 : 1e-2 * eps) : 0.0);
    int s = 0, nh = 0, last_entry_sweep = -1;
    while (s < max_sweeps && n_frozen < nunits) {
        const bool check_now = ((s + 1) % check_every == 0) || (s + 1 == max_sweeps);
        const bool red_even = fused && pend_stage == 1;
        const uint32_t idx = first_sweep_index + (uint32_t)s;
        rc = launch_half(ctx, gauge, algo, param, seed, idx, 0, red_even ? ctx->red_part[0] : nullptr, skip);
        if (rc) return rc;
        if (red_even) pend_stage = 2;
        if (lag_decide) {   // the decision of the check at sweep s, now that theta_even(s) is known
            rc = fetch_red(true, false);
            if (rc) return rc;
            CU(cudaStreamSynchronize(ctx->stream));
            rc = finish_red();
            if (rc) return rc;
            const double* ev0 = ctx->red_host;
            const double th_s = stop_range(0, NS, [&](int sl) { return pend_odd[(size_t)sl] + ev0[3 * sl + 2]; });
            complete_pending(ev0);
            lag_decide = false;
            if (th_s < eps) { lag_stopped = true; break; }
        }
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
            const bool had_pending = pend_stage == 2;
            if (had_pending) {
                rc = fetch_red(true, false);
                if (rc) return rc;
            }
            rc = exact_measure(ctx, gauge);
            if (rc) return rc;
            if (had_pending) {
                rc = finish_red();
                if (rc) return rc;
                complete_pending(ctx->red_host);
            }
            pend_stage = 0;
            rc = after_exact(s);
            if (rc) return rc;
        } else {
            rc = fetch_red(pend_stage == 2, true);
            if (rc) return rc;
            CU(cudaStreamSynchronize(ctx->stream));
            rc = finish_red();
            if (rc) return rc;
            const double* ev = ctx->red_host;            // [sl][3]: even half-sweep of this or an earlier sweep
            const double* od = ctx->red_host + 3 * NS;   // [sl][3]: odd half-sweep of sweep s
            if (pend_stage == 2) complete_pending(ev);
            // lower bounds theta_odd(s) of the running units
            bool need_exact = false;
            for (int u = 0; u < nunits && !need_exact; ++u)
                need_exact = !unit_frozen[(size_t)u] &&
                             stop_range(u * uspan, (u + 1) * uspan, [&](int sl) { return od[3 * sl + 1]; }) < trig;
            if (need_exact && lagged && s < max_sweeps) {
                lag_decide = true;
                need_exact = false;
            }
            if (need_exact) {
                rc = exact_measure(ctx, gauge);
                if (rc) return rc;
                rc = after_exact(s);
                if (rc) return rc;
            } else {
                for (int c = 0; c < B; ++c) {
                    double fs = 0.0;
                    for (int sl = c * Nt; sl < (c + 1) * Nt; ++sl) fs += frozen[(size_t)sl] ? fz_F[(size_t)sl] : od[3 * sl];
                    Fc[(size_t)c] = fs / (ncd * nd * (double)ctx->VG);
                    stopc[(size_t)c] = stop_range(c * Nt, (c + 1) * Nt, [&](int sl) { return od[3 * sl + 1]; });
                }
                for (int sl = 0; sl < NS; ++sl) pend_odd[(size_t)sl] = od[3 * sl + 1];
                pend_stage = 1;
                pend_entry = nh;
            }
        }
        if (hist)
            for (int c = 0; c < B; ++c) {
                double* h = hist + 3 * ((size_t)nh * B + c);
                h[0] = (double)s; h[1] = Fc[(size_t)c]; h[2] = stopc[(size_t)c];
            }
        last_entry_sweep = s;
        ++nh;
    }
    if (!have_exact) {
        rc = exact_measure(ctx, gauge);
        if (rc) return rc;
        rc = after_exact(s);
        if (rc) return rc;
        if (hist && nh > 0 && last_entry_sweep == s && !lag_stopped)   // (lagged stop: the entry stays that of the check)
            for (int c = 0; c < B; ++c) {
                double* h = hist + 3 * ((size_t)(nh - 1) * B + c);
                h[1] = Fc[(size_t)c]; h[2] = stopc[(size_t)c];
            }
    }
    if (lag_stopped && !unit_frozen[0]) freeze_unit(0, s);   // converged by theta(s); the links are half a sweep further
    for (int sl = 0; sl < NS; ++sl)
        if (!frozen[(size_t)sl]) ctx->slice_sweeps[(size_t)sl] = s;
    ctx->slice_frozen = frozen;
    if (coulomb && ctx->gtot) {
        rc = gf_coulomb_finalize(ctx);
        if (rc) return rc;
        CU(cudaStreamSynchronize(ctx->stream));
    }
    if (out)
        for (int c = 0; c < B; ++c) {
            int sw = 0;
            for (int sl = c * Nt; sl < (c + 1) * Nt; ++sl)
                if (ctx->slice_sweeps[(size_t)sl] > sw) sw = ctx->slice_sweeps[(size_t)sl];
            out[c].sweeps = sw; out[c].F = Fc[(size_t)c]; out[c].theta = stopc[(size_t)c];
        }
    if (all_converged) *all_converged = (n_frozen == nunits);
    return GF_OK;
}

int gf_run_batch(gf_ctx* ctx, int gauge, int algo, double param, uint64_t seed, uint32_t first_sweep_index,
                 int max_sweeps, double eps, int check_every, int reunit_every, gf_result* out, double* hist) {
    if (!ctx) return GF_EINVAL;
    bool conv = false;
    int rc = run_impl(ctx, gauge, algo, param, seed, first_sweep_index, max_sweeps, eps, check_every, reunit_every,
                      nullptr, out, hist, &conv);
    if (rc) return rc;
    return conv ? GF_OK : GF_NOT_CONVERGED;
}

int gf_run(gf_ctx* ctx, int gauge, int algo, double param, uint64_t seed, uint32_t first_sweep_index,
           int max_sweeps, double eps, int check_every, int reunit_every, gf_result* out, double* hist) {
    if (!ctx) return GF_EINVAL;
    int rc = single_only(ctx, "gf_run");
    if (rc) return rc;
    return gf_run_batch(ctx, gauge, algo, param, seed, first_sweep_index, max_sweeps, eps, check_every, reunit_every,
                        out, hist);
}

int gf_get_slice_sweeps(gf_ctx* ctx, int* sweeps) {
    if (!ctx) return GF_EINVAL;
    if (!sweeps) return fail(ctx, GF_EINVAL, "gf_get_slice_sweeps: NULL pointer");
    if (!ctx->have_slice_sweeps) return fail(ctx, GF_ESTATE, "gf_get_slice_sweeps: no gf_run yet");
    for (int t = 0; t < ctx->NSG; ++t) sweeps[t] = ctx->slice_sweeps[(size_t)t];
    return GF_OK;
}

// (GF_RECON12_REUNIT is defined above run_impl)
// With 12-real storage the third row is rebuilt as (u x v)^* from stored rows that are never re-orthonormalised:
// a rotation that mixes it back into the stored rows compounds their norm errors, and under the large rotations of
// heatbath and microcanonical sweeps |1 - det U| grows by about a third per sweep (measured: 7e-6 -> 1e+7 in 60
// sweeps in SP, 6e-14 -> 2e-7 in DP; overrelaxation near a maximum is benign).  Schedules made of such sweeps
// therefore reproject at least this often on 12-real contexts.
// the annealing schedule; reunit_every > 0 reprojects after every reunit_every-th sweep of the schedule
static int anneal_impl(gf_ctx* ctx, int gauge, double T_hi, double T_lo, int n_steps, int n_micro, uint64_t seed,
                       uint32_t first_sweep_index, int reunit_every, uint32_t* next_sweep_index) {
    int rc = check_sweep_args(ctx, gauge, GF_SA, T_hi);
    if (rc) return rc;
    if (!(T_lo > 0.0) || n_steps < 0 || n_micro < 0 || reunit_every < 0) return fail(ctx, GF_EINVAL, "gf_anneal: bad schedule");
    rc = pre_sweep(ctx, gauge);
    if (rc) return rc;
    if (ctx->recon == 12 && (reunit_every == 0 || reunit_every > GF_RECON12_REUNIT)) reunit_every = GF_RECON12_REUNIT;
    uint32_t idx = first_sweep_index;
    int done = 0;
    auto one = [&](int algo, double par) -> int {
        for (int p = 0; p < 2; ++p) {
            int r = launch_half(ctx, gauge, algo, par, seed, idx, p);
            if (r) return r;
        }
        ++idx;
        ++done;
        if (reunit_every && done % reunit_every == 0) return gf_reunitarize(ctx);
        return GF_OK;
    };
    for (int k = 0; k < n_steps; ++k) {
        const double T = (n_steps <= 1) ? T_hi : T_hi - k * (T_hi - T_lo) / (n_steps - 1);
        rc = one(GF_SA, T);
        if (rc) return rc;
        for (int m = 0; m < n_micro; ++m) {
            rc = one(GF_MICRO, 0.0);
            if (rc) return rc;
        }
    }
    if (next_sweep_index) *next_sweep_index = idx;
    return GF_OK;
}

int gf_anneal(gf_ctx* ctx, int gauge, double T_hi, double T_lo, int n_steps, int n_micro, uint64_t seed,
              uint32_t first_sweep_index, uint32_t* next_sweep_index) {
    return anneal_impl(ctx, gauge, T_hi, T_lo, n_steps, n_micro, seed, first_sweep_index, 0, next_sweep_index);
}

// ---- the SA -> SR -> OR pipeline ------------------------------------------
int gf_fix(gf_ctx* ctx, const gf_fix_params* p, gf_result* out) {
    if (!ctx) return GF_EINVAL;
    if (!p) return fail(ctx, GF_EINVAL, "gf_fix: NULL parameters");
    if (p->sa_steps < 0 || p->sr_max_sweeps < 0 || p->or_max_sweeps < 0 || p->check_every < 1 || p->reunit_every < 0)
        return fail(ctx, GF_EINVAL, "gf_fix: bad stage lengths");
    const int B = ctx->B, Nt = ctx->NtG, NS = ctx->NSG;   // per global slice (run_impl)
    uint32_t idx = 0;
    int rc;
    std::vector<int> total((size_t)NS, 0);   // sweeps per slice, all stages
    std::vector<unsigned char> done;
    std::vector<gf_result> res((size_t)B);
    bool have_res = false, all = false;
    if (p->sa_steps > 0) {   // stage 1: simulated annealing, every copy
        rc = anneal_impl(ctx, p->gauge, p->sa_T_hi, p->sa_T_lo, p->sa_steps, p->sa_micro, p->seed, idx, p->reunit_every, &idx);
        if (rc) return rc;
        for (int sl = 0; sl < NS; ++sl) total[(size_t)sl] += (int)idx;
    }
    if (p->sr_max_sweeps > 0) {   // stage 2: stochastic relaxation until theta < eps, at most sr_max_sweeps
        // (stochastic relaxation takes microcanonical steps: run_impl applies GF_RECON12_REUNIT on 12-real contexts)
        rc = run_impl(ctx, p->gauge, GF_SR, p->sr_p, p->seed, idx, p->sr_max_sweeps, p->eps, p->check_every,
                      p->reunit_every, nullptr, res.data(), nullptr, &all);
        if (rc) return rc;
        have_res = true;
        for (int sl = 0; sl < NS; ++sl) total[(size_t)sl] += ctx->slice_sweeps[(size_t)sl];
        done = ctx->slice_frozen;
    }
    if (p->or_max_sweeps > 0 && !(have_res && all)) {   // stage 3: overrelaxation of the units still running
        rc = run_impl(ctx, p->gauge, GF_OR, p->or_omega, p->seed, idx, p->or_max_sweeps, p->eps, p->check_every,
                      p->reunit_every, have_res ? done.data() : nullptr, res.data(), nullptr, &all);
        if (rc) return rc;
        for (int sl = 0; sl < NS; ++sl) total[(size_t)sl] += ctx->slice_sweeps[(size_t)sl];
        have_res = true;
    }
    if (!have_res) {   // annealing only: report the exact F / theta of what it left
        rc = run_impl(ctx, p->gauge, GF_OR, 1.0, p->seed, idx, 0, p->eps, 1, 0, nullptr, res.data(), nullptr, &all);
        if (rc) return rc;
    }
    ctx->slice_sweeps = total;
    if (out)
        for (int c = 0; c < B; ++c) {
            out[c] = res[(size_t)c];
            int sw = 0;
            for (int sl = c * Nt; sl < (c + 1) * Nt; ++sl)
                if (total[(size_t)sl] > sw) sw = total[(size_t)sl];
            out[c].sweeps = sw;
        }
    return all ? GF_OK : GF_NOT_CONVERGED;
}

// ---- random start on the gauge orbit ------------------------------------------
#define GAUGE_APPLY(R, RECON, hf)                                                                               \
    gauge_apply_kernel<R, RECON><<<dim3((unsigned)((ctx->Vh + 127) / 128), (unsigned)ctx->B, 2), 128, 0, ctx->stream>>>( \
        ctx->links, ctx->gtot, (hf), dims_of(ctx), link_store_bytes(ctx), field_store_bytes(ctx), seed, top_site0)

int gf_random_gauge(gf_ctx* ctx, uint64_t seed) {
    if (!ctx) return GF_EINVAL;
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_random_gauge: no links set");
    // t-shards: h(x) is a function of the site index in the whole lattice, so a shard draws its own sites' h and
    // recomputes h of the slice above for the temporal links of its last slice; nothing is exchanged
    const int64_t slice_sites = (int64_t)ctx->Nx * ctx->Ny * ctx->Nz;
    const int64_t site_off = (int64_t)ctx->t0 * slice_sites;
    const int64_t top_site0 = ctx->sharded ? (int64_t)((ctx->t0 + ctx->Nt) % ctx->NtG) * slice_sites : -1;
    if (ctx->temporal_stale && ctx->gtot) {
        int rc = gf_coulomb_finalize(ctx);
        if (rc) return rc;
    }
    char* h = nullptr;
    CU(cudaMalloc((void**)&h, (size_t)(ctx->B * field_store_bytes(ctx))));
    const dim3 g((unsigned)((ctx->V + 127) / 128), (unsigned)ctx->B);
    const dim3 ga((unsigned)((ctx->Vh + 127) / 128), (unsigned)ctx->B, 2);
    cudaError_t e;
    if (ctx->nc == 2) {
        if (ctx->real_bytes == 4) haar_field2_kernel<float><<<g, 128, 0, ctx->stream>>>(h, dims_of(ctx), seed, field_store_bytes(ctx));
        else haar_field2_kernel<double><<<g, 128, 0, ctx->stream>>>(h, dims_of(ctx), seed, field_store_bytes(ctx));
        e = cudaGetLastError();
        if (e == cudaSuccess) {
            if (ctx->real_bytes == 4)
                gauge_apply2_kernel<float><<<ga, 128, 0, ctx->stream>>>(ctx->links, ctx->gtot, h, dims_of(ctx), link_store_bytes(ctx), field_store_bytes(ctx));
            else
                gauge_apply2_kernel<double><<<ga, 128, 0, ctx->stream>>>(ctx->links, ctx->gtot, h, dims_of(ctx), link_store_bytes(ctx), field_store_bytes(ctx));
            e = cudaGetLastError();
        }
    } else {
        if (ctx->real_bytes == 4) haar_field_kernel<float><<<g, 128, 0, ctx->stream>>>(h, dims_of(ctx), seed, field_store_bytes(ctx), site_off);
        else haar_field_kernel<double><<<g, 128, 0, ctx->stream>>>(h, dims_of(ctx), seed, field_store_bytes(ctx), site_off);
        e = cudaGetLastError();
        if (e == cudaSuccess) {
            DISPATCH_RR(ctx, GAUGE_APPLY, h);
            e = cudaGetLastError();
        }
    }
    ctx->launches += 2;
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(h);
    CU(e);
    // h was applied to all four directions: Coulomb sweeps that follow snapshot g(x) = h g(x) as already applied
    transform_changed(ctx);
    shard_barrier(ctx);
    (void)top_site0;
    return GF_OK;
}

// ---- input generator: Wilson-action heatbath, plaquette ---------------------
#define WILSON_HB(R, RECON, mu_, par_, sw_)                                                                      \
    wilson_heatbath_kernel<R, RECON><<<dim3((unsigned)((Vsh + 127) / 128), (unsigned)ctx->NS), 128, 0, ctx->stream>>>( \
        ctx->links, dims_of(ctx), (mu_), (par_), beta, seed, (sw_), link_store_bytes(ctx))

int gf_wilson_heatbath(gf_ctx* ctx, double beta, uint64_t seed, uint32_t first_sweep_index, int n_sweeps) {
    if (!ctx) return GF_EINVAL;
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_wilson_heatbath: no links set");
    if (!(beta > 0.0) || n_sweeps < 0) return fail(ctx, GF_EINVAL, "gf_wilson_heatbath: beta = %g, n_sweeps = %d", beta, n_sweeps);
    if (int rcs = not_on_shards(ctx, "gf_wilson_heatbath")) return rcs;
    if (ctx->temporal_stale && ctx->gtot) {
        int rc = gf_coulomb_finalize(ctx);
        if (rc) return rc;
    }
    const int Vsh = ctx->Nx * ctx->Ny * (ctx->Nz / 2);
    for (int k = 0; k < n_sweeps; ++k)
        for (int mu = 0; mu < 4; ++mu)
            for (int par = 0; par < 2; ++par) {
                if (ctx->nc == 2) {
                    const dim3 g2((unsigned)((Vsh + 127) / 128), (unsigned)ctx->NS);
                    if (ctx->real_bytes == 4)
                        wilson_heatbath2_kernel<float><<<g2, 128, 0, ctx->stream>>>(ctx->links, dims_of(ctx), mu, par, beta, seed,
                                                                                     first_sweep_index + (uint32_t)k, link_store_bytes(ctx));
                    else
                        wilson_heatbath2_kernel<double><<<g2, 128, 0, ctx->stream>>>(ctx->links, dims_of(ctx), mu, par, beta, seed,
                                                                                      first_sweep_index + (uint32_t)k, link_store_bytes(ctx));
                } else
                    DISPATCH_RR(ctx, WILSON_HB, mu, par, first_sweep_index + (uint32_t)k);
                CU(cudaGetLastError());
                ++ctx->launches;
                if (mu == 3 && par == 1 && ((ctx->recon == 12 && (k + 1) % GF_RECON12_REUNIT == 0) ||
                                            (ctx->recon != 12 && ctx->real_bytes == 4 && (k + 1) % 100 == 0))) {
                    // 12-real storage under heatbath rotations: reproject as the annealing schedules do;
                    // float links otherwise: every 100 sweeps
                    int rc = gf_reunitarize(ctx);
                    if (rc) return rc;
                }
            }
    // a new configuration, not a gauge transform of the old one: the accumulated g(x) restarts
    for (int c = 0; c < ctx->B && ctx->gtot; ++c) {
        int rc = reset_transform(ctx, c);
        if (rc) return rc;
    }
    return GF_OK;
}

#define PLAQUETTE(R, RECON, dummy)                                                                               \
    plaquette_kernel<R, RECON><<<dim3((unsigned)ctx->meas_gx, (unsigned)ctx->NS, 2), ctx->meas_block, 0, ctx->stream>>>( \
        ctx->links, dims_of(ctx), ctx->partial, link_store_bytes(ctx), ctx->links_up, ctx->Vh_up)

int gf_plaquette(gf_ctx* ctx, double* plaq) {
    if (!ctx) return GF_EINVAL;
    if (!plaq) return fail(ctx, GF_EINVAL, "gf_plaquette: NULL pointer");
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_plaquette: no links set");
    if (int rca = need_attached(ctx, "gf_plaquette")) return rca;
    if (ctx->temporal_stale && ctx->gtot) {
        int rc = gf_coulomb_finalize(ctx);
        if (rc) return rc;
    }
    shard_barrier(ctx);   // the last slice reads the first one of the store above
    if (ctx->nc == 2) {
        const dim3 g2((unsigned)ctx->meas_gx, (unsigned)ctx->NS, 2);
        if (ctx->real_bytes == 4) plaquette2_kernel<float><<<g2, ctx->meas_block, 0, ctx->stream>>>(ctx->links, dims_of(ctx), ctx->partial, link_store_bytes(ctx));
        else plaquette2_kernel<double><<<g2, ctx->meas_block, 0, ctx->stream>>>(ctx->links, dims_of(ctx), ctx->partial, link_store_bytes(ctx));
    } else
        DISPATCH_RR(ctx, PLAQUETTE, 0);
    CU(cudaGetLastError());
    slice_reduce_kernel<<<ctx->NS, 128, 0, ctx->stream>>>(ctx->partial, 2 * ctx->meas_gx, ctx->NS, ctx->slice_dev);
    CU(cudaGetLastError());
    ctx->launches += 2;
    if (ctx->sharded) {   // per global slice, completed over the shards and summed in slice order on every shard
        memset(ctx->slice_host, 0, (size_t)2 * ctx->NSG * sizeof(double));
        CU(cudaMemcpyAsync(ctx->slice_host + ctx->t0, ctx->slice_dev, (size_t)ctx->NS * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    } else {
        CU(cudaMemcpyAsync(ctx->slice_host, ctx->slice_dev, (size_t)2 * ctx->NS * sizeof(double), cudaMemcpyDeviceToHost,
                           ctx->stream));
    }
    int rcf = finish_enqueued_measure(ctx);
    if (rcf) return rcf;
    for (int c = 0; c < ctx->B; ++c) {
        double tot = 0.0;
        for (int t = 0; t < ctx->NtG; ++t) tot += ctx->slice_host[(size_t)c * ctx->NtG + t];
        plaq[c] = tot / ((double)ctx->nc * 6.0 * (double)ctx->VG);
    }
    return GF_OK;
}

// ---- unitarity measure, Eq. (33) ------------------------------------------------------------------
int gf_unitarity(gf_ctx* ctx, double* avg, double* max) {
    if (!ctx) return GF_EINVAL;
    if (!ctx->have_links) return fail(ctx, GF_ESTATE, "gf_unitarity: no links set");
    const int nb = (int)((8 * ctx->Vh + 255) / 256);
    double* part = nullptr;
    double* out = nullptr;
    CU(cudaMalloc((void**)&part, (size_t)nb * ctx->B * 2 * sizeof(double)));
    cudaError_t e = cudaMalloc((void**)&out, (size_t)ctx->B * 2 * sizeof(double));
    std::vector<double> h((size_t)ctx->B * 2, 0.0);
    if (e == cudaSuccess) {
        const dim3 g((unsigned)nb, (unsigned)ctx->B);
#define UNITARITY(R, RECON, dummy) unitarity_kernel<R, RECON><<<g, 256, 0, ctx->stream>>>(ctx->links, ctx->Vh, link_store_bytes(ctx), part)
        if (ctx->nc == 2) {
            if (ctx->real_bytes == 4) unitarity2_kernel<float><<<g, 256, 0, ctx->stream>>>(ctx->links, ctx->Vh, link_store_bytes(ctx), part);
            else unitarity2_kernel<double><<<g, 256, 0, ctx->stream>>>(ctx->links, ctx->Vh, link_store_bytes(ctx), part);
        } else
            DISPATCH_RR(ctx, UNITARITY, 0);
#undef UNITARITY
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) {
        unitarity_reduce_kernel<<<ctx->B, 256, 0, ctx->stream>>>(part, nb, out);
        e = cudaGetLastError();
        ctx->launches += 2;
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(h.data(), out, h.size() * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(part);
    cudaFree(out);
    CU(e);
    for (int c = 0; c < ctx->B; ++c) {
        if (avg) avg[c] = h[(size_t)c * 2] / (4.0 * (double)ctx->V);
        if (max) max[c] = h[(size_t)c * 2 + 1];
    }
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

// tuning hook (gf.h "Tuning hooks"): 0 = gf_run measures after every check with the measure kernels
int gf_debug_set_fused(gf_ctx* ctx, int fused) {
    if (!ctx) return GF_EINVAL;
    ctx->fused = fused != 0;
    return GF_OK;
}

// tuning hook (gf.h "Tuning hooks"): 0 = half-sweeps launched without programmatic dependent launch
int gf_debug_set_pdl(gf_ctx* ctx, int pdl) {
    if (!ctx) return GF_EINVAL;
    ctx->pdl = pdl != 0;
    return GF_OK;
}

// tuning hook (gf.h "Tuning hooks"): CTA size of the half-sweep kernel, 0 = default
int gf_debug_set_block(gf_ctx* ctx, int block) {
    if (!ctx || block < 0 || (block & 31)) return GF_EINVAL;
    ctx->block_override = block;
    return GF_OK;
}

}  // extern "C"
