// sweep_inst.cuh — host launcher for one (storage type R, Step-1 type A, RECON) family of
// half-sweep kernels.  Included by sweep_<prec><recon>.cu, one translation unit per family so the
// families compile in parallel.
#pragma once
#include <atomic>

#include "sweep.cuh"

namespace gf {

template <class R, class A, int RECON, int GAUGE, bool STOCH, bool TRACK, bool RED>
static cudaError_t launch_one(const SweepArgs& args, int block, cudaStream_t stream) {
    constexpr int ND = (GAUGE == GAUGE_COULOMB) ? 3 : 4;
    auto kern = sweep_kernel<R, A, RECON, GAUGE, STOCH, TRACK, RED>;
    const int Vsh = args.Nx * args.Ny * (args.Nz / 2);
    block = sweep_block<R, A>(Vsh, block, STOCH);
    // the slice stride is the maximal CTA size of the instantiation whatever the block (sweep.cuh, smem_get)
    const size_t smem = (size_t)SweepLaunch<R, A>::max_block(STOCH) * 2 * ND * Layout<R, RECON>::LINK_BYTES;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    DevLimits lim;
    e = dev_limits(dev, lim);   // SM count and shared-memory limits of this device (cached)
    if (e != cudaSuccess) return e;
    const dim3 grid((unsigned)((Vsh + block - 1) / block), (unsigned)(args.ncopies * args.Nt));
    // A grid of fewer CTAs than the SMs have slots is not spread evenly by the hardware (measured: 512 CTAs of 64
    // threads with nine slots per SM run 1.5x slower than with four).  Ask for as much shared memory per CTA as leaves
    // room for ceil(CTAs / SMs) of them on an SM: the CTAs then spread over all SMs.  Where the device's limits leave
    // no room for that (or the kernel's own need already exceeds the cap) the launch asks for what the kernel needs.
    size_t smem_launch = smem;
    {
        const long long ctas = (long long)grid.x * grid.y;
        const long long per_sm = (ctas + lim.sms - 1) / lim.sms;
        const size_t budget = lim.smem_per_sm / (size_t)(per_sm > 0 ? per_sm : 1);
        if (per_sm <= 8 && budget > smem + 1024) {
            smem_launch = ((budget - 1024) / 1024) * 1024;     // 1 KB per CTA is the driver's
            if (smem_launch > lim.smem_cta_cap) smem_launch = lim.smem_cta_cap;
            if (smem_launch < smem) smem_launch = smem;
        }
    }
    // function attributes are per device: remember what was set for this instantiation on each device.  Contexts may
    // be driven from several host threads (one thread per context, gf.h): the cache is atomic, and setting the same
    // attribute twice is harmless.  The opt-in limit asked for is the device's cap, so that any spreading request
    // fits; a device whose cap is below the kernel's own need gets the plain request (and the launch reports the error).
    static std::atomic<size_t> smem_set[64];
    if (dev < 0 || dev >= 64 || smem > smem_set[dev].load(std::memory_order_acquire)) {
        const size_t optin = lim.smem_cta_cap > smem ? lim.smem_cta_cap : smem;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)optin);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) smem_set[dev].store(smem, std::memory_order_release);
    }
    return launch_with_pdl(kern, grid, dim3((unsigned)block), smem_launch, stream, args);
}

template <class R, class A, int RECON, int GAUGE>
static cudaError_t launch_gauge(const SweepArgs& args, bool track, int block, cudaStream_t stream) {
    const bool stoch = (args.algo == ALGO_SR || args.algo == ALGO_SA);
    const int which = (stoch ? 4 : 0) | (track ? 2 : 0) | (args.red ? 1 : 0);
    switch (which) {
        case 0: return launch_one<R, A, RECON, GAUGE, false, false, false>(args, block, stream);
        case 1: return launch_one<R, A, RECON, GAUGE, false, false, true>(args, block, stream);
        case 2: return launch_one<R, A, RECON, GAUGE, false, true, false>(args, block, stream);
        case 3: return launch_one<R, A, RECON, GAUGE, false, true, true>(args, block, stream);
        case 4: return launch_one<R, A, RECON, GAUGE, true, false, false>(args, block, stream);
        case 5: return launch_one<R, A, RECON, GAUGE, true, false, true>(args, block, stream);
        case 6: return launch_one<R, A, RECON, GAUGE, true, true, false>(args, block, stream);
        default: return launch_one<R, A, RECON, GAUGE, true, true, true>(args, block, stream);
    }
}

template <class R, class A, int RECON>
cudaError_t launch_sweep(const SweepArgs& args, int gauge, bool track, int block, cudaStream_t stream) {
    switch (gauge) {
        case GAUGE_LANDAU: return launch_gauge<R, A, RECON, GAUGE_LANDAU>(args, track, block, stream);
        case GAUGE_COULOMB: return launch_gauge<R, A, RECON, GAUGE_COULOMB>(args, track, block, stream);
        case GAUGE_MAG: return launch_gauge<R, A, RECON, GAUGE_MAG>(args, track, block, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace gf
