// sweep_inst.cuh — host launcher for one (storage type R, Step-1 type A, RECON) family of
// half-sweep kernels.  Included by sweep_<prec><recon>.cu, one translation unit per family so the
// families compile in parallel.
#pragma once
#include "sweep.cuh"

namespace gf {

template <class R, class A, int RECON, int GAUGE, bool STOCH, bool TRACK>
static cudaError_t launch_one(const SweepArgs& args, int block, cudaStream_t stream) {
    constexpr int ND = (GAUGE == GAUGE_COULOMB) ? 3 : 4;
    auto kern = sweep_kernel<R, A, RECON, GAUGE, STOCH, TRACK>;
    const int64_t Vh = (int64_t)args.Nt * args.Nx * args.Ny * (args.Nz / 2);
    if (block <= 0 || block > SweepLaunch<R>::MAX_BLOCK) block = SweepLaunch<R>::MAX_BLOCK;
    const size_t smem = (size_t)block * 2 * ND * Layout<R, RECON>::LINK_BYTES;
    static size_t smem_set = 0;   // per instantiation
    if (smem > smem_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        if (e != cudaSuccess) return e;
        smem_set = smem;
    }
    const unsigned grid = (unsigned)((Vh + block - 1) / block);
    kern<<<grid, block, smem, stream>>>(args);
    return cudaGetLastError();
}

template <class R, class A, int RECON, int GAUGE>
static cudaError_t launch_gauge(const SweepArgs& args, bool track, int block, cudaStream_t stream) {
    const bool stoch = (args.algo == ALGO_SR || args.algo == ALGO_SA);
    if (stoch) {
        if (track) return launch_one<R, A, RECON, GAUGE, true, true>(args, block, stream);
        return launch_one<R, A, RECON, GAUGE, true, false>(args, block, stream);
    }
    if (track) return launch_one<R, A, RECON, GAUGE, false, true>(args, block, stream);
    return launch_one<R, A, RECON, GAUGE, false, false>(args, block, stream);
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
