// half-sweep kernels: storage float, Step 1 in float, 12 reals per stored link
#include "sweep_inst.cuh"
namespace gf {
template cudaError_t launch_sweep<float, float, 12>(const SweepArgs&, int, bool, int, cudaStream_t);
}
