// half-sweep kernels: storage double, Step 1 in double, 18 reals per stored link
#include "sweep_inst.cuh"
namespace gf {
template cudaError_t launch_sweep<double, double, 18>(const SweepArgs&, int, bool, int, cudaStream_t);
}
