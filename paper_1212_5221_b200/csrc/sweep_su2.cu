// half-sweep kernels for the gauge group SU(2): float, float with Step 1 in double, double
#include "sweep_su2.cuh"
namespace gf {
template cudaError_t launch_sweep_su2<float, float>(const SweepArgs&, int, bool, int, cudaStream_t);
template cudaError_t launch_sweep_su2<float, double>(const SweepArgs&, int, bool, int, cudaStream_t);
template cudaError_t launch_sweep_su2<double, double>(const SweepArgs&, int, bool, int, cudaStream_t);
}
