// tu_plane_yz8.cu — YZFused for slabs of 8 cells (one lane per ky column)
#include "launcher.cuh"
namespace bd {
int cu_plane_yz8(CudaLauncher& run, const PlanView& p) { return enqueue_plane_yz_nz<8>(run, p); }
}  // namespace bd
