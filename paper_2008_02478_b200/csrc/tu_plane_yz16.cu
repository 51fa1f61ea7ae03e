// tu_plane_yz16.cu — YZFused for slabs of 16 cells (two lanes per ky column)
#include "launcher.cuh"
namespace bd {
int cu_plane_yz16(CudaLauncher& run, const PlanView& p) { return enqueue_plane_yz_nz<16>(run, p); }
}  // namespace bd
