// tu_plane_yz64.cu — YZFused for slabs of 64 cells (eight lanes per ky column)
#include "launcher.cuh"
namespace bd {
int cu_plane_yz64(CudaLauncher& run, const PlanView& p) { return enqueue_plane_yz_nz<64>(run, p); }
}  // namespace bd
