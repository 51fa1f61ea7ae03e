// tu_plane_yz8.cu — YZFused for slabs of 8, 4 and 2 cells (one lane per ky column)
#include "launcher.cuh"
namespace bd {
int cu_plane_yz8(CudaLauncher& run, const PlanView& p) {
    if (p.nz == 4) return enqueue_plane_yz_nz<4>(run, p);
    if (p.nz == 2) return enqueue_plane_yz_nz<2>(run, p);
    return enqueue_plane_yz_nz<8>(run, p);
}
}  // namespace bd
