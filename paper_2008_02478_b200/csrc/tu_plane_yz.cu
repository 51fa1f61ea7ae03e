// tu_plane_yz.cu — the fused y/z kernel of the plane path (YZFused) for slabs of 32 cells
#include "launcher.cuh"
namespace bd {
int cu_plane_yz16(CudaLauncher& run, const PlanView& p);     // tu_plane_yz16.cu
int cu_plane_yz8(CudaLauncher& run, const PlanView& p);      // tu_plane_yz8.cu
int cu_plane_yz64(CudaLauncher& run, const PlanView& p);     // tu_plane_yz64.cu
int cu_plane_yz(CudaLauncher& run, const PlanView& p) {
    if (p.nz == 64) return cu_plane_yz64(run, p);
    if (p.nz == 16) return cu_plane_yz16(run, p);
    if (p.nz <= 8) return cu_plane_yz8(run, p);
    return enqueue_plane_yz_nz<32>(run, p);
}
}  // namespace bd
