// tu_plane_yz.cu — the fused y/z kernel of the plane path (YZFused) of libborisdemag.so
#include "launcher.cuh"
namespace bd {
int cu_plane_yz(CudaLauncher& run, const PlanView& p) { return enqueue_plane_yz(run, p); }
}  // namespace bd
