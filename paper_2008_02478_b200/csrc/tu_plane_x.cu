// tu_plane_x.cu — x transforms of the plane path (XFwdT<LX,1>, XInvP) of libborisdemag.so
#include "launcher.cuh"
namespace bd {
int cu_plane_x(CudaLauncher& run, const PlanView& p, const float* M, float* H, bool fwd) {
    return enqueue_plane_x(run, p, M, H, fwd);
}
}  // namespace bd
