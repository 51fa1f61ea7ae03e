// tu_t2d.cu — tiled 2-D path (XFwdT, YFused, XInvT) of libborisdemag.so
#include "launcher.cuh"
namespace bd {
int cu_tiled_2d(CudaLauncher& run, const PlanView& p, const float* M, float* H) { return dispatch_tiled_2d(run, p, M, H); }
}  // namespace bd
