// tu_xz_c.cu — XZFwd / ZXInv for nz = 64..256 (tiled 3-D path) of libborisdemag.so
#include "launcher.cuh"
namespace bd {
int cu_xz_big(CudaLauncher& run, const PlanView& p, const float* M, float* H, bool fwd) {
    return enqueue_xz<64, 256>(run, p, M, H, fwd);
}
}  // namespace bd
