// tu_xz_a.cu — XZFwd / ZXInv for nz = 2..16 (tiled 3-D path) of libborisdemag.so
#include "launcher.cuh"
namespace bd {
int cu_xz_small(CudaLauncher& run, const PlanView& p, const float* M, float* H, bool fwd) {
    return enqueue_xz<2, 16>(run, p, M, H, fwd);
}
}  // namespace bd
