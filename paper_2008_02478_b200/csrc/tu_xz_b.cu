// tu_xz_b.cu — XZFwd / ZXInv for nz = 32 (tiled 3-D path) of libborisdemag.so
#include "launcher.cuh"
namespace bd {
int cu_xz_32(CudaLauncher& run, const PlanView& p, const float* M, float* H, bool fwd) {
    return enqueue_xz<32, 32>(run, p, M, H, fwd);
}
}  // namespace bd
