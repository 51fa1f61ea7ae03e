// tu_y3.cu — YFused with the 6-component multiply (tiled 3-D path) of libborisdemag.so
#include "launcher.cuh"
namespace bd {
int cu_yfused3(CudaLauncher& run, const PlanView& p) { return enqueue_yfused3(run, p); }
}  // namespace bd
