// vg_k_box.cu -- instantiates the streaming query kernels of the box (five queries x {128-bit, 64-bit} paths).
#include "vg_kernels.cuh"

namespace vg {

cudaError_t launch_box(int q, const BoxP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                          cudaStream_t s)
{
    return launch_any<Box>(q, p, t, step_max, n, out, vec, s);
}

cudaError_t launch_box_all(const BoxP &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec,
                           cudaStream_t s)
{
    return launch_all<Box>(p, t, step_max, n, o, vec, s);
}

} // namespace vg
