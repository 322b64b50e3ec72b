// vg_k_cone.cu -- instantiates the streaming query kernels of the cone (five queries x {128-bit, 64-bit} paths).
#include "vg_kernels.cuh"

namespace vg {

cudaError_t launch_cone(int q, const ConeP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                          cudaStream_t s)
{
    return launch_any<Cone>(q, p, t, step_max, n, out, vec, s);
}

} // namespace vg
