// vg_k_orb.cu -- instantiates the streaming query kernels of the orb (five queries x {128-bit, 64-bit} paths).
#include "vg_kernels.cuh"

namespace vg {

cudaError_t launch_orb(int q, const OrbP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                          cudaStream_t s)
{
    return launch_any<Orb>(q, p, t, step_max, n, out, vec, s);
}

cudaError_t launch_orb_all(const OrbP &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec,
                           cudaStream_t s)
{
    return launch_all<Orb>(p, t, step_max, n, o, vec, s);
}

} // namespace vg
