// vg_k_trd.cu -- instantiates the streaming query kernels of the trd (five queries x {128-bit, 64-bit} paths).
#include "vg_kernels.cuh"

namespace vg {

cudaError_t launch_trd(int q, const TrdP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                          cudaStream_t s)
{
    return launch_any<Trd>(q, p, t, step_max, n, out, vec, s);
}

cudaError_t launch_trd_all(const TrdP &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec,
                           cudaStream_t s)
{
    return launch_all<Trd>(p, t, step_max, n, o, vec, s);
}

} // namespace vg
