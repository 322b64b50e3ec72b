// vg_k_polycone.cu -- instantiates the query kernels of the polycone: the run-time-flag form and the full-phi
// specialisation (configs[3]), picked here from the constants.
#include "vg_kernels.cuh"

namespace vg {

cudaError_t launch_polycone(int q, const PolyconeP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                            cudaStream_t s)
{
    if (p.w.full) return launch_any<Polycone, PolyconeT<solid_flags(false, kWmFull)>>(q, p, t, step_max, n, out, vec, s);
    return launch_any<Polycone>(q, p, t, step_max, n, out, vec, s);
}

} // namespace vg
