// vg_k_cone.cu -- instantiates the query kernels of the cone: the run-time-flag form (pipelined kernel, navigator)
// and one straight-line specialisation per (hollow, phi mode), picked here from the constants.
#include "vg_kernels.cuh"

namespace vg {

template <int WM>
static cudaError_t launch_cone_w(int q, const ConeP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                                 cudaStream_t s)
{
    if (p.hollow) return launch_any<Cone, ConeT<solid_flags(true, WM)>>(q, p, t, step_max, n, out, vec, s);
    return launch_any<Cone, ConeT<solid_flags(false, WM)>>(q, p, t, step_max, n, out, vec, s);
}

cudaError_t launch_cone(int q, const ConeP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                        cudaStream_t s)
{
    if (p.w.full) return launch_cone_w<kWmFull>(q, p, t, step_max, n, out, vec, s);
    if (p.w.wide) return launch_cone_w<kWmWide>(q, p, t, step_max, n, out, vec, s);
    return launch_cone_w<kWmNarrow>(q, p, t, step_max, n, out, vec, s);
}

template <int WM>
static cudaError_t launch_cone_all_w(const ConeP &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec,
                                     cudaStream_t s)
{
    if (p.hollow) return launch_all<ConeT<solid_flags(true, WM)>>(p, t, step_max, n, o, vec, s);
    return launch_all<ConeT<solid_flags(false, WM)>>(p, t, step_max, n, o, vec, s);
}

cudaError_t launch_cone_all(const ConeP &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec,
                            cudaStream_t s)
{
    if (p.w.full) return launch_cone_all_w<kWmFull>(p, t, step_max, n, o, vec, s);
    if (p.w.wide) return launch_cone_all_w<kWmWide>(p, t, step_max, n, o, vec, s);
    return launch_cone_all_w<kWmNarrow>(p, t, step_max, n, o, vec, s);
}

} // namespace vg
