// vg_k_tube.cu -- instantiates the query kernels of the tube: the run-time-flag form (pipelined kernel, navigator)
// and one straight-line specialisation per (hollow, phi mode), picked here from the constants.
#include "vg_kernels.cuh"

namespace vg {

template <int WM>
static cudaError_t launch_tube_w(int q, const TubeP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                                 cudaStream_t s)
{
    if (p.hollow) return launch_any<Tube, TubeT<solid_flags(true, WM)>>(q, p, t, step_max, n, out, vec, s);
    return launch_any<Tube, TubeT<solid_flags(false, WM)>>(q, p, t, step_max, n, out, vec, s);
}

cudaError_t launch_tube(int q, const TubeP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                        cudaStream_t s)
{
    if (p.w.full) return launch_tube_w<kWmFull>(q, p, t, step_max, n, out, vec, s);
    if (p.w.wide) return launch_tube_w<kWmWide>(q, p, t, step_max, n, out, vec, s);
    return launch_tube_w<kWmNarrow>(q, p, t, step_max, n, out, vec, s);
}

template <int WM>
static cudaError_t launch_tube_all_w(const TubeP &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec,
                                     cudaStream_t s)
{
    if (p.hollow) return launch_all<TubeT<solid_flags(true, WM)>>(p, t, step_max, n, o, vec, s);
    return launch_all<TubeT<solid_flags(false, WM)>>(p, t, step_max, n, o, vec, s);
}

cudaError_t launch_tube_all(const TubeP &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec,
                            cudaStream_t s)
{
    if (p.w.full) return launch_tube_all_w<kWmFull>(p, t, step_max, n, o, vec, s);
    if (p.w.wide) return launch_tube_all_w<kWmWide>(p, t, step_max, n, o, vec, s);
    return launch_tube_all_w<kWmNarrow>(p, t, step_max, n, o, vec, s);
}

} // namespace vg
