// vg_boolx.cu -- boolean solids with a POLYCONE operand ("boolean operations" of the elementary bodies, of
// which the polycone is one; readings R27-R29, R32).  The polycone's constants (about 4 KiB) do
// not fit a by-value operand record, so vg_boolean_create puts them in device memory and the operand record carries a
// pointer (SolidU::u.pcon); the kernels are those of vg_bool.cuh -- same combination rules, same state machine over
// "inside A / inside B" -- instantiated with X = true, where an operand of kind kPolycone is answered by PolyconeT's
// own Inside / safety / sense-picked distances.  One kernel per query, operand kinds read at run time.
#include "vg_bool.cuh"

namespace vg {

cudaError_t launch_boolx(int q, const BoolP &p, const Tracks &t, double step_max, int64_t n, void *out, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    const unsigned grid = unsigned((n + kBoolBlock - 1) / kBoolBlock);
    switch (q) {
    case qInside: return launch_kernel(bool_kernel<qInside, -1, -1, true>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    case qSafeIn: return launch_kernel(bool_kernel<qSafeIn, -1, -1, true>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    case qSafeOut: return launch_kernel(bool_kernel<qSafeOut, -1, -1, true>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    case qDistIn: return launch_kernel(bool_kernel<qDistIn, -1, -1, true>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    case qDistOut: return launch_kernel(bool_kernel<qDistOut, -1, -1, true>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    }
    return cudaErrorInvalidValue;
}

} // namespace vg
