// vg_csg.cu -- booleans whose operands include booleans (reading R31): the tree is flattened at vg_boolean_create into
// up to eight primitives and a postfix program (vg_params.h CsgP); the five queries evaluate that program.
//
// Inside runs it on (in, out) flag pairs, the safeties on the operands' signed distances (R27, R29, read recursively).
// The distances generalise the two-operand state machine of vg_bool.cu: one "inside" bit per primitive; every event
// asks each primitive for its next crossing in the sense its bit calls for, advances to the nearest (lowest leaf first on
// a tie = the oracle's "a tie goes to the left operand"), flips that bit and re-evaluates the program on the bits; the
// first event that changes the value of the whole tree is the answer.  O(primitives) solid evaluations per event: the
// general path; a boolean of two primitives keeps the specialised kernels of vg_bool.cu.
#include "vg_csg.cuh"

namespace vg {

constexpr int kCsgBlock = 128;

template <int Q>
__global__ void __launch_bounds__(kCsgBlock)
    csg_kernel(const __grid_constant__ CsgP p, Tracks t, double step_max, int64_t n, void *out)
{
    pdl_launch_dependents();
    pdl_wait();
    const int64_t i = int64_t(blockIdx.x) * kCsgBlock + threadIdx.x;
    if (i >= n) return;
    const double x = ldg1(t.x + i), y = ldg1(t.y + i), z = ldg1(t.z + i);
    if (Q == qSafeIn || Q == qSafeOut) {
        const double s = csg_sdf(p, x, y, z);
        stg1(static_cast<double *>(out) + i, Q == qSafeIn ? s : -s);
    } else if (Q == qInside) {
        unsigned in, o;
        csg_classes(p, x, y, z, in, o);
        stg1i(static_cast<int32_t *>(out) + i, csg_classify(p, in, o));
    } else {
        const double dx = ldg1(t.dx + i), dy = ldg1(t.dy + i), dz = ldg1(t.dz + i);
        const double r = csg_distance(p, Q == qDistOut, x, y, z, dx, dy, dz);
        stg1(static_cast<double *>(out) + i, r <= step_max ? r : inf());
    }
}

cudaError_t launch_csg(int q, const CsgP &p, const Tracks &t, double step_max, int64_t n, void *out, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    const unsigned grid = unsigned((n + kCsgBlock - 1) / kCsgBlock);
    switch (q) {
    case qInside: return launch_kernel(csg_kernel<qInside>, grid, kCsgBlock, 0, s, p, t, step_max, n, out);
    case qDistIn: return launch_kernel(csg_kernel<qDistIn>, grid, kCsgBlock, 0, s, p, t, step_max, n, out);
    case qDistOut: return launch_kernel(csg_kernel<qDistOut>, grid, kCsgBlock, 0, s, p, t, step_max, n, out);
    case qSafeIn: return launch_kernel(csg_kernel<qSafeIn>, grid, kCsgBlock, 0, s, p, t, step_max, n, out);
    case qSafeOut: return launch_kernel(csg_kernel<qSafeOut>, grid, kCsgBlock, 0, s, p, t, step_max, n, out);
    }
    return cudaErrorInvalidValue;
}

} // namespace vg
