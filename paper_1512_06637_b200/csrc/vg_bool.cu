// vg_bool.cu -- boolean solids C = A op B of two primitives ("boolean operations", "logical
// operations"; readings R27-R29 in DESIGN.md): the five queries of vg.h on a vg_shape of kind
// VG_BOOLEAN.
//
// Inside and the safeties combine the two operands' answers (R27, R29).  The distances follow the membership of C
// along the ray (R28) WITHOUT enumerating every crossing as the oracle does: a small state machine holds "inside A",
// "inside B" and the ray parameter t, asks each operand for its NEXT crossing in the sense its state calls for (the
// leaving crossing if inside, the entering one if outside), advances to the nearer one, flips that state, and stops as
// soon as the membership of C differs from its value at the start.  After a flip the point sits ON the operand's
// surface; the operands' DistanceToIn / DistanceToOut select crossings by their sense (entering / leaving), not by
// "smallest positive root", so the crossing just taken (t ~ +-1e-16) is never taken again.  Box, trd and orb get
// sense-aware forms here for that reason (their stand-alone kernels may assume a start point clear of the surface).
#include "vg_bool.cuh"

namespace vg {

cudaError_t launch_boolean(int q, const BoolP &p, const Tracks &t, double step_max, int64_t n, void *out, cudaStream_t s, bool vec)
{
    if (n <= 0) return cudaSuccess;
    const unsigned grid = unsigned((n + kBoolBlock - 1) / kBoolBlock);
    if (vec && n >= 2 * 148 * VG_BOOL_PT_BLOCK) // (smaller batches: one track per thread fills more SMs)
        switch (q) {
        case qInside: return launch_bool_point2<qInside>(p, t, n, out, s);
        case qSafeIn: return launch_bool_point2<qSafeIn>(p, t, n, out, s);
        case qSafeOut: return launch_bool_point2<qSafeOut>(p, t, n, out, s);
        }
    switch (q) {
    case qInside: return launch_kernel(bool_kernel<qInside, -1, -1>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    case qSafeIn: return launch_kernel(bool_kernel<qSafeIn, -1, -1>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    case qSafeOut: return launch_kernel(bool_kernel<qSafeOut, -1, -1>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    case qDistIn:
    case qDistOut:
        switch (p.a.kind) { // the distance kernels are compiled per pair of operand kinds (vg_bool_k<A>.cu)
        case kBox: return launch_boolean_dist_kBox(q, p.b.kind, p, t, step_max, n, out, grid, s);
        case kOrb: return launch_boolean_dist_kOrb(q, p.b.kind, p, t, step_max, n, out, grid, s);
        case kTube: return launch_boolean_dist_kTube(q, p.b.kind, p, t, step_max, n, out, grid, s);
        case kCone: return launch_boolean_dist_kCone(q, p.b.kind, p, t, step_max, n, out, grid, s);
        case kTrd: return launch_boolean_dist_kTrd(q, p.b.kind, p, t, step_max, n, out, grid, s);
        }
    }
    return cudaErrorInvalidValue;
}

} // namespace vg
