// vg_k_polycone.cu -- instantiates the query kernels of the polycone and picks the form a call runs as (VG_FORM_AUTO; any
// forced form runs the generic streaming kernels over all sections):
//   n <= VG_OPT_COOP_MAX_N, full phi   a group of lanes per track (vg_pcon_coop.cuh)
//   above it                            one track per thread, section / segment tables in device memory
//                                       (vg_pcon_walk.cuh: ordered walks for Inside and the distances, candidate grids
//                                       for the safeties; full phi or a phi cut, any alignment)
//   tables not on the current device,   the persistent kernels with the tables staged per CTA (16-byte aligned arrays),
//   or VG_OPT_COOP_MAX_N = 0            else the generic kernels
#include "vg_pcon_coop.cuh"
#include "vg_pcon_walk.cuh"

namespace vg {

cudaError_t launch_polycone(int q, const PolyconeP &p, const PconGrid &g, const Tracks &t, double step_max, int64_t n,
                            void *out, bool vec, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    if (p.w.full) {
        // small batches: a group of lanes per track (vg_pcon_coop.cuh), any alignment
        if (g.coop && g_form.load(std::memory_order_relaxed) == 0 && n <= g_coop_max_n.load(std::memory_order_relaxed)) {
            switch (q) {
            case qInside: return launch_pcon_coop<qInside>(p, g, t, step_max, n, out, s);
            case qDistIn: return launch_pcon_coop<qDistIn>(p, g, t, step_max, n, out, s);
            case qDistOut: return launch_pcon_coop<qDistOut>(p, g, t, step_max, n, out, s);
            case qSafeIn: return launch_pcon_coop<qSafeIn>(p, g, t, step_max, n, out, s);
            case qSafeOut: return launch_pcon_coop<qSafeOut>(p, g, t, step_max, n, out, s);
            }
        }
        // Inside and the distances: one track per thread, section table in device memory (vg_pcon_walk.cuh), any alignment
        // (VG_OPT_COOP_MAX_N = 0 keeps the persistent kernels in use: the tests run every form)
        if (g.wtab && g_form.load(std::memory_order_relaxed) == 0 && g_coop_max_n.load(std::memory_order_relaxed) > 0) {
            if (q == qInside) return launch_pcon_walk_small<qInside, false>(p, g, t, step_max, n, out, s);
            if (q == qDistIn) return launch_pcon_walk_small<qDistIn, false>(p, g, t, step_max, n, out, s);
            if (q == qDistOut) return launch_pcon_walk_small<qDistOut, false>(p, g, t, step_max, n, out, s);
            if (g.masks && g.segs && q == qSafeIn) return launch_pcon_safety_small<qSafeIn, false>(p, g, t, n, out, s);
            if (g.masks && g.segs && q == qSafeOut) return launch_pcon_safety_small<qSafeOut, false>(p, g, t, n, out, s);
        }
        if (vec && g_form.load(std::memory_order_relaxed) == 0) {
            double *o = static_cast<double *>(out);
            if (q == qDistIn) return launch_pcon_walk<qDistIn, false>(p, g, t, step_max, n, o, s);
            if (q == qDistOut) return launch_pcon_walk<qDistOut, false>(p, g, t, step_max, n, o, s);
            if (q == qInside) return launch_pcon_walk<qInside, false>(p, g, t, step_max, n, out, s);
            // the safeties: candidate grid (built at vg_shape_create on the device it was created on), else the walk
            if (q == qSafeIn)
                return g.masks ? launch_pcon_walk<qSafeIn, true>(p, g, t, step_max, n, o, s)
                               : launch_pcon_walk<qSafeIn, false>(p, g, t, step_max, n, o, s);
            if (q == qSafeOut)
                return g.masks ? launch_pcon_walk<qSafeOut, true>(p, g, t, step_max, n, o, s)
                               : launch_pcon_walk<qSafeOut, false>(p, g, t, step_max, n, o, s);
        }
        return launch_any<Polycone, PolyconeT<solid_flags(false, kWmFull)>>(q, p, t, step_max, n, out, vec, s);
    }
    // a phi cut: the ordered walk serves DistanceToIn (every candidate also tested against the segment, the phi faces added)
    if (g.wtab && g_form.load(std::memory_order_relaxed) == 0 && g_coop_max_n.load(std::memory_order_relaxed) > 0) {
        if (q == qInside) return launch_pcon_walk_small<qInside, true>(p, g, t, step_max, n, out, s);
        if (q == qDistIn) return launch_pcon_walk_small<qDistIn, true>(p, g, t, step_max, n, out, s);
        if (q == qDistOut) return launch_pcon_walk_small<qDistOut, true>(p, g, t, step_max, n, out, s);
        if (g.masks && g.face_masks && g.segs && q == qSafeIn) return launch_pcon_safety_small<qSafeIn, true>(p, g, t, n, out, s);
        if (g.masks && g.face_masks && g.segs && q == qSafeOut) return launch_pcon_safety_small<qSafeOut, true>(p, g, t, n, out, s);
    }
    if (vec && g_form.load(std::memory_order_relaxed) == 0) {
        if (q == qDistIn) return launch_pcon_walk<qDistIn, false, true>(p, g, t, step_max, n, out, s);
        if (q == qDistOut) return launch_pcon_walk<qDistOut, false, true>(p, g, t, step_max, n, out, s);
        if (q == qInside) return launch_pcon_walk<qInside, false, true>(p, g, t, step_max, n, out, s);
    }
    // ... and the two candidate grids (surface of revolution, phi face) the safeties
    if (vec && g.masks && g.face_masks && g_form.load(std::memory_order_relaxed) == 0) {
        if (q == qSafeIn) return launch_pcon_walk<qSafeIn, true, true>(p, g, t, step_max, n, static_cast<double *>(out), s);
        if (q == qSafeOut) return launch_pcon_walk<qSafeOut, true, true>(p, g, t, step_max, n, static_cast<double *>(out), s);
    }
    return launch_any<Polycone>(q, p, t, step_max, n, out, vec, s);
}

// the fused five-query kernel of a polycone: needs 16-byte aligned arrays and, for the safeties of a polycone with a phi
// cut, its candidate grids; cudaErrorNotSupported tells the caller to run the five queries as separate launches
cudaError_t launch_polycone_all(const PolyconeP &p, const PconGrid &g, const Tracks &t, double step_max, int64_t n, const AllOut &o,
                                bool vec, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    // one track per thread with every table in device memory (any alignment); VG_OPT_COOP_MAX_N = 0 keeps the persistent kernel
    if (g_form.load(std::memory_order_relaxed) == 0 && g_coop_max_n.load(std::memory_order_relaxed) > 0 && g.wtab && g.segs && g.masks) {
        if (p.w.full) return launch_pcon_all_small<false>(p, g, t, step_max, n, o, s);
        if (g.face_masks) return launch_pcon_all_small<true>(p, g, t, step_max, n, o, s);
    }
    if (!vec || g_form.load(std::memory_order_relaxed) != 0) return cudaErrorNotSupported;
    if (p.w.full)
        return g.masks ? launch_pcon_all<true, false>(p, g, t, step_max, n, o, s) : launch_pcon_all<false, false>(p, g, t, step_max, n, o, s);
    if (g.masks && g.face_masks) return launch_pcon_all<true, true>(p, g, t, step_max, n, o, s);
    return cudaErrorNotSupported;
}

} // namespace vg
