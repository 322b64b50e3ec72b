// vg_bool.cuh -- device code of the boolean solids; see vg_bool.cu for the design.  Included by vg_bool.cu (Inside, the
// safeties, the dispatch) and by vg_bool_k<A>.cu (the distance kernels of operand kind A against every kind B: one
// translation unit per A so that the 50 instantiations compile in parallel).
#pragma once
#include "vg_kernels.cuh"
#include "vg_solid.cuh"

namespace vg {

constexpr int kBoolBlock = 128;
constexpr int kBoolMaxEvents = 64; // an operand has at most ~10 crossings with a line; the loop ends long before

// next crossing of the operand's boundary in the given sense (leaving: the track is inside it) that lies ahead of the
// point or at it (R32: t > -kRayTol, clamped at 0), +inf if none.  The crossing is picked by its SENSE, so the one just
// taken (the point sits on it to rounding) is never taken again: it has the other sense now.
// K = the operand's kind at compile time (the distance kernels are instantiated per pair of kinds: straight-line code,
// no divergence between lanes over the kind), or -1 to read it from the record.
template <int K>
VG_DEV double solid_next(const SolidU &s, bool inside, double x, double y, double z, double dx, double dy, double dz)
{
    double t;
    switch (K < 0 ? s.kind : K) {
    case kBox: {
        double tin, tout;
        Box::slabs(s.u.box, x, y, z, dx, dy, dz, tin, tout);
        t = inside ? tout : ((tin < tout) ? tin : inf());
        break;
    }
    case kTrd: {
        double tin, tout;
        Trd::clip_all(s.u.trd, x, y, z, dx, dy, dz, tin, tout);
        t = inside ? tout : ((tin < tout) ? tin : inf());
        break;
    }
    case kOrb: { // a = 1: the entering root is -b - s, the leaving root -b + s
        const double pp = fma(x, x, fma(y, y, z * z)), b = fma(x, dx, fma(y, dy, z * dz));
        const double c = pp - s.u.orb.r2, D = fma(b, b, -c);
        t = D > 0.0 ? quad_root(1.0, b, c, sqrt_pos(D), inside) : inf();
        break;
    }
    case kTube: t = inside ? Tube::dist_out(s.u.tube, x, y, z, dx, dy, dz) : Tube::dist_in(s.u.tube, x, y, z, dx, dy, dz); break;
    default: t = inside ? Cone::dist_out(s.u.cone, x, y, z, dx, dy, dz) : Cone::dist_in(s.u.cone, x, y, z, dx, dy, dz); break;
    }
    return ahead(t) ? dmax(t, 0.0) : inf(); // a crossing behind the point, a wrong-side -1 or a NaN is "no crossing"
}

// ---- operands that may be polycones (X = true: vg_boolx.cu): kind == kPolycone reads the constants through u.pcon ----
template <bool X> VG_DEV int opnd_inside(const SolidU &s, double x, double y, double z)
{
    if (X && s.kind == kPolycone) return Polycone::inside(*s.u.pcon, x, y, z);
    return solid_inside(s, x, y, z);
}

template <bool X> VG_DEV double opnd_sdf(const SolidU &s, double x, double y, double z)
{
    if (X && s.kind == kPolycone) return Polycone::safety(*s.u.pcon, x, y, z);
    return solid_sdf(s, x, y, z);
}

template <int K, bool X>
VG_DEV double opnd_next(const SolidU &s, bool inside, double x, double y, double z, double dx, double dy, double dz)
{
    if (X && s.kind == kPolycone) { // the polycone's distances pick crossings by their sense, like every solid's (R32)
        const double t = inside ? Polycone::dist_out(*s.u.pcon, x, y, z, dx, dy, dz) : Polycone::dist_in(*s.u.pcon, x, y, z, dx, dy, dz);
        return ahead(t) ? dmax(t, 0.0) : inf();
    }
    return solid_next<K>(s, inside, x, y, z, dx, dy, dz);
}

VG_DEV bool bool_member(int op, bool ina, bool inb)
{
    return op == kUnion ? (ina || inb) : (op == kIntersection ? (ina && inb) : (ina && !inb));
}

VG_DEV int bool_classify(int op, int ca, int cb)
{
    const bool ain = ca == cInside, aout = ca == cOutside, bin = cb == cInside, bout = cb == cOutside;
    bool in, out;
    if (op == kUnion) in = ain || bin, out = aout && bout;
    else if (op == kIntersection) in = ain && bin, out = aout || bout;
    else in = ain && bout, out = aout || bin;
    return classify(in, out);
}

// ---- the three answers as device functions (the kernel below and the world kernels of vg_world.cu call them) ----

VG_DEV void bool_to_b(const BoolP &p, double x, double y, double z, double &bx, double &by, double &bz)
{
    const double *m = p.X;
    bx = fma(m[0], x, fma(m[1], y, fma(m[2], z, m[3])));
    by = fma(m[4], x, fma(m[5], y, fma(m[6], z, m[7])));
    bz = fma(m[8], x, fma(m[9], y, fma(m[10], z, m[11])));
}

template <bool X = false> VG_DEV int bool_inside_pt(const BoolP &p, double x, double y, double z) // R27
{
    double bx, by, bz;
    bool_to_b(p, x, y, z, bx, by, bz);
    return bool_classify(p.op, opnd_inside<X>(p.a, x, y, z), opnd_inside<X>(p.b, bx, by, bz));
}

template <bool X = false> VG_DEV double bool_sdf_pt(const BoolP &p, double x, double y, double z) // R29
{
    double bx, by, bz;
    bool_to_b(p, x, y, z, bx, by, bz);
    const double sa = opnd_sdf<X>(p.a, x, y, z), sb = opnd_sdf<X>(p.b, bx, by, bz);
    return p.op == kUnion ? dmin(sa, sb) : (p.op == kIntersection ? dmax(sa, sb) : dmax(sa, -sb));
}

// R28 / R32: DistanceToIn (to_out = false) or DistanceToOut (true): -1 on the wrong side, +inf if the membership never
// changes.  A state machine over (inside A, inside B, t): each operand is asked for its next crossing in the sense its
// state calls for, the nearer one is taken and flips that state; the answer is the first event after which C's
// membership is what the query looks for (a member for DistanceToIn, a non-member for DistanceToOut -- the class test
// has already sent the wrong side home, so the start value need not be read off the operands).  An operand whose class
// at the start is SURFACE has no state yet: it starts as "outside", and if its entering crossing is not AT the start
// (t <= kRayTol after the clamp) the crossing the point sits on is a leaving one and the operand was inside (R32: the
// sense of motion decides); that operand's event at t ~ 0 then runs through the loop like any other.
template <int KA, int KB, bool X = false>
VG_DEV double bool_distance(const BoolP &p, bool to_out, double x, double y, double z, double dx, double dy, double dz)
{
    const double *m = p.X;
    double bx, by, bz;
    bool_to_b(p, x, y, z, bx, by, bz);
    const int ca = opnd_inside<X>(p.a, x, y, z), cb = opnd_inside<X>(p.b, bx, by, bz);
    const int cls = bool_classify(p.op, ca, cb);
    if ((!to_out && cls == cInside) || (to_out && cls == cOutside)) return -1.0;
    const double bdx = fma(m[0], dx, fma(m[1], dy, m[2] * dz));
    const double bdy = fma(m[4], dx, fma(m[5], dy, m[6] * dz));
    const double bdz = fma(m[8], dx, fma(m[9], dy, m[10] * dz));
    bool ina = ca == cInside, inb = cb == cInside;
    bool pend_a = ca == cSurface, pend_b = cb == cSurface;
    double tt = 0.0;
    int last = 0;                 // the operand whose crossing the previous event was: 1 = A, 2 = B
    double offa = 0.0, offb = 0.0; // see below
#pragma unroll 1
    for (int it = 0; it < kBoolMaxEvents; ++it) {
        const double ta = tt + offa, tb = tt + offb;
        const double ea = offa + opnd_next<KA, X>(p.a, ina, fma(ta, dx, x), fma(ta, dy, y), fma(ta, dz, z), dx, dy, dz);
        const double eb = offb + opnd_next<KB, X>(p.b, inb, fma(tb, bdx, bx), fma(tb, bdy, by), fma(tb, bdz, bz), bdx, bdy, bdz);
        // An operand asked again from the very crossing it has just taken must answer with a LATER one.  It answers 0
        // when it has just been left through a chord shorter than kRayTol: the entering crossing, that little behind,
        // counts as lying at the start (R32), and the machine would enter and leave on the spot until the event limit.
        // A zero from the operand of the last event is asked again, once, from 2 kRayTol further on (a rare extra trip).
        if (last == 1 && offa == 0.0 && !(ea > 0.0)) {
            offa = 2.0 * kRayTol;
            continue;
        }
        if (last == 2 && offb == 0.0 && !(eb > 0.0)) {
            offb = 2.0 * kRayTol;
            continue;
        }
        offa = offb = 0.0;
        if (pend_a || pend_b) { // first pass only, and only for a start on an operand's surface
            const bool fix_a = pend_a && !(ea <= kRayTol), fix_b = pend_b && !(eb <= kRayTol);
            pend_a = pend_b = false;
            ina = ina || fix_a;
            inb = inb || fix_b;
            if (fix_a || fix_b) continue; // (last stays 0: no event yet)
        }
        const bool a_first = ea <= eb; // a tie goes to A, as in the oracle's merge
        const double e = a_first ? ea : eb;
        if (!(e < inf())) break;
        tt += e;
        ina = a_first ? !ina : ina;
        inb = a_first ? inb : !inb;
        last = a_first ? 1 : 2;
        if (bool_member(p.op, ina, inb) != to_out) return tt;
    }
    return inf();
}

#ifndef VG_BOOL_MINB
#define VG_BOOL_MINB 3
#endif

template <int Q, int KA, int KB, bool X = false>
__global__ void __launch_bounds__(kBoolBlock, (Q == qDistIn || Q == qDistOut) ? VG_BOOL_MINB : 1)
    bool_kernel(const __grid_constant__ BoolP p, Tracks t, double step_max, int64_t n, void *out)
{
    pdl_launch_dependents();
    pdl_wait();
    const int64_t i = int64_t(blockIdx.x) * kBoolBlock + threadIdx.x;
    if (i >= n) return;
    const double x = ldg1(t.x + i), y = ldg1(t.y + i), z = ldg1(t.z + i);
    if (Q == qSafeIn || Q == qSafeOut) {
        const double s = bool_sdf_pt<X>(p, x, y, z);
        stg1(static_cast<double *>(out) + i, Q == qSafeIn ? s : -s);
    } else if (Q == qInside) {
        stg1i(static_cast<int32_t *>(out) + i, bool_inside_pt<X>(p, x, y, z));
    } else {
        const double dx = ldg1(t.dx + i), dy = ldg1(t.dy + i), dz = ldg1(t.dz + i);
        const double r = bool_distance<KA, KB, X>(p, Q == qDistOut, x, y, z, dx, dy, dz);
        stg1(static_cast<double *>(out) + i, r <= step_max ? r : inf());
    }
}

// Inside and the safeties over 16-byte aligned arrays: two tracks per thread, 128-bit loads and stores as in the
// primitives' query_kernel (a warp reads 512 contiguous bytes per array).  The one-track form above took 35-38 us at
// 4 Mi tracks with a third of the DRAM rate: too few bytes in flight per warp for kernels this light.
#ifndef VG_BOOL_PT_BLOCK
#define VG_BOOL_PT_BLOCK 256
#endif
template <int Q, bool X = false>
__global__ void __launch_bounds__(VG_BOOL_PT_BLOCK)
    bool_point2_kernel(const __grid_constant__ BoolP p, Tracks t, int64_t n, void *out)
{
    static_assert(Q == qInside || Q == qSafeIn || Q == qSafeOut, "point queries only");
    pdl_launch_dependents();
    pdl_wait();
    const int64_t i = (int64_t(blockIdx.x) * VG_BOOL_PT_BLOCK + threadIdx.x) * 2;
    if (i >= n) return;
    if (i + 1 < n) {
        const double2 x = ldg2(t.x + i), y = ldg2(t.y + i), z = ldg2(t.z + i);
        if (Q == qInside) {
            stg2i(static_cast<int32_t *>(out) + i, bool_inside_pt<X>(p, x.x, y.x, z.x), bool_inside_pt<X>(p, x.y, y.y, z.y));
        } else {
            const double s0 = bool_sdf_pt<X>(p, x.x, y.x, z.x), s1 = bool_sdf_pt<X>(p, x.y, y.y, z.y);
            stg2(static_cast<double *>(out) + i, Q == qSafeIn ? s0 : -s0, Q == qSafeIn ? s1 : -s1);
        }
    } else { // the last track of an odd batch
        const double x = ldg1(t.x + i), y = ldg1(t.y + i), z = ldg1(t.z + i);
        if (Q == qInside) {
            stg1i(static_cast<int32_t *>(out) + i, bool_inside_pt<X>(p, x, y, z));
        } else {
            const double s = bool_sdf_pt<X>(p, x, y, z);
            stg1(static_cast<double *>(out) + i, Q == qSafeIn ? s : -s);
        }
    }
}

template <int Q, bool X = false>
cudaError_t launch_bool_point2(const BoolP &p, const Tracks &t, int64_t n, void *out, cudaStream_t s)
{
    const int64_t threads = (n + 1) / 2;
    return launch_kernel(bool_point2_kernel<Q, X>, unsigned((threads + VG_BOOL_PT_BLOCK - 1) / VG_BOOL_PT_BLOCK), VG_BOOL_PT_BLOCK, 0, s, p, t, n, out);
}

// the two distance kernels for operand kinds (A, kb), kb at run time: one plain function per kind of A, each defined in
// its own translation unit vg_bool_k<A>.cu
#define VG_BOOL_DECLARE_DIST(NAME)                                                                                     \
    cudaError_t launch_boolean_dist_##NAME(int q, int kb, const BoolP &p, const Tracks &t, double step_max, int64_t n, \
                                           void *out, unsigned grid, cudaStream_t s);
VG_BOOL_DECLARE_DIST(kBox)
VG_BOOL_DECLARE_DIST(kOrb)
VG_BOOL_DECLARE_DIST(kTube)
VG_BOOL_DECLARE_DIST(kCone)
VG_BOOL_DECLARE_DIST(kTrd)

template <int Q, int KA>
cudaError_t launch_boolean_dist_b(int kb, const BoolP &p, const Tracks &t, double step_max, int64_t n, void *out, unsigned grid,
                                  cudaStream_t s)
{
    switch (kb) {
    case kBox: return launch_kernel(bool_kernel<Q, KA, kBox>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    case kOrb: return launch_kernel(bool_kernel<Q, KA, kOrb>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    case kTube: return launch_kernel(bool_kernel<Q, KA, kTube>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    case kCone: return launch_kernel(bool_kernel<Q, KA, kCone>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    case kTrd: return launch_kernel(bool_kernel<Q, KA, kTrd>, grid, kBoolBlock, 0, s, p, t, step_max, n, out);
    }
    return cudaErrorInvalidValue;
}

#define VG_BOOL_DEFINE_DIST(NAME)                                                                                      \
    cudaError_t launch_boolean_dist_##NAME(int q, int kb, const BoolP &p, const Tracks &t, double step_max, int64_t n, \
                                           void *out, unsigned grid, cudaStream_t s)                                   \
    {                                                                                                                  \
        return q == qDistIn ? launch_boolean_dist_b<qDistIn, NAME>(kb, p, t, step_max, n, out, grid, s)                \
                            : launch_boolean_dist_b<qDistOut, NAME>(kb, p, t, step_max, n, out, grid, s);              \
    }

} // namespace vg
