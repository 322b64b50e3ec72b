// vg_csg.cuh -- device code of the nested booleans (reading R31); see vg_csg.cu for the design.
#pragma once
#include "vg_bool.cuh"

namespace vg {

constexpr int kCsgMaxEvents = 16 * kCsgMaxLeaf;

// the tree's membership from one bit per primitive; the stack lives in the bits of `st`
VG_DEV bool csg_member(const CsgP &p, unsigned bits)
{
    unsigned st = 0;
    int sp = 0;
#pragma unroll 1
    for (int k = 0; k < p.nprog; ++k) {
        const unsigned tok = p.prog[k];
        if (tok < 0x80u) {
            st = (st & ~(1u << sp)) | (((bits >> tok) & 1u) << sp);
            ++sp;
        } else {
            const bool b = (st >> (sp - 1)) & 1u, a = (st >> (sp - 2)) & 1u;
            const bool r = bool_member(int(tok & 0x7fu), a, b);
            sp -= 1;
            st = (st & ~(1u << (sp - 1))) | (unsigned(r) << (sp - 1));
        }
    }
    return st & 1u;
}

VG_DEV void csg_to_leaf(const double *m, double x, double y, double z, double &lx, double &ly, double &lz)
{
    lx = fma(m[0], x, fma(m[1], y, fma(m[2], z, m[3])));
    ly = fma(m[4], x, fma(m[5], y, fma(m[6], z, m[7])));
    lz = fma(m[8], x, fma(m[9], y, fma(m[10], z, m[11])));
}

// classes of all primitives as two bit sets (strictly inside / strictly outside)
VG_DEV void csg_classes(const CsgP &p, double x, double y, double z, unsigned &in, unsigned &out)
{
    in = out = 0;
#pragma unroll 1
    for (int i = 0; i < p.nleaf; ++i) {
        double lx, ly, lz;
        csg_to_leaf(p.X[i], x, y, z, lx, ly, lz);
        const int c = solid_inside(p.leaf[i], lx, ly, lz);
        in |= unsigned(c == cInside) << i;
        out |= unsigned(c == cOutside) << i;
    }
}

// R27 read recursively: the program on (in, out) pairs
VG_DEV int csg_classify(const CsgP &p, unsigned in, unsigned out)
{
    unsigned sin = 0, sout = 0;
    int sp = 0;
#pragma unroll 1
    for (int k = 0; k < p.nprog; ++k) {
        const unsigned tok = p.prog[k];
        if (tok < 0x80u) {
            sin = (sin & ~(1u << sp)) | (((in >> tok) & 1u) << sp);
            sout = (sout & ~(1u << sp)) | (((out >> tok) & 1u) << sp);
            ++sp;
        } else {
            const bool bin = (sin >> (sp - 1)) & 1u, bout = (sout >> (sp - 1)) & 1u;
            const bool ain = (sin >> (sp - 2)) & 1u, aout = (sout >> (sp - 2)) & 1u;
            const int op = int(tok & 0x7fu);
            bool rin, rout;
            if (op == kUnion) rin = ain || bin, rout = aout && bout;
            else if (op == kIntersection) rin = ain && bin, rout = aout || bout;
            else rin = ain && bout, rout = aout || bin;
            sp -= 1;
            sin = (sin & ~(1u << (sp - 1))) | (unsigned(rin) << (sp - 1));
            sout = (sout & ~(1u << (sp - 1))) | (unsigned(rout) << (sp - 1));
        }
    }
    return classify(sin & 1u, sout & 1u);
}

// R29 read recursively: the program on signed distances
VG_DEV double csg_sdf(const CsgP &p, double x, double y, double z)
{
    double st[kCsgMaxLeaf];
    int sp = 0;
#pragma unroll 1
    for (int k = 0; k < p.nprog; ++k) {
        const unsigned tok = p.prog[k];
        if (tok < 0x80u) {
            double lx, ly, lz;
            csg_to_leaf(p.X[tok], x, y, z, lx, ly, lz);
            st[sp++] = solid_sdf(p.leaf[tok], lx, ly, lz);
        } else {
            const double b = st[sp - 1], a = st[sp - 2];
            const int op = int(tok & 0x7fu);
            sp -= 1;
            st[sp - 1] = op == kUnion ? dmin(a, b) : (op == kIntersection ? dmax(a, b) : dmax(a, -b));
        }
    }
    return st[0];
}

// next crossing of primitive i in the sense of its bit, seen from the point at ray parameter tt; +inf if none
VG_DEV double csg_leaf_next(const CsgP &p, int i, bool inside, double tt, double x, double y, double z, double dx, double dy,
                            double dz)
{
    const double *m = p.X[i];
    double lx, ly, lz;
    csg_to_leaf(m, fma(tt, dx, x), fma(tt, dy, y), fma(tt, dz, z), lx, ly, lz);
    const double ldx = fma(m[0], dx, fma(m[1], dy, m[2] * dz));
    const double ldy = fma(m[4], dx, fma(m[5], dy, m[6] * dz));
    const double ldz = fma(m[8], dx, fma(m[9], dy, m[10] * dz));
    return solid_next<-1>(p.leaf[i], inside, lx, ly, lz, ldx, ldy, ldz);
}

// R28 / R32 read recursively: the state machine of bool_distance over one "inside" bit per primitive; primitives whose
// class at the start is SURFACE get their bit from the sense of motion in the first pass.  Every primitive's NEXT
// crossing (an absolute ray parameter) is kept: an event flips one primitive, and only that one is asked again -- the
// others' next crossings lie at or beyond the event and stay valid.  nleaf + events solid evaluations instead of
// nleaf x events (698 -> 417 us for the four-primitive tree of bench.py at 4 Mi tracks).
VG_DEV double csg_distance(const CsgP &p, bool to_out, double x, double y, double z, double dx, double dy, double dz)
{
    unsigned in, out;
    csg_classes(p, x, y, z, in, out);
    const int cls = csg_classify(p, in, out);
    if ((!to_out && cls == cInside) || (to_out && cls == cOutside)) return -1.0;
    unsigned bits = in;
    const unsigned pend = ~(in | out) & ((1u << p.nleaf) - 1u);
    double tn[kCsgMaxLeaf];
    unsigned fix = 0;
#pragma unroll 1
    for (int i = 0; i < p.nleaf; ++i) {
        const double e = csg_leaf_next(p, i, (bits >> i) & 1u, 0.0, x, y, z, dx, dy, dz);
        fix |= unsigned(((pend >> i) & 1u) && !(e <= kRayTol)) << i;
        tn[i] = e;
    }
    if (fix) { // those primitives are being left, not entered: they were inside; ask them for the crossing they sit on
        bits |= fix;
#pragma unroll 1
        for (int i = 0; i < p.nleaf; ++i)
            if ((fix >> i) & 1u) tn[i] = csg_leaf_next(p, i, true, 0.0, x, y, z, dx, dy, dz);
    }
#pragma unroll 1
    for (int it = 0; it < kCsgMaxEvents; ++it) {
        double emin = inf();
        int imin = -1;
#pragma unroll 1
        for (int i = 0; i < p.nleaf; ++i)
            if (tn[i] < emin) emin = tn[i], imin = i; // strict: the lowest leaf wins a tie
        if (imin < 0) break;
        bits ^= 1u << imin;
        if (csg_member(p, bits) != to_out) return emin;
        // the primitive's next crossing must lie beyond the one just taken: a zero (it has just been left through a chord
        // shorter than kRayTol, and the entering crossing that little behind counts as lying at the start, R32) is asked
        // again from 2 kRayTol further on, or the machine would enter and leave on the spot until the event limit
        double nx = csg_leaf_next(p, imin, (bits >> imin) & 1u, emin, x, y, z, dx, dy, dz);
        if (!(nx > 0.0)) nx = 2.0 * kRayTol + csg_leaf_next(p, imin, (bits >> imin) & 1u, emin + 2.0 * kRayTol, x, y, z, dx, dy, dz);
        tn[imin] = emin + nx;
    }
    return inf();
}

} // namespace vg
