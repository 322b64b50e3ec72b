// vg_shapes.cuh -- per-solid device code: Inside, exact signed distance (safeties), DistanceToIn, DistanceToOut.
//
// Semantics: SURVEY.md sec. 8(c) c.1-c.4 and readings R1-R21 (the paper names the three questions only,
// PAPER.md:110-114).  Unlike the oracle (brute force over every boundary patch, both roots, atan2), the code
// here is specialised per solid and evaluates only the crossings that CAN be the answer:
//   * DistanceToIn looks only at crossings in the entering sense, DistanceToOut only in the leaving sense
//     (for a surface F(t) = a t^2 + 2 b t + c with the material on the F < 0 side, the entering root is
//     (-b - sqrt(D))/a and the leaving root (-b + sqrt(D))/a for either sign of a);
//   * the phi test is two cross products with the stored plane vectors instead of atan2;
//   * everything is select-based (no data-dependent branch inside a solid), zero direction components are
//     replaced by +-1e-300 so that no 0/0 or inf-inf can arise (R9, hard part H4);
//   * `valid` flags are conjunctions of positive comparisons, so a NaN candidate is always discarded.
// Inside uses per-surface tolerance tests (an L-infinity band); it equals the oracle's Euclidean band except
// for points within [kTol, sqrt(3) kTol] of an edge, which the parity contract excludes (R6).
// Start points in the surface band (R32): a crossing of the wanted sense counts when ahead(t) (t > -kRayTol) and every
// distance is clamped at 0, so a surface point moving inward has DistanceToIn 0 and DistanceToOut = its chord, and
// one moving outward DistanceToOut 0 and DistanceToIn = the next entry.
#pragma once
#include "vg_math.cuh"
#include "vg_params.h"

namespace vg {

enum : int { cOutside = 0, cSurface = 1, cInside = 2 };

VG_DEV int classify(bool in, bool out) { return in ? cInside : (out ? cOutside : cSurface); }

// ------------------------------------------------------------------------------------------------ phi wedge
//
// The solids with a phi cut (tube, cone, polycone) exist in a run-time form (flags read from the constants: the
// navigator's daughters) and in compile-time specialisations that the streaming kernels are instantiated with, so
// that their code is straight-line: WM = -1 reads w.full / w.wide, 0 = full (no cut), 1 = dphi <= pi, 2 = dphi > pi.
constexpr int kWmRuntime = -1, kWmFull = 0, kWmNarrow = 1, kWmWide = 2;

template <int WM> VG_DEV bool w_full(const Wedge &w) { return WM < 0 ? w.full != 0 : WM == kWmFull; }
template <int WM> VG_DEV bool w_wide(const Wedge &w) { return WM < 0 ? w.wide != 0 : WM == kWmWide; }

struct WedgeEval {
    double c0, c1; // signed distances into the segment from plane 0 / plane 1 (>= 0 on the material side)
    double u0, u1; // coordinates along the two bounding half-planes (>= 0 on the half-plane itself)
};

// linear in (x, y): the same function gives the rates of c and u along a direction
VG_DEV WedgeEval wedge_eval(const Wedge &w, double x, double y)
{
    WedgeEval e;
    e.c0 = fma(w.e0x, y, -w.e0y * x);
    e.c1 = fma(w.e1y, x, -w.e1x * y);
    e.u0 = fma(w.e0x, x, w.e0y * y);
    e.u1 = fma(w.e1x, x, w.e1y * y);
    return e;
}

template <int WM> VG_DEV bool wedge_member(const Wedge &w, double c0, double c1)
{
    return w_wide<WM>(w) ? (c0 >= 0.0 || c1 >= 0.0) : (c0 >= 0.0 && c1 >= 0.0);
}

// is the point p + t d inside the segment?  c is linear along the ray: c(t) = c(p) + t c(d)
template <int WM> VG_DEV bool wedge_member_at(const Wedge &w, const WedgeEval &ep, const WedgeEval &ed, double t)
{
    return wedge_member<WM>(w, fma(t, ed.c0, ep.c0), fma(t, ed.c1, ep.c1));
}

// squared distance from (x, y) to the nearer of the two bounding half-planes (not the full planes)
VG_DEV double wedge_clear2(const WedgeEval &e, double rho2)
{
    double f0 = e.u0 >= 0.0 ? e.c0 * e.c0 : rho2;
    double f1 = e.u1 >= 0.0 ? e.c1 * e.c1 : rho2;
    return dmin(f0, f1);
}

template <int WM> VG_DEV void wedge_classify(const Wedge &w, const WedgeEval &e, double rho2, bool &in, bool &out)
{
    bool mem = wedge_member<WM>(w, e.c0, e.c1);
    bool clear = wedge_clear2(e, rho2) > kTol * kTol;
    in = in && mem && clear;
    out = out || (!mem && clear);
}

// squared distance from (u, v) to the segment (r0, z0) + t (er, ez), t in [0, 1]
VG_DEV double seg_d2(double u, double v, double r0, double z0, double er, double ez, double inv_l2)
{
    double wu = u - r0, wv = v - z0;
    double t = fma(wu, er, wv * ez) * inv_l2;
    t = dmin(dmax(t, 0.0), 1.0);
    double du = fma(-t, er, wu), dv = fma(-t, ez, wv);
    return fma(du, du, dv * dv);
}

// one root of a t^2 + 2 b t + c = 0 chosen by the sign of F' there: leaving = false gives the root with
// F' < 0 ((-b - s)/a), leaving = true the root with F' > 0 ((-b + s)/a).  Evaluated as q/a or c/q with
// q = -(b + sgn(b) s), whichever does not cancel, so it stays accurate for a -> 0 (ray along a generator).
// Returns NaN/inf garbage when D <= 0; the caller tests D > 0.
VG_DEV double quad_root(double a, double b, double c, double s, bool leaving)
{
    bool bpos = not_neg(b); // the SIGN BIT, as copysign_bits reads it: b = -0.0 (a point on the axis of a cylinder) must
                            // take the same branch here and there, or the two roots swap and the hit is lost
    double q = -(b + copysign_bits(s, b));
    // bpos: q = -(b+s): (-b - s)/a = q/a, (-b + s)/a = c/q.   !bpos: q = -b + s: (-b + s)/a = q/a, (-b - s)/a = c/q
    bool use_qa = (bpos != leaving);
    double num = use_qa ? q : c;
    double den = use_qa ? a : q;
    return num * rcp(den);
}

// ------------------------------------------------------------------------------------------------------ box

struct Box {
    using P = BoxP;

    VG_DEV static void slack(const P &p, double x, double y, double z, double &m, double &s2)
    {
        double qx = fabs(x) - p.hx, qy = fabs(y) - p.hy, qz = fabs(z) - p.hz;
        m = dmax(dmax(qx, qy), qz);
        double ax = dmax(qx, 0.0), ay = dmax(qy, 0.0), az = dmax(qz, 0.0);
        s2 = fma(ax, ax, fma(ay, ay, az * az));
    }
    VG_DEV static int inside(const P &p, double x, double y, double z)
    {
        double m, s2;
        slack(p, x, y, z, m, s2);
        return classify(m < -kTol, s2 > kTol * kTol);
    }
    // c.3: sdf = |max(q, 0)| + min(max(qx, qy, qz), 0)
    VG_DEV static double safety(const P &p, double x, double y, double z)
    {
        double m, s2;
        slack(p, x, y, z, m, s2);
        return m > 0.0 ? sqrt_pos(s2) : m;
    }
    // c.4 slabs, written for the direction folded to d >= 0: t1 = (-h - p s)/|d|, t2 = (h - p s)/|d|
    VG_DEV static void slabs(const P &p, double x, double y, double z, double dx, double dy, double dz, double &tin,
                             double &tout)
    {
        double ix = rcp(fabs(nonzero(dx))), iy = rcp(fabs(nonzero(dy))), iz = rcp(fabs(nonzero(dz)));
        double px = flipsign_bits(x, dx), py = flipsign_bits(y, dy), pz = flipsign_bits(z, dz);
        double hx = p.hx * ix, hy = p.hy * iy, hz = p.hz * iz;
        double t1x = fma(-px, ix, -hx), t2x = fma(-px, ix, hx);
        double t1y = fma(-py, iy, -hy), t2y = fma(-py, iy, hy);
        double t1z = fma(-pz, iz, -hz), t2z = fma(-pz, iz, hz);
        tin = dmax(dmax(t1x, t1y), t1z);
        tout = dmin(dmin(t2x, t2y), t2z);
    }
    VG_DEV static double dist_in(const P &p, double x, double y, double z, double dx, double dy, double dz)
    {
        double m, s2, tin, tout;
        slack(p, x, y, z, m, s2);
        slabs(p, x, y, z, dx, dy, dz, tin, tout);
        double t = (tin < tout && ahead(tin)) ? dmax(tin, 0.0) : inf(); // an outside point with tin < tout has tin > 0
        return m < -kTol ? -1.0 : t;
    }
    VG_DEV static double dist_out(const P &p, double x, double y, double z, double dx, double dy, double dz)
    {
        double m, s2, tin, tout;
        slack(p, x, y, z, m, s2);
        slabs(p, x, y, z, dx, dy, dz, tin, tout);
        return s2 > kTol * kTol ? -1.0 : dmax(tout, 0.0);
    }
};

// ------------------------------------------------------------------------------------------------------ orb

struct Orb {
    using P = OrbP;

    VG_DEV static int inside(const P &p, double x, double y, double z)
    {
        double pp = fma(x, x, fma(y, y, z * z));
        return classify(pp < p.rin2, pp > p.rout2);
    }
    VG_DEV static double safety(const P &p, double x, double y, double z)
    {
        double pp = fma(x, x, fma(y, y, z * z));
        return sqrt_nn(pp) - p.r;
    }
    // c.4: a = 1, b = p.d, c = p.p - r^2.  The crossing is picked by its SENSE, not as the smallest positive root: the
    // entering root is -b - s, the leaving root -b + s (evaluated as q or c/q, whichever does not cancel), so a track that
    // sits on the sphere to rounding sees the crossing it sits on only in the query whose sense it has (R32).
    VG_DEV static double root(const P &p, double pp, double b, bool leaving)
    {
        double c = pp - p.r2;
        double D = fma(b, b, -c);
        double t = quad_root(1.0, b, c, sqrt_pos(D), leaving);
        return (D > 0.0 && ahead(t)) ? dmax(t, 0.0) : inf();
    }
    VG_DEV static double dist_in(const P &p, double x, double y, double z, double dx, double dy, double dz)
    {
        double pp = fma(x, x, fma(y, y, z * z));
        double b = fma(x, dx, fma(y, dy, z * dz));
        double t = root(p, pp, b, false);
        return pp < p.rin2 ? -1.0 : t;
    }
    VG_DEV static double dist_out(const P &p, double x, double y, double z, double dx, double dy, double dz)
    {
        double pp = fma(x, x, fma(y, y, z * z));
        double b = fma(x, dx, fma(y, dy, z * dz));
        double t = root(p, pp, b, true);
        return pp > p.rout2 ? -1.0 : t;
    }
};

// ----------------------------------------------------------------------------------------------------- tube

// F = -1: flags read at run time (navigator daughters); F >= 0: bit 0 = hollow, bits 1.. = wedge mode (kWm*)
constexpr int kFlagsRuntime = -1;
constexpr int solid_flags(bool hollow, int wm) { return (hollow ? 1 : 0) | (wm << 1); }

template <int F> struct TubeT {
    using P = TubeP;
    static constexpr int WM = F < 0 ? kWmRuntime : (F >> 1);
    VG_DEV static bool hollow(const P &p) { return F < 0 ? p.hollow != 0 : (F & 1) != 0; }
    VG_DEV static bool full(const P &p) { return w_full<WM>(p.w); }

    VG_DEV static void classify_pt(const P &p, double x, double y, double z, double rho2, const WedgeEval &ep, bool &in,
                                   bool &out)
    {
        double az = fabs(z);
        in = az < p.dz - kTol && rho2 < p.rmax_in2;
        out = az > p.dz + kTol || rho2 > p.rmax_out2;
        if (hollow(p)) {
            in = in && rho2 > p.rmin_in2;
            out = out || rho2 < p.rmin_out2;
        }
        if (!full(p)) wedge_classify<WM>(p.w, ep, rho2, in, out);
    }
    VG_DEV static int inside(const P &p, double x, double y, double z)
    {
        bool in, out;
        WedgeEval ep = {};
        if (!full(p)) ep = wedge_eval(p.w, x, y);
        classify_pt(p, x, y, z, fma(x, x, y * y), ep, in, out);
        return classify(in, out);
    }
    // c.3 for the rectangle [rmin, rmax] x [-dz, dz] in (rho, z) cut by the phi segment
    VG_DEV static double safety(const P &p, double x, double y, double z)
    {
        double rho2 = fma(x, x, y * y);
        double rho = sqrt_nn(rho2);
        // distance to an interval [lo, hi] as max(|u - c| - h, 0) (one compare less than max(lo - u, u - hi, 0)); the square
        // of max(q, 0) as (q + |q|)^2 / 4 (no compare at all)
        double qr = hollow(p) ? fabs(rho - p.rc) - p.rh : rho - p.rmax;
        double qz = fabs(z) - p.dz;
        double sr = qr + fabs(qr), sz = qz + fabs(qz);
        double az2 = 0.25 * sz * sz;
        double out2 = fma(0.25 * sr, sr, az2);
        double m = dmax(qr, qz);
        bool in_rect = m < 0.0;
        if (full(p)) return in_rect ? m : sqrt_nn(out2);
        double D2 = in_rect ? m * m : out2;
        WedgeEval e = wedge_eval(p.w, x, y);
        bool mem = wedge_member<WM>(p.w, e.c0, e.c1);
        D2 = mem ? D2 : inf();
        // the two phi faces: filled rectangle [rmin, rmax] x [-dz, dz] in the half-plane (u >= 0)
        double q0 = fabs(e.u0 - p.rc) - p.rh, q1 = fabs(e.u1 - p.rc) - p.rh;
        double s0 = q0 + fabs(q0), s1 = q1 + fabs(q1);
        D2 = dmin(D2, fma(e.c0, e.c0, fma(0.25 * s0, s0, az2)));
        D2 = dmin(D2, fma(e.c1, e.c1, fma(0.25 * s1, s1, az2)));
        double D = sqrt_nn(D2);
        return (mem && in_rect) ? -D : D;
    }

    // Every candidate carries its own validity tests, so a zero denominator needs no special case: rcp(0) is NaN
    // after the refinement, the candidate's t is NaN and fails its tests (a ray parallel to a surface does not
    // cross it, R8).  Hit points are tested against the phi segment with c(t) = c(p) + t c(d) (linear along the ray).
    VG_DEV static double dist_in(const P &p, double x, double y, double z, double dx, double dy, double dz)
    {
        bool in, out;
        double rho2 = fma(x, x, y * y);
        WedgeEval ep = {}, ed = {};
        if (!full(p)) ep = wedge_eval(p.w, x, y), ed = wedge_eval(p.w, dx, dy);
        classify_pt(p, x, y, z, rho2, ep, in, out);
        double a = fma(dx, dx, dy * dy);
        double b = fma(x, dx, y * dy);
        double inv_a = rcp(a);
        double best = inf();
        // outer cylinder, entering root
        {
            double D = fma(b, b, -a * (rho2 - p.rmax2));
            double t = (-b - sqrt_pos(D)) * inv_a;
            bool ok = D > 0.0 && ahead(t) && fabs(fma(t, dz, z)) <= p.dz;
            if (!full(p)) ok = ok && wedge_member_at<WM>(p.w, ep, ed, t);
            best = ok ? t : best;
        }
        // inner cylinder: the ray enters the material where it LEAVES the bore
        if (hollow(p)) {
            double D = fma(b, b, -a * (rho2 - p.rmin2));
            double t = (sqrt_pos(D) - b) * inv_a;
            bool ok = D > 0.0 && ahead(t) && fabs(fma(t, dz, z)) <= p.dz;
            if (!full(p)) ok = ok && wedge_member_at<WM>(p.w, ep, ed, t);
            best = (ok && t < best) ? t : best;
        }
        // the cap the ray moves towards, from beyond it or from on it (R32); rho_hit^2 = rho^2 + 2 b t + a t^2
        {
            double az = fabs(z);
            double t = (az - p.dz) * rcp(fabs(dz));
            double rh2 = fma(t, fma(t, a, b + b), rho2);
            bool ok = ahead(t) && sign_differs(z, dz) && rh2 >= p.rmin2 && rh2 <= p.rmax2;
            if (!full(p)) ok = ok && wedge_member_at<WM>(p.w, ep, ed, t);
            best = (ok && t < best) ? t : best;
        }
        // phi faces, entering sense: c_k(d) > 0, from behind the plane or from on it (R32)
        if (!full(p)) {
            {
                double t = -ep.c0 * rcp(ed.c0);
                double uh = fma(t, ed.u0, ep.u0);
                bool ok = ed.c0 > 0.0 && ahead(t) && uh >= p.rmin && uh <= p.rmax && fabs(fma(t, dz, z)) <= p.dz;
                best = (ok && t < best) ? t : best;
            }
            {
                double t = -ep.c1 * rcp(ed.c1);
                double uh = fma(t, ed.u1, ep.u1);
                bool ok = ed.c1 > 0.0 && ahead(t) && uh >= p.rmin && uh <= p.rmax && fabs(fma(t, dz, z)) <= p.dz;
                best = (ok && t < best) ? t : best;
            }
        }
        return in ? -1.0 : dmax(best, 0.0);
    }

    VG_DEV static double dist_out(const P &p, double x, double y, double z, double dx, double dy, double dz)
    {
        bool in, out;
        double rho2 = fma(x, x, y * y);
        WedgeEval ep = {}, ed = {};
        if (!full(p)) ep = wedge_eval(p.w, x, y), ed = wedge_eval(p.w, dx, dy);
        classify_pt(p, x, y, z, rho2, ep, in, out);
        double a = fma(dx, dx, dy * dy);
        double b = fma(x, dx, y * dy);
        double inv_a = rcp(a);
        double best = inf();
        {
            double D = fma(b, b, -a * (rho2 - p.rmax2));
            double t = (sqrt_pos(D) - b) * inv_a;
            best = (D > 0.0 && ahead(t)) ? t : best;
        }
        if (hollow(p)) { // the ray leaves the material where it ENTERS the bore: (-b - s)/a, which needs b < 0 to lie ahead
            double D = fma(b, b, -a * (rho2 - p.rmin2));
            double t = (-b - sqrt_pos(D)) * inv_a;
            best = (D > 0.0 && b < 0.0 && ahead(t) && t < best) ? t : best;
        }
        {
            double t = (p.dz - flipsign_bits(z, dz)) * rcp(fabs(dz));
            best = (ahead(t) && t < best) ? t : best;
        }
        if (!full(p)) {
            {
                double t = -ep.c0 * rcp(ed.c0);
                bool ok = ed.c0 < 0.0 && ahead(t) && fma(t, ed.u0, ep.u0) >= 0.0;
                best = (ok && t < best) ? t : best;
            }
            {
                double t = -ep.c1 * rcp(ed.c1);
                bool ok = ed.c1 < 0.0 && ahead(t) && fma(t, ed.u1, ep.u1) >= 0.0;
                best = (ok && t < best) ? t : best;
            }
        }
        return out ? -1.0 : dmax(best, 0.0);
    }
};
using Tube = TubeT<kFlagsRuntime>;

// ------------------------------------------------------------------------------- conical patches (cone, polycone)

// coefficients of F(t) = rho(t)^2 - k(t)^2 on the ray, k = A + B z (c.4 "slanted or vertical edge")
struct RayRZ {
    double rho2, a_xy, b_xy; // x^2+y^2, dx^2+dy^2, x dx + y dy
};

VG_DEV double frustum_root(const Frustum &f, const RayRZ &r, double z, double dz, bool leaving, bool &ok)
{
    double k = fma(f.B, z, f.A);
    double Bd = f.B * dz;
    double a = fma(-Bd, Bd, r.a_xy);
    double b = fma(-Bd, k, r.b_xy);
    double c = fma(-k, k, r.rho2);
    double D = fma(b, b, -a * c);
    double t = quad_root(a, b, c, sqrt_pos(D), leaving);
    ok = D > 0.0 && ahead(t);
    return t;
}

// ----------------------------------------------------------------------------------------------------- cone

template <int F> struct ConeT {
    using P = ConeP;
    static constexpr int WM = F < 0 ? kWmRuntime : (F >> 1);
    VG_DEV static bool hollow(const P &p) { return F < 0 ? p.hollow != 0 : (F & 1) != 0; }
    VG_DEV static bool full(const P &p) { return w_full<WM>(p.w); }

    VG_DEV static void classify_pt(const P &p, double x, double y, double z, double rho2, const WedgeEval &ep, bool &in,
                                   bool &out)
    {
        double az = fabs(z);
        double ro = fma(p.out.B, z, p.out.A), to = kTol * p.out.sec;
        double ro_in = ro - to, ro_out = ro + to;
        in = az < p.dz - kTol && ro_in > 0.0 && rho2 < ro_in * ro_in;
        out = az > p.dz + kTol || rho2 > ro_out * ro_out;
        if (hollow(p)) {
            double ri = fma(p.in.B, z, p.in.A), ti = kTol * p.in.sec;
            double ri_in = ri + ti, ri_out = ri - ti;
            in = in && (ri_in < 0.0 || rho2 > ri_in * ri_in);
            out = out || (ri_out > 0.0 && rho2 < ri_out * ri_out);
        }
        if (!full(p)) wedge_classify<WM>(p.w, ep, rho2, in, out);
    }
    VG_DEV static int inside(const P &p, double x, double y, double z)
    {
        bool in, out;
        WedgeEval ep = {};
        if (!full(p)) ep = wedge_eval(p.w, x, y);
        classify_pt(p, x, y, z, fma(x, x, y * y), ep, in, out);
        return classify(in, out);
    }
    // squared distance from (u, v) to the outline of the quadrilateral; `axis` adds the edge on the axis
    // (part of a phi face, not of the surface of revolution) when rmin1 = rmin2 = 0
    VG_DEV static double outline_d2(const P &p, double u, double v, bool axis)
    {
        double ez = 2.0 * p.dz;
        double d2 = seg_d2(u, v, p.out.r0, -p.dz, p.out.er, ez, p.out.inv_l2);
        if (hollow(p) || axis) d2 = dmin(d2, seg_d2(u, v, p.in.r0, -p.dz, p.in.er, ez, p.in.inv_l2));
        // The cap on the point's side of the mid-plane only: the other cap cannot hold the nearest point in its interior
        // (the vertical segment to it comes from inside the outline, so it has crossed a nearer edge), and its rims are
        // end points of the two edges above.  Distance to the annulus [rmin, rmax] as max(|u - c| - h, 0); its square
        // from s = q + |q| = 2 max(q, 0) without a compare.
        const bool top = not_neg(v);
        double q = fabs(u - (top ? p.cap_c2 : p.cap_c1)) - (top ? p.cap_h2 : p.cap_h1);
        double s = q + fabs(q), vc = fabs(v) - p.dz;
        d2 = dmin(d2, fma(0.25 * s, s, vc * vc));
        return d2;
    }
    VG_DEV static bool in_quad(const P &p, double u, double v)
    {
        double ro = fma(p.out.B, v, p.out.A), ri = fma(p.in.B, v, p.in.A);
        return fabs(v) < p.dz && u < ro && u > ri;
    }
    VG_DEV static double safety(const P &p, double x, double y, double z)
    {
        double rho2 = fma(x, x, y * y);
        double rho = sqrt_nn(rho2);
        double ro = fma(p.out.B, z, p.out.A), ri = fma(p.in.B, z, p.in.A);
        bool in2d = fabs(z) < p.dz && rho < ro && (rho > ri || !hollow(p));
        double D2 = outline_d2(p, rho, z, false);
        if (full(p)) {
            double D = sqrt_nn(D2);
            return in2d ? -D : D;
        }
        WedgeEval e = wedge_eval(p.w, x, y);
        bool mem = wedge_member<WM>(p.w, e.c0, e.c1);
        D2 = mem ? D2 : inf();
        double f0 = in_quad(p, e.u0, z) ? 0.0 : outline_d2(p, e.u0, z, true);
        double f1 = in_quad(p, e.u1, z) ? 0.0 : outline_d2(p, e.u1, z, true);
        D2 = dmin(D2, fma(e.c0, e.c0, f0));
        D2 = dmin(D2, fma(e.c1, e.c1, f1));
        double D = sqrt_nn(D2);
        return (mem && in2d) ? -D : D;
    }

    VG_DEV static double dist_in(const P &p, double x, double y, double z, double dx, double dy, double dz)
    {
        bool in, out;
        RayRZ r;
        r.rho2 = fma(x, x, y * y);
        WedgeEval ep = {}, ed = {};
        if (!full(p)) ep = wedge_eval(p.w, x, y), ed = wedge_eval(p.w, dx, dy);
        classify_pt(p, x, y, z, r.rho2, ep, in, out);
        r.a_xy = fma(dx, dx, dy * dy);
        r.b_xy = fma(x, dx, y * dy);
        double best = inf();
        {
            bool ok;
            double t = frustum_root(p.out, r, z, dz, false, ok);
            ok = ok && fabs(fma(t, dz, z)) <= p.dz;
            if (!full(p)) ok = ok && wedge_member_at<WM>(p.w, ep, ed, t);
            best = ok ? t : best;
        }
        if (hollow(p)) {
            bool ok;
            double t = frustum_root(p.in, r, z, dz, true, ok);
            ok = ok && fabs(fma(t, dz, z)) <= p.dz;
            if (!full(p)) ok = ok && wedge_member_at<WM>(p.w, ep, ed, t);
            best = (ok && t < best) ? t : best;
        }
        {
            double az = fabs(z);
            double t = (az - p.dz) * rcp(fabs(dz)); // > 0 from beyond the cap, ~0 from on it (R32); NaN (rejected) for dz = 0
            double rh2 = fma(t, fma(t, r.a_xy, r.b_xy + r.b_xy), r.rho2);
            bool top = z > 0.0;
            double rlo = top ? p.rmin2 : p.rmin1, rhi = top ? p.rmax2 : p.rmax1;
            bool ok = ahead(t) && sign_differs(z, dz) && rh2 >= rlo * rlo && rh2 <= rhi * rhi;
            if (!full(p)) ok = ok && wedge_member_at<WM>(p.w, ep, ed, t);
            best = (ok && t < best) ? t : best;
        }
        if (!full(p)) {
            {
                double t = -ep.c0 * rcp(ed.c0);
                double uh = fma(t, ed.u0, ep.u0), zh = fma(t, dz, z);
                bool ok = ed.c0 > 0.0 && ahead(t) && fabs(zh) <= p.dz &&
                          uh >= fma(p.in.B, zh, p.in.A) && uh <= fma(p.out.B, zh, p.out.A);
                best = (ok && t < best) ? t : best;
            }
            {
                double t = -ep.c1 * rcp(ed.c1);
                double uh = fma(t, ed.u1, ep.u1), zh = fma(t, dz, z);
                bool ok = ed.c1 > 0.0 && ahead(t) && fabs(zh) <= p.dz &&
                          uh >= fma(p.in.B, zh, p.in.A) && uh <= fma(p.out.B, zh, p.out.A);
                best = (ok && t < best) ? t : best;
            }
        }
        return in ? -1.0 : dmax(best, 0.0);
    }

    VG_DEV static double dist_out(const P &p, double x, double y, double z, double dx, double dy, double dz)
    {
        bool in, out;
        RayRZ r;
        r.rho2 = fma(x, x, y * y);
        WedgeEval ep = {}, ed = {};
        if (!full(p)) ep = wedge_eval(p.w, x, y), ed = wedge_eval(p.w, dx, dy);
        classify_pt(p, x, y, z, r.rho2, ep, in, out);
        r.a_xy = fma(dx, dx, dy * dy);
        r.b_xy = fma(x, dx, y * dy);
        double best = inf();
        {
            bool ok;
            double t = frustum_root(p.out, r, z, dz, true, ok);
            best = ok ? t : best;
        }
        if (hollow(p)) {
            bool ok;
            double t = frustum_root(p.in, r, z, dz, false, ok);
            // the mirror nappe (k < 0) lies beyond a cap, but guard the apex-at-the-cap case
            ok = ok && fma(p.in.B, fma(t, dz, z), p.in.A) >= 0.0;
            best = (ok && t < best) ? t : best;
        }
        {
            double t = (p.dz - flipsign_bits(z, dz)) * rcp(fabs(dz));
            best = (ahead(t) && t < best) ? t : best;
        }
        if (!full(p)) {
            {
                double t = -ep.c0 * rcp(ed.c0);
                bool ok = ed.c0 < 0.0 && ahead(t) && fma(t, ed.u0, ep.u0) >= 0.0;
                best = (ok && t < best) ? t : best;
            }
            {
                double t = -ep.c1 * rcp(ed.c1);
                bool ok = ed.c1 < 0.0 && ahead(t) && fma(t, ed.u1, ep.u1) >= 0.0;
                best = (ok && t < best) ? t : best;
            }
        }
        return out ? -1.0 : dmax(best, 0.0);
    }
};
using Cone = ConeT<kFlagsRuntime>;

// ------------------------------------------------------------------------------------------------------ trd

struct Trd {
    using P = TrdP;

    // max over the six planes of the signed plane distance (exact sdf inside a convex body)
    VG_DEV static double gmax(const P &p, double ax, double ay, double z, double &gx, double &gy)
    {
        gx = (fma(-p.fx, z, ax) - p.mx) * p.icx;
        gy = (fma(-p.fy, z, ay) - p.my) * p.icy;
        return dmax(dmax(gx, gy), fabs(z) - p.dz);
    }
    VG_DEV static int inside(const P &p, double x, double y, double z)
    {
        double gx, gy;
        double g = gmax(p, fabs(x), fabs(y), z, gx, gy);
        return classify(g < -kTol, g > kTol);
    }
    // squared in-plane distance from (v, s), v >= 0, to the filled symmetric trapezoid with half-widths r1 at
    // s = -he and r2 at s = +he; 0 inside.  (kx, ky) = the slanted side's edge vector (r2 - r1, 2 he), (kxs, kys) = the
    // same divided by its squared length: the foot parameter is one FMA + one MUL, the offsets reuse (r2 - v), (he - s).
    VG_DEV static double trapezoid_d2(double v, double s, double r1, double r2, double he, double kx, double ky, double kxs,
                                      double kys)
    {
        double rc = s < 0.0 ? r1 : r2;
        double qa = v - rc, sa = qa + fabs(qa), cay = fabs(s) - he; // max(v - rc, 0)^2 = (qa + |qa|)^2 / 4
        double wv = r2 - v, ws = he - s;
        double h = fma(wv, kxs, ws * kys);
        h = dmin(dmax(h, 0.0), 1.0);
        double cbx = fma(kx, h, -wv), cby = fma(ky, h, -ws);
        double d2 = dmin(fma(0.25 * sa, sa, cay * cay), fma(cbx, cbx, cby * cby));
        return (cbx < 0.0 && cay < 0.0) ? 0.0 : d2;
    }
    VG_DEV static double safety(const P &p, double x, double y, double z)
    {
        double ax = fabs(x), ay = fabs(y), gx, gy;
        double g = gmax(p, ax, ay, z, gx, gy);
        // the z face on the point's side of the mid-plane (a rectangle).  The other one cannot hold the nearest point in its
        // interior (that needs the point beyond it), and its edges belong to the slanted faces below as well.
        const bool top = not_neg(z);
        double zx = dmax(ax - (top ? p.dx2 : p.dx1), 0.0), zy = dmax(ay - (top ? p.dy2 : p.dy1), 0.0), zz = fabs(z) - p.dz;
        double D2 = fma(zx, zx, fma(zy, zy, zz * zz));
        // +x face: foot of the perpendicular, in-plane coordinates (|y|, slant coordinate)
        {
            double zf = fma(gx, p.sfx, z);
            D2 = dmin(D2, fma(gx, gx, trapezoid_d2(ay, zf * p.cx, p.dy1, p.dy2, p.hex, p.kxx, p.kyx, p.kxx_s, p.kyx_s)));
        }
        {
            double zf = fma(gy, p.sfy, z);
            D2 = dmin(D2, fma(gy, gy, trapezoid_d2(ax, zf * p.cy, p.dx1, p.dx2, p.hey, p.kxy, p.kyy, p.kxy_s, p.kyy_s)));
        }
        return g > 0.0 ? sqrt_nn(D2) : g;
    }
    // c.4 generic convex clip over the six half-spaces (normals need not be unit: num/den is scale free)
    VG_DEV static void clip(double num, double den, double &tin, double &tout)
    {
        double dn = nonzero(den); // den = +-0 -> +-1e-300: t = -+huge decides hit / miss like the oracle's branch
        double t = num * rcp(dn);
        tout = (dn > 0.0 && t < tout) ? t : tout;
        tin = (dn < 0.0 && t > tin) ? t : tin;
    }
    VG_DEV static void clip_all(const P &p, double x, double y, double z, double dx, double dy, double dz, double &tin,
                                double &tout)
    {
        tin = -inf();
        tout = inf();
        double sx = fma(p.fx, z, p.mx), sdx = p.fx * dz; // X(z) and its rate along the ray
        double sy = fma(p.fy, z, p.my), sdy = p.fy * dz;
        clip(sx - x, dx - sdx, tin, tout);
        clip(sx + x, -dx - sdx, tin, tout);
        clip(sy - y, dy - sdy, tin, tout);
        clip(sy + y, -dy - sdy, tin, tout);
        clip(p.dz - z, dz, tin, tout);
        clip(p.dz + z, -dz, tin, tout);
    }
    VG_DEV static double dist_in(const P &p, double x, double y, double z, double dx, double dy, double dz)
    {
        double gx, gy, tin, tout;
        double g = gmax(p, fabs(x), fabs(y), z, gx, gy);
        clip_all(p, x, y, z, dx, dy, dz, tin, tout);
        double t = (tin < tout && ahead(tin)) ? dmax(tin, 0.0) : inf();
        return g < -kTol ? -1.0 : t;
    }
    VG_DEV static double dist_out(const P &p, double x, double y, double z, double dx, double dy, double dz)
    {
        double gx, gy, tin, tout;
        double g = gmax(p, fabs(x), fabs(y), z, gx, gy);
        clip_all(p, x, y, z, dx, dy, dz, tin, tout);
        return g > kTol ? -1.0 : dmax(tout, 0.0);
    }
};

// ------------------------------------------------------------------------------------------------- polycone

template <int F> struct PolyconeT {
    using P = PolyconeP;
    static constexpr int WM = F < 0 ? kWmRuntime : (F >> 1);
    VG_DEV static bool full(const P &p) { return w_full<WM>(p.w); }

    VG_DEV static bool has_inner(const P &p, int k) { return (p.inner_mask >> k) & 1u; }

    // membership of (u, v) in the (r, z) outline (closed), by section
    VG_DEV static bool in_outline(const P &p, double u, double v)
    {
        bool mem = false;
#pragma unroll 1
        for (int k = 0; k < p.nsec; ++k) {
            const PconSec &s = p.sec[k];
            double ro = fma(s.out.B, v, s.out.A), ri = fma(s.in.B, v, s.in.A);
            mem = mem || (v >= s.z0 && v <= s.z1 && u <= ro && u >= ri);
        }
        return mem;
    }
    VG_DEV static void classify_pt(const P &p, double x, double y, double z, bool &in, bool &out)
    {
        double rho2 = fma(x, x, y * y);
        double rho = sqrt_nn(rho2);
        bool any_in = false, any_near = false;
#pragma unroll 1
        for (int k = 0; k < p.nsec; ++k) {
            const PconSec &s = p.sec[k];
            double ro = fma(s.out.B, z, s.out.A), ri = fma(s.in.B, z, s.in.A);
            double to = kTol * s.out.sec, ti = kTol * s.in.sec;
            bool zin = z >= s.z0 && z <= s.z1;
            bool znear = z >= s.z0 - kTol && z <= s.z1 + kTol;
            bool inner = has_inner(p, k);
            any_in = any_in || (zin && rho < ro - to && (!inner || rho > ri + ti));
            any_near = any_near || (znear && rho <= ro + to && (!inner || rho >= ri - ti));
        }
        in = any_in && z > p.zlo + kTol && z < p.zhi - kTol;
        out = !any_near;
        // z steps (R26): within kTol of an annular step face the point is on the surface, whatever the sections say
#pragma unroll 1
        for (int k = 0; k + 1 < p.nsec; ++k) {
            if (!((p.step_mask >> k) & 1u)) continue;
            const PconStep &t = p.step[k];
            bool near_face = (rho >= t.olo - kTol && rho <= t.ohi + kTol) || (rho >= t.ilo - kTol && rho <= t.ihi + kTol);
            in = in && !(fabs(z - t.z) <= kTol && near_face);
        }
        if (!full(p)) wedge_classify<WM>(p.w, wedge_eval(p.w, x, y), rho2, in, out);
    }
    VG_DEV static int inside(const P &p, double x, double y, double z)
    {
        bool in, out;
        classify_pt(p, x, y, z, in, out);
        return classify(in, out);
    }
    VG_DEV static double outline_d2(const P &p, double u, double v, bool axis)
    {
        double b1 = dmax(dmax(p.cap_lo_rmin - u, u - p.cap_lo_rmax), 0.0), v1 = v - p.zlo;
        double b2 = dmax(dmax(p.cap_hi_rmin - u, u - p.cap_hi_rmax), 0.0), v2 = v - p.zhi;
        double d2 = dmin(fma(b1, b1, v1 * v1), fma(b2, b2, v2 * v2));
#pragma unroll 1
        for (int k = 0; k < p.nsec; ++k) {
            const PconSec &s = p.sec[k];
            double ez = s.z1 - s.z0;
            d2 = dmin(d2, seg_d2(u, v, s.out.r0, s.z0, s.out.er, ez, s.out.inv_l2));
            double di = seg_d2(u, v, s.in.r0, s.z0, s.in.er, ez, s.in.inv_l2);
            d2 = (has_inner(p, k) || axis) ? dmin(d2, di) : d2;
            if ((p.step_mask >> k) & 1u) { // the horizontal edges of the z step above this section (empty ranges: lo > hi)
                const PconStep &t = p.step[k];
                double vz = v - t.z, vz2 = vz * vz;
                double bo = dmax(dmax(t.olo - u, u - t.ohi), 0.0), bi = dmax(dmax(t.ilo - u, u - t.ihi), 0.0);
                d2 = t.ohi > t.olo ? dmin(d2, fma(bo, bo, vz2)) : d2;
                d2 = t.ihi > t.ilo ? dmin(d2, fma(bi, bi, vz2)) : d2;
            }
        }
        return d2;
    }
    VG_DEV static double safety(const P &p, double x, double y, double z)
    {
        double rho2 = fma(x, x, y * y);
        double rho = sqrt_nn(rho2);
        bool in2d = in_outline(p, rho, z);
        double D2 = outline_d2(p, rho, z, false);
        if (full(p)) {
            double D = sqrt_nn(D2);
            return in2d ? -D : D;
        }
        WedgeEval e = wedge_eval(p.w, x, y);
        bool mem = wedge_member<WM>(p.w, e.c0, e.c1);
        D2 = mem ? D2 : inf();
        double f0 = in_outline(p, e.u0, z) ? 0.0 : outline_d2(p, e.u0, z, true);
        double f1 = in_outline(p, e.u1, z) ? 0.0 : outline_d2(p, e.u1, z, true);
        D2 = dmin(D2, fma(e.c0, e.c0, f0));
        D2 = dmin(D2, fma(e.c1, e.c1, f1));
        double D = sqrt_nn(D2);
        return (mem && in2d) ? -D : D;
    }

    // first crossing in the entering (leaving = false) or leaving (leaving = true) sense over all patches
    VG_DEV static double cross(const P &p, double x, double y, double z, double dx, double dy, double dz, bool leaving)
    {
        RayRZ r;
        r.rho2 = fma(x, x, y * y);
        r.a_xy = fma(dx, dx, dy * dy);
        r.b_xy = fma(x, dx, y * dy);
        WedgeEval ep = {}, ed = {};
        if (!full(p)) ep = wedge_eval(p.w, x, y), ed = wedge_eval(p.w, dx, dy);
        double best = inf();
#pragma unroll 1
        for (int k = 0; k < p.nsec; ++k) {
            const PconSec &s = p.sec[k];
            {
                bool ok;
                double t = frustum_root(s.out, r, z, dz, leaving, ok);
                double zh = fma(t, dz, z);
                ok = ok && zh >= s.z0 && zh <= s.z1;
                if (!full(p)) ok = ok && wedge_member_at<WM>(p.w, ep, ed, t);
                best = (ok && t < best) ? t : best;
            }
            if (has_inner(p, k)) {
                bool ok;
                double t = frustum_root(s.in, r, z, dz, !leaving, ok);
                double zh = fma(t, dz, z);
                ok = ok && zh >= s.z0 && zh <= s.z1;
                if (!full(p)) ok = ok && wedge_member_at<WM>(p.w, ep, ed, t);
                best = (ok && t < best) ? t : best;
            }
        }
        double idz = rcp(dz); // NaN for dz = 0: caps and step faces rejected
        // z steps (R26): annular faces at internal planes; a face whose material lies below (normal +z) is entered going
        // down and left going up, and the other way round
#pragma unroll 1
        for (int k = 0; k + 1 < p.nsec; ++k) {
            if (!((p.step_mask >> k) & 1u)) continue;
            const PconStep &st = p.step[k];
            double t = (st.z - z) * idz;
            double rh2 = fma(t, fma(t, r.a_xy, r.b_xy + r.b_xy), r.rho2);
            bool up = dz > 0.0;
            bool on_o = rh2 >= st.olo * st.olo && rh2 <= st.ohi * st.ohi && st.ohi > st.olo && (leaving ? (st.oup != 0) == up : (st.oup != 0) != up);
            bool on_i = rh2 >= st.ilo * st.ilo && rh2 <= st.ihi * st.ihi && st.ihi > st.ilo && (leaving ? (st.iup != 0) == up : (st.iup != 0) != up);
            bool ok = ahead(t) && (on_o || on_i);
            if (!full(p)) ok = ok && wedge_member_at<WM>(p.w, ep, ed, t);
            best = (ok && t < best) ? t : best;
        }
        // end caps: entering from beyond, leaving from within
        {
            double t = (p.zlo - z) * idz;
            double hx = fma(t, dx, x), hy = fma(t, dy, y), rh2 = fma(hx, hx, hy * hy);
            bool sense = leaving ? dz < 0.0 : dz > 0.0;
            bool ok = sense && ahead(t) && rh2 >= p.cap_lo_rmin * p.cap_lo_rmin && rh2 <= p.cap_lo_rmax * p.cap_lo_rmax;
            if (!full(p)) ok = ok && wedge_member_at<WM>(p.w, ep, ed, t);
            best = (ok && t < best) ? t : best;
        }
        {
            double t = (p.zhi - z) * idz;
            double hx = fma(t, dx, x), hy = fma(t, dy, y), rh2 = fma(hx, hx, hy * hy);
            bool sense = leaving ? dz > 0.0 : dz < 0.0;
            bool ok = sense && ahead(t) && rh2 >= p.cap_hi_rmin * p.cap_hi_rmin && rh2 <= p.cap_hi_rmax * p.cap_hi_rmax;
            if (!full(p)) ok = ok && wedge_member_at<WM>(p.w, ep, ed, t);
            best = (ok && t < best) ? t : best;
        }
        if (!full(p)) {
            {
                double t = -ep.c0 * rcp(ed.c0);
                bool sense = leaving ? ed.c0 < 0.0 : ed.c0 > 0.0;
                bool ok = sense && ahead(t) && in_outline(p, fma(t, ed.u0, ep.u0), fma(t, dz, z));
                best = (ok && t < best) ? t : best;
            }
            {
                double t = -ep.c1 * rcp(ed.c1);
                bool sense = leaving ? ed.c1 < 0.0 : ed.c1 > 0.0;
                bool ok = sense && ahead(t) && in_outline(p, fma(t, ed.u1, ep.u1), fma(t, dz, z));
                best = (ok && t < best) ? t : best;
            }
        }
        return dmax(best, 0.0);
    }
    VG_DEV static double dist_in(const P &p, double x, double y, double z, double dx, double dy, double dz)
    {
        bool in, out;
        classify_pt(p, x, y, z, in, out);
        double t = cross(p, x, y, z, dx, dy, dz, false);
        return in ? -1.0 : t;
    }
    VG_DEV static double dist_out(const P &p, double x, double y, double z, double dx, double dy, double dz)
    {
        bool in, out;
        classify_pt(p, x, y, z, in, out);
        double t = cross(p, x, y, z, dx, dy, dz, true);
        return out ? -1.0 : t;
    }
};
using Polycone = PolyconeT<kFlagsRuntime>;

} // namespace vg
