// vg_pcon_walk.cuh -- ordered-walk kernels of the full-phi polycone (configs[3]: DistanceToIn, SafetyToIn/Out).
//
// The generic polycone code (vg_shapes.cuh) evaluates all 2 (nz - 1) conical patches for every track.  These
// kernels give the same results (min over the same candidates) but visit only the sections that can hold it:
//   DistanceToIn -- z(t) is monotonic along a ray and the sections are disjoint slabs in z, so the ray meets them in
//                   z order; every crossing found in a section is earlier than every crossing of a later section.
//                   The ray is first clipped against the bounding cylinder (largest rmax, [zlo, zhi]): a ray that
//                   misses it is a miss; otherwise the walk starts in the section where the clipped ray starts and
//                   stops at the first section that yields a valid crossing or where the clipped ray ends.
//   Safety       -- the squared distance to a segment of section k is at least the squared z gap between the point
//                   and the slab [z0_k, z1_k]; the walk goes outwards from the point's own section, up and down,
//                   until the gap alone exceeds the best distance so far.
// The walks are per-lane loops with lane-dependent section indices, so the section constants are staged in shared
// memory (one compact record per section) instead of the constant bank, whose reads serialise on divergent indices.
#pragma once
#include "vg_kernels.cuh"

namespace vg {

constexpr int kWalkBlock = 256;

VG_DEV void pcon_stage(const PolyconeP &p, PconWalkSec *tab)
{
    for (int k = threadIdx.x; k < p.nsec; k += blockDim.x) {
        const PconSec &s = p.sec[k];
        PconWalkSec w;
        w.z0 = s.z0, w.z1 = s.z1;
        w.Ao = s.out.A, w.Bo = s.out.B, w.Ai = s.in.A, w.Bi = s.in.B;
        w.ro0 = s.out.r0, w.ero = s.out.er, w.ilo = s.out.inv_l2;
        w.ri0 = s.in.r0, w.eri = s.in.er, w.ili = s.in.inv_l2;
        w.seco = s.out.sec, w.seci = s.in.sec;
        tab[k] = w;
    }
}

// index of the section whose slab holds z: number of internal planes <= z (warp-uniform loop, constant-bank reads)
VG_DEV int pcon_section_of(const PolyconeP &p, double z)
{
    int k = 0;
#pragma unroll 1
    for (int j = 1; j < p.nsec; ++j) k += (p.sec[j].z0 <= z) ? 1 : 0;
    return k;
}

// three section indices in one warp-uniform pass over the internal planes
VG_DEV void pcon_sections_of(const PolyconeP &p, double za, double zb, double zc, int &ka, int &kb, int &kc)
{
    ka = kb = kc = 0;
#pragma unroll 1
    for (int j = 1; j < p.nsec; ++j) {
        const double zp = p.sec[j].z0;
        ka += (zp <= za) ? 1 : 0;
        kb += (zp <= zb) ? 1 : 0;
        kc += (zp <= zc) ? 1 : 0;
    }
}

// ---- z steps (reading R26).  Step k sits on the plane between section k and section k + 1; its constants are read from
// the constant bank with a lane-dependent index, but only by the lanes whose walk reaches a step (step_mask is uniform).

// is (rho^2, z) within kTol of an annular face of step k?  (such a point is on the surface, not inside)
VG_DEV bool pcon_near_step(const PolyconeP &p, int k, double rho2, double z)
{
    if (k < 0 || k + 1 >= p.nsec || !((p.step_mask >> k) & 1u)) return false;
    const PconStep &t = p.step[k];
    const double rho = sqrt_nn(rho2);
    return fabs(z - t.z) <= kTol && ((rho >= t.olo - kTol && rho <= t.ohi + kTol) || (rho >= t.ilo - kTol && rho <= t.ihi + kTol));
}

// entering crossing of the faces of step k by the ray, +inf if none; same tests as PolyconeT::cross(leaving = false)
VG_DEV double pcon_step_enter(const PolyconeP &p, int k, const RayRZ &r, double z, double dz, double idz)
{
    if (k < 0 || k + 1 >= p.nsec || !((p.step_mask >> k) & 1u)) return inf();
    const PconStep &st = p.step[k];
    const double t = (st.z - z) * idz;
    const double rh2 = fma(t, fma(t, r.a_xy, r.b_xy + r.b_xy), r.rho2);
    const bool up = dz > 0.0;
    const bool on_o = rh2 >= st.olo * st.olo && rh2 <= st.ohi * st.ohi && st.ohi > st.olo && (st.oup != 0) != up;
    const bool on_i = rh2 >= st.ilo * st.ilo && rh2 <= st.ihi * st.ihi && st.ihi > st.ilo && (st.iup != 0) != up;
    return (ahead(t) && (on_o || on_i)) ? t : inf();
}

// squared distance from (u, v) to the horizontal edges of step k (the running minimum d2 goes in and comes out)
VG_DEV double pcon_step_d2(const PolyconeP &p, int k, double u, double v, double d2)
{
    if (k < 0 || k + 1 >= p.nsec || !((p.step_mask >> k) & 1u)) return d2;
    const PconStep &t = p.step[k];
    const double vz = v - t.z, vz2 = vz * vz;
    const double bo = dmax(dmax(t.olo - u, u - t.ohi), 0.0), bi = dmax(dmax(t.ilo - u, u - t.ihi), 0.0);
    d2 = t.ohi > t.olo ? dmin(d2, fma(bo, bo, vz2)) : d2;
    d2 = t.ihi > t.ilo ? dmin(d2, fma(bi, bi, vz2)) : d2;
    return d2;
}

// (u, v) in the closed (r, z) outline?  Same set as PolyconeT::in_outline (the union of the closed sections), from the
// section that holds v and, on a shared plane, the one below it
VG_DEV bool pcon_in_outline(const PolyconeP &p, const PconWalkSec *tab, double u, double v)
{
    const int k = pcon_section_of(p, v);
    const PconWalkSec &w = tab[k];
    bool in = v >= w.z0 && v <= w.z1 && u <= fma(w.Bo, v, w.Ao) && u >= fma(w.Bi, v, w.Ai);
    if (k > 0 && v <= tab[k - 1].z1) {
        const PconWalkSec &b = tab[k - 1];
        in = in || (v >= b.z0 && u <= fma(b.Bo, v, b.Ao) && u >= fma(b.Bi, v, b.Ai));
    }
    return in;
}

// DistanceToIn of the polycone; same candidates and validity tests as PolyconeT::dist_in.  WEDGE: the polycone has a phi
// cut: every crossing must also lie in the segment (linear test along the ray), the two phi faces are two more candidates
// (entering sense, hit point inside the (r, z) outline) taken after the walk, and Inside includes the wedge.
template <bool WEDGE>
VG_DEV double pcon_walk_dist_in(const PolyconeP &p, const PconWalkSec *tab, double x, double y, double z, double dx,
                                double dy, double dz)
{
    RayRZ r;
    WedgeEval ep = {}, ed = {};
    if (WEDGE) ep = wedge_eval(p.w, x, y), ed = wedge_eval(p.w, dx, dy);
    r.rho2 = fma(x, x, y * y);
    r.a_xy = fma(dx, dx, dy * dy);
    r.b_xy = fma(x, dx, y * dy);
    const double a = r.a_xy, b = r.b_xy;

    // clip the ray against the bounding cylinder rho^2 <= rb2, zlo - slack <= z <= zhi + slack
    const double kSlack = 1e-7;
    const double c = r.rho2 - p.rb2;
    const double D = fma(b, b, -a * c);
    const double s = sqrt_pos(D);
    const double inv_a = rcp(a);
    const bool vertical = !(a >= kTiny); // ray parallel to the axis
    const double tr0 = vertical ? -inf() : (-b - s) * inv_a;
    const double tr1 = vertical ? inf() : (s - b) * inv_a;
    const bool rad_ok = vertical ? c <= 0.0 : D > 0.0;
    const bool horizontal = !(fabs(dz) >= kTiny);
    const double idz = rcp(dz);
    const double ta = (p.zlo - z) * idz, tb = (p.zhi - z) * idz; // times of the two end planes
    const double sl = kSlack * fabs(idz);
    const bool up = not_neg(dz);
    const double tz0 = horizontal ? -inf() : (up ? ta : tb) - sl;
    const double tz1 = horizontal ? inf() : (up ? tb : ta) + sl;
    const bool z_ok = horizontal ? (z >= p.zlo && z <= p.zhi) : true;
    const double t0 = dmax(dmax(tr0, tz0), 0.0), t1 = dmin(tr1, tz1);
    const double zs = fma(t0, dz, z), ze = fma(t1, dz, z);

    int kz, k, kend;
    pcon_sections_of(p, z, (up ? zs : ze) - kSlack, (up ? ze : zs) + kSlack, kz, k, kend);

    // Inside (R6: strictly inside by kTol) on the point's own section
    bool in;
    {
        const PconWalkSec &w = tab[kz];
        const double ro = fma(w.Bo, z, w.Ao) - kTol * w.seco;
        const double ri = fma(w.Bi, z, w.Ai) + kTol * w.seci;
        const bool inner = (p.inner_mask >> kz) & 1u;
        in = z > p.zlo + kTol && z < p.zhi - kTol && ro > 0.0 && r.rho2 < ro * ro && (!inner || ri < 0.0 || r.rho2 > ri * ri);
        if (p.step_mask) in = in && !pcon_near_step(p, kz, r.rho2, z) && !pcon_near_step(p, kz - 1, r.rho2, z);
        if (WEDGE) {
            bool out_unused = false;
            wedge_classify<kWmRuntime>(p.w, ep, r.rho2, in, out_unused);
        }
    }

    // a ray that starts beyond an end plane meets that cap before anything else
    const double tc = up ? ta : tb;
    const double rc2 = fma(tc, fma(tc, a, b + b), r.rho2);
    const double clo = up ? p.cap_lo_rmin : p.cap_hi_rmin, chi = up ? p.cap_lo_rmax : p.cap_hi_rmax;
    const bool beyond = ahead(tc); // beyond the end plane, or on it (R32); NaN for a horizontal ray
    bool cap_hit = beyond && !horizontal && rc2 >= clo * clo && rc2 <= chi * chi;
    if (WEDGE) cap_hit = cap_hit && wedge_member_at<kWmRuntime>(p.w, ep, ed, tc);

    double best = cap_hit ? tc : inf();
    bool go = rad_ok && z_ok && t0 <= t1 && !in && !cap_hit;
    if (!up) {
        const int tmp = k;
        k = kend;
        kend = tmp;
    }
    const int step = up ? 1 : -1;
    while (go) {
        const PconWalkSec w = tab[k];
        Frustum f;
        bool ok;
        f.A = w.Ao, f.B = w.Bo;
        double t = frustum_root(f, r, z, dz, false, ok); // outer patch, entering root
        double zh = fma(t, dz, z);
        ok = ok && zh >= w.z0 && zh <= w.z1;
        if (WEDGE) ok = ok && wedge_member_at<kWmRuntime>(p.w, ep, ed, t);
        best = (ok && t < best) ? t : best;
        f.A = w.Ai, f.B = w.Bi;
        t = frustum_root(f, r, z, dz, true, ok); // inner patch: the ray enters where it leaves the bore
        zh = fma(t, dz, z);
        ok = ok && ((p.inner_mask >> k) & 1u) && zh >= w.z0 && zh <= w.z1;
        if (WEDGE) ok = ok && wedge_member_at<kWmRuntime>(p.w, ep, ed, t);
        best = (ok && t < best) ? t : best;
        go = !(best < inf()) && k != kend;
        if (go && p.step_mask) { // the step face on the plane the ray crosses next comes before anything of the next section
            const double ts = pcon_step_enter(p, up ? k : k - 1, r, z, dz, idz);
            const bool ok_s = ts < inf() && (!WEDGE || wedge_member_at<kWmRuntime>(p.w, ep, ed, ts));
            best = ok_s ? ts : best;
            go = !ok_s;
        }
        k += step;
    }
    if (WEDGE) { // the two phi faces, entering sense; the hit point must lie in the (r, z) outline (R1: closed)
        {
            const double t = -ep.c0 * rcp(ed.c0);
            const bool ok = ed.c0 > 0.0 && ahead(t) && t < best &&
                            pcon_in_outline(p, tab, fma(t, ed.u0, ep.u0), fma(t, dz, z));
            best = ok ? t : best;
        }
        {
            const double t = -ep.c1 * rcp(ed.c1);
            const bool ok = ed.c1 > 0.0 && ahead(t) && t < best &&
                            pcon_in_outline(p, tab, fma(t, ed.u1, ep.u1), fma(t, dz, z));
            best = ok ? t : best;
        }
    }
    return in ? -1.0 : dmax(best, 0.0);
}

// exact signed distance of the full-phi polycone; same segments as PolyconeT::safety
VG_DEV double pcon_walk_sdf(const PolyconeP &p, const PconWalkSec *tab, double x, double y, double z)
{
    const double rho2 = fma(x, x, y * y);
    const double rho = sqrt_nn(rho2);
    const int kz = pcon_section_of(p, z);
    bool in2d;
    {
        const PconWalkSec &w = tab[kz];
        in2d = z >= p.zlo && z <= p.zhi && rho <= fma(w.Bo, z, w.Ao) && rho >= fma(w.Bi, z, w.Ai);
    }
    const double b1 = dmax(dmax(p.cap_lo_rmin - rho, rho - p.cap_lo_rmax), 0.0), v1 = z - p.zlo;
    const double b2 = dmax(dmax(p.cap_hi_rmin - rho, rho - p.cap_hi_rmax), 0.0), v2 = z - p.zhi;
    double d2 = dmin(fma(b1, b1, v1 * v1), fma(b2, b2, v2 * v2));
    for (int k = kz; k < p.nsec; ++k) { // upwards
        const PconWalkSec w = tab[k];
        const double gap = dmax(w.z0 - z, 0.0);
        if (gap * gap >= d2) break;
        const double ez = w.z1 - w.z0;
        d2 = dmin(d2, seg_d2(rho, z, w.ro0, w.z0, w.ero, ez, w.ilo));
        const double di = seg_d2(rho, z, w.ri0, w.z0, w.eri, ez, w.ili);
        d2 = ((p.inner_mask >> k) & 1u) ? dmin(d2, di) : d2;
        if (p.step_mask) d2 = pcon_step_d2(p, k, rho, z, d2); // the step on top of section k (never nearer than the section's slab)
    }
    for (int k = kz - 1; k >= 0; --k) { // downwards
        const PconWalkSec w = tab[k];
        const double gap = dmax(z - w.z1, 0.0);
        if (gap * gap >= d2) break;
        const double ez = w.z1 - w.z0;
        d2 = dmin(d2, seg_d2(rho, z, w.ro0, w.z0, w.ero, ez, w.ilo));
        const double di = seg_d2(rho, z, w.ri0, w.z0, w.eri, ez, w.ili);
        d2 = ((p.inner_mask >> k) & 1u) ? dmin(d2, di) : d2;
        if (p.step_mask) d2 = pcon_step_d2(p, k, rho, z, d2);
    }
    const double dist = sqrt_nn(d2);
    return in2d ? -dist : dist;
}

// ---- candidate-grid form of the same signed distance (vg_pcon_grid.h) ----
//
// One record per segment of the (r, z) outline, numbered like the mask bits of the grid: (r0, z0), the edge vector
// (er, ez) and the edge vector divided by |edge|^2, so that the foot parameter is t = w . e' (one FMA + one MUL).  Six
// doubles, 16-byte aligned: three 128-bit shared loads per candidate.

VG_DEV void pcon_stage_segs(const PolyconeP &p, double *seg)
{
    for (int s = threadIdx.x; s < 64; s += blockDim.x) pcon_seg_record(p, s, seg + kPconSegStride * s);
}

// squared distance from (u, v) to the segment of record q (same value as seg_d2 up to the rounding of e' = e / |e|^2)
VG_DEV double pcon_seg_d2(double u, double v, const double *q)
{
    const double2 a = *reinterpret_cast<const double2 *>(q), e = *reinterpret_cast<const double2 *>(q + 2),
                  f = *reinterpret_cast<const double2 *>(q + 4);
    const double wu = u - a.x, wv = v - a.y;
    double t = fma(wu, f.x, wv * f.y);
    t = dmin(dmax(t, 0.0), 1.0);
    const double du = fma(-t, e.x, wu), dv = fma(-t, e.y, wv);
    return fma(du, du, dv * dv);
}

// exact signed distance: minimum over the candidate segments of the point's cell (the cell's mask holds every segment
// that can be nearest to any point of the cell), sign from the point's own section.  Off the grid: the ordered walk.
VG_DEV double pcon_grid_sdf(const PolyconeP &p, const PconWalkSec *tab, const double *seg, const PconGrid &g, double x,
                            double y, double z)
{
    const double rho2 = fma(x, x, y * y);
    const double rho = sqrt_nn(rho2);
    const double fr = rho * g.g.inv_cr, fz = (z - g.g.zg0) * g.g.inv_cz;
    if (!(fr < double(kPconGridR) && fz >= 0.0 && fz < double(kPconGridZ))) return pcon_walk_sdf(p, tab, x, y, z);
    const int ir = int(fr), iz = int(fz);
    const uint2 m = __ldg(reinterpret_cast<const uint2 *>(g.masks) + iz * kPconGridR + ir);
    int kz = __ldg(g.rows + iz);
    while (kz + 1 < p.nsec && tab[kz + 1].z0 <= z) ++kz;
    bool in2d;
    {
        const PconWalkSec &w = tab[kz];
        in2d = z >= p.zlo && z <= p.zhi && rho <= fma(w.Bo, z, w.Ao) && rho >= fma(w.Bi, z, w.Ai);
    }
    double d2 = inf();
    unsigned w = m.x; // caps and sections 0..14
    while (w) {
        const int s = __ffs(int(w)) - 1;
        w &= w - 1;
        d2 = dmin(d2, pcon_seg_d2(rho, z, seg + kPconSegStride * s));
    }
    w = m.y; // sections 15..30
    while (w) {
        const int s = __ffs(int(w)) + 31;
        w &= w - 1;
        d2 = dmin(d2, pcon_seg_d2(rho, z, seg + kPconSegStride * s));
    }
    const double dist = sqrt_nn(d2);
    return in2d ? -dist : dist;
}

// minimum squared distance from (u, v) to the candidate segments of its cell; `col0` / `ncol`: the surface grid starts at
// u = 0 with kPconGridR columns, the face grid at u = -R with twice as many.  Off the grid: NaN.
VG_DEV double pcon_grid_d2(const unsigned long long *masks, int ncol, double u_shift, const double *seg, const PconGrid &g,
                           double u, double v)
{
    const double fr = (u + u_shift) * g.g.inv_cr, fz = (v - g.g.zg0) * g.g.inv_cz;
    if (!(fr >= 0.0 && fr < double(ncol) && fz >= 0.0 && fz < double(kPconGridZ))) return __longlong_as_double(0x7ff8000000000000LL);
    const uint2 m = __ldg(reinterpret_cast<const uint2 *>(masks) + int(fz) * ncol + int(fr));
    double d2 = inf();
    unsigned w = m.x;
    while (w) {
        const int s = __ffs(int(w)) - 1;
        w &= w - 1;
        d2 = dmin(d2, pcon_seg_d2(u, v, seg + kPconSegStride * s));
    }
    w = m.y;
    while (w) {
        const int s = __ffs(int(w)) + 31;
        w &= w - 1;
        d2 = dmin(d2, pcon_seg_d2(u, v, seg + kPconSegStride * s));
    }
    return d2;
}

// signed distance of a polycone WITH a phi cut from the two grids (c.3): the surface of revolution where the point is
// in the segment, and per phi face the in-plane distance to the filled outline (0 inside it, else the face grid: every
// edge incl. those on the axis) combined with the distance to the face's plane.  Any look-up off its grid: the generic
// code (all segments).
VG_DEV double pcon_grid_sdf_wedge(const PolyconeP &p, const PconWalkSec *tab, const double *seg, const PconGrid &g, double x,
                                  double y, double z)
{
    const double rho2 = fma(x, x, y * y);
    const double rho = sqrt_nn(rho2);
    const WedgeEval e = wedge_eval(p.w, x, y);
    const bool mem = wedge_member<kWmRuntime>(p.w, e.c0, e.c1);
    const double R = double(kPconGridR) / g.g.inv_cr;
    const double dB = pcon_grid_d2(g.masks, kPconGridR, 0.0, seg, g, rho, z);
    const bool in0 = pcon_in_outline(p, tab, e.u0, z), in1 = pcon_in_outline(p, tab, e.u1, z);
    const double f0 = in0 ? 0.0 : pcon_grid_d2(g.face_masks, 2 * kPconGridR, R, seg, g, e.u0, z);
    const double f1 = in1 ? 0.0 : pcon_grid_d2(g.face_masks, 2 * kPconGridR, R, seg, g, e.u1, z);
    if (!(dB == dB && f0 == f0 && f1 == f1)) return PolyconeT<kFlagsRuntime>::safety(p, x, y, z); // a NaN: off a grid
    const bool in2d = pcon_in_outline(p, tab, rho, z);
    double D2 = mem ? dB : inf();
    D2 = dmin(D2, fma(e.c0, e.c0, f0));
    D2 = dmin(D2, fma(e.c1, e.c1, f1));
    const double D = sqrt_nn(D2);
    return (mem && in2d) ? -D : D;
}

// Inside flags from the point's own section and its two neighbours (a tolerance band reaches at most the next section):
// the same tests as PolyconeT::classify_pt, which loops over every section
template <bool WEDGE>
VG_DEV void pcon_walk_classify(const PolyconeP &p, const PconWalkSec *tab, double x, double y, double z, bool &in, bool &out)
{
    const double rho2 = fma(x, x, y * y);
    const double rho = sqrt_nn(rho2);
    const int kz = pcon_section_of(p, z);
    bool any_in = false, any_near = false;
#pragma unroll
    for (int j = -1; j <= 1; ++j) {
        const int k = kz + j;
        if (k < 0 || k >= p.nsec) continue;
        const PconWalkSec &w = tab[k];
        const double ro = fma(w.Bo, z, w.Ao), ri = fma(w.Bi, z, w.Ai);
        const double to = kTol * w.seco, ti = kTol * w.seci;
        const bool zin = z >= w.z0 && z <= w.z1;
        const bool znear = z >= w.z0 - kTol && z <= w.z1 + kTol;
        const bool inner = (p.inner_mask >> k) & 1u;
        any_in = any_in || (zin && rho < ro - to && (!inner || rho > ri + ti));
        any_near = any_near || (znear && rho <= ro + to && (!inner || rho >= ri - ti));
    }
    in = any_in && z > p.zlo + kTol && z < p.zhi - kTol;
    out = !any_near;
    if (p.step_mask) in = in && !pcon_near_step(p, kz, rho2, z) && !pcon_near_step(p, kz - 1, rho2, z);
    if (WEDGE) wedge_classify<kWmRuntime>(p.w, wedge_eval(p.w, x, y), rho2, in, out);
}

// leaving crossing of the faces of step k, +inf if none (PolyconeT::cross with leaving = true)
VG_DEV double pcon_step_leave(const PolyconeP &p, int k, const RayRZ &r, double z, double dz, double idz)
{
    if (k < 0 || k + 1 >= p.nsec || !((p.step_mask >> k) & 1u)) return inf();
    const PconStep &st = p.step[k];
    const double t = (st.z - z) * idz;
    const double rh2 = fma(t, fma(t, r.a_xy, r.b_xy + r.b_xy), r.rho2);
    const bool up = dz > 0.0;
    const bool on_o = rh2 >= st.olo * st.olo && rh2 <= st.ohi * st.ohi && st.ohi > st.olo && (st.oup != 0) == up;
    const bool on_i = rh2 >= st.ilo * st.ilo && rh2 <= st.ihi * st.ihi && st.ihi > st.ilo && (st.iup != 0) == up;
    return (ahead(t) && (on_o || on_i)) ? t : inf();
}

// DistanceToOut: from the point's own section the ray stays in the material until it leaves through a patch of the
// section it is in (outer: leaving root, inner: entering root), through a step face on the plane it crosses next, or
// through an end cap; sections are visited in the order the ray meets them.  Same candidates and tests as
// PolyconeT::dist_out, which evaluates every section.
template <bool WEDGE>
VG_DEV double pcon_walk_dist_out(const PolyconeP &p, const PconWalkSec *tab, double x, double y, double z, double dx,
                                 double dy, double dz)
{
    bool in, out;
    pcon_walk_classify<WEDGE>(p, tab, x, y, z, in, out);
    RayRZ r;
    r.rho2 = fma(x, x, y * y);
    r.a_xy = fma(dx, dx, dy * dy);
    r.b_xy = fma(x, dx, y * dy);
    WedgeEval ep = {}, ed = {};
    if (WEDGE) ep = wedge_eval(p.w, x, y), ed = wedge_eval(p.w, dx, dy);
    const double idz = rcp(dz); // NaN for dz = 0: a horizontal ray never reaches a plane and ends in its own section
    const bool up = not_neg(dz);
    const int step = up ? 1 : -1;
    int k = pcon_section_of(p, z);
    double best = inf();
    bool go = !out;
    if (go && p.step_mask) { // a start ON a step face (R32): the plane just behind the point's section, leaving sense, t ~ 0
        const double tb = pcon_step_leave(p, up ? k - 1 : k, r, z, dz, idz);
        const bool okb = tb < inf() && (!WEDGE || wedge_member_at<kWmRuntime>(p.w, ep, ed, tb));
        best = okb ? tb : best;
        go = !okb;
    }
    while (go) {
        const PconWalkSec w = tab[k];
        Frustum f;
        bool ok;
        f.A = w.Ao, f.B = w.Bo;
        double t = frustum_root(f, r, z, dz, true, ok);
        double zh = fma(t, dz, z);
        ok = ok && zh >= w.z0 && zh <= w.z1;
        if (WEDGE) ok = ok && wedge_member_at<kWmRuntime>(p.w, ep, ed, t);
        best = (ok && t < best) ? t : best;
        f.A = w.Ai, f.B = w.Bi;
        t = frustum_root(f, r, z, dz, false, ok);
        zh = fma(t, dz, z);
        ok = ok && ((p.inner_mask >> k) & 1u) && zh >= w.z0 && zh <= w.z1;
        if (WEDGE) ok = ok && wedge_member_at<kWmRuntime>(p.w, ep, ed, t);
        best = (ok && t < best) ? t : best;
        if (best < inf() || !(fabs(dz) >= kTiny)) break;
        const int kn = k + step;
        if (kn < 0 || kn >= p.nsec) { // the end cap
            const double tc = ((up ? p.zhi : p.zlo) - z) * idz;
            const bool okc = ahead(tc) && (!WEDGE || wedge_member_at<kWmRuntime>(p.w, ep, ed, tc));
            best = okc ? tc : best;
            break;
        }
        if (p.step_mask) {
            const double ts = pcon_step_leave(p, up ? k : kn, r, z, dz, idz);
            const bool oks = ts < inf() && (!WEDGE || wedge_member_at<kWmRuntime>(p.w, ep, ed, ts));
            best = oks ? ts : best;
            if (oks) break;
        }
        k = kn;
    }
    if (WEDGE && !out) { // the phi faces in the leaving sense
        {
            const double t = -ep.c0 * rcp(ed.c0);
            const bool ok = ed.c0 < 0.0 && ahead(t) && t < best && pcon_in_outline(p, tab, fma(t, ed.u0, ep.u0), fma(t, dz, z));
            best = ok ? t : best;
        }
        {
            const double t = -ep.c1 * rcp(ed.c1);
            const bool ok = ed.c1 < 0.0 && ahead(t) && t < best && pcon_in_outline(p, tab, fma(t, ed.u1, ep.u1), fma(t, dz, z));
            best = ok ? t : best;
        }
    }
    return out ? -1.0 : dmax(best, 0.0);
}

template <int Q, bool GRID, bool WEDGE>
VG_DEV double pcon_walk_eval(const PolyconeP &p, const PconWalkSec *tab, const double *seg, const PconGrid &g, double x,
                             double y, double z, double dx, double dy, double dz, double step_max)
{
    if (Q == qSafeIn || Q == qSafeOut) {
        const double s = WEDGE ? pcon_grid_sdf_wedge(p, tab, seg, g, x, y, z)
                               : (GRID ? pcon_grid_sdf(p, tab, seg, g, x, y, z) : pcon_walk_sdf(p, tab, x, y, z));
        return Q == qSafeIn ? s : -s;
    }
    const double t = Q == qDistOut ? pcon_walk_dist_out<WEDGE>(p, tab, x, y, z, dx, dy, dz)
                                   : pcon_walk_dist_in<WEDGE>(p, tab, x, y, z, dx, dy, dz);
    return t <= step_max ? t : inf();
}

#ifndef VG_WALK_MINB
#define VG_WALK_MINB 3
#endif

// persistent CTAs striding over tiles of 512 tracks, two tracks per thread (128-bit loads; arrays 16-byte aligned)
template <int Q, bool GRID, bool WEDGE>
__global__ void __launch_bounds__(kWalkBlock, VG_WALK_MINB)
    pcon_walk_kernel(const __grid_constant__ PolyconeP p, const __grid_constant__ PconGrid g, Tracks t, double step_max,
                     int64_t n, void *out_any)
{
    constexpr bool kDir = (Q == qDistIn || Q == qDistOut);
    double *out = static_cast<double *>(out_any);
    int32_t *outi = static_cast<int32_t *>(out_any);
    __shared__ __align__(16) PconWalkSec tab[kMaxSec];
    __shared__ __align__(16) double seg[GRID ? 64 * kPconSegStride : 2];
    pcon_stage(p, tab);
    if (GRID) pcon_stage_segs(p, seg);
    pdl_launch_dependents();
    __syncthreads();
    pdl_wait();
    // every CTA owns ONE contiguous range of track pairs, the same number for all (rounded to a warp's row of 32): with
    // whole 512-track tiles handed out round-robin, a batch of 1.15 resident waves (n = 2^18) took two full wave times
    const int64_t npairs = (n + 1) >> 1;
    int64_t per = (npairs + gridDim.x - 1) / gridDim.x;
    per = (per + 31) / 32 * 32;
    const int64_t lo = int64_t(blockIdx.x) * per, hi = lo + per < npairs ? lo + per : npairs;
    for (int64_t j = lo + threadIdx.x; j < hi; j += kWalkBlock) {
        const int64_t i = 2 * j;
        if (i + 1 < n) {
            double2 x = ldg2(t.x + i), y = ldg2(t.y + i), z = ldg2(t.z + i);
            double2 dx = make_double2(0, 0), dy = dx, dz = dx;
            if (kDir) dx = ldg2(t.dx + i), dy = ldg2(t.dy + i), dz = ldg2(t.dz + i);
            if (Q == qInside) {
                bool in0, out0, in1, out1;
                pcon_walk_classify<WEDGE>(p, tab, x.x, y.x, z.x, in0, out0);
                pcon_walk_classify<WEDGE>(p, tab, x.y, y.y, z.y, in1, out1);
                stg2i(outi + i, classify(in0, out0), classify(in1, out1));
                continue;
            }
            const double r0 = pcon_walk_eval<Q, GRID, WEDGE>(p, tab, seg, g, x.x, y.x, z.x, dx.x, dy.x, dz.x, step_max);
            const double r1 = pcon_walk_eval<Q, GRID, WEDGE>(p, tab, seg, g, x.y, y.y, z.y, dx.y, dy.y, dz.y, step_max);
            stg2(out + i, r0, r1);
        } else {
            double x = ldg1(t.x + i), y = ldg1(t.y + i), z = ldg1(t.z + i);
            double dx = 0, dy = 0, dz = 0;
            if (kDir) dx = ldg1(t.dx + i), dy = ldg1(t.dy + i), dz = ldg1(t.dz + i);
            if (Q == qInside) {
                bool in0, out0;
                pcon_walk_classify<WEDGE>(p, tab, x, y, z, in0, out0);
                stg1i(outi + i, classify(in0, out0));
                continue;
            }
            stg1(out + i, pcon_walk_eval<Q, GRID, WEDGE>(p, tab, seg, g, x, y, z, dx, dy, dz, step_max));
        }
    }
}

// ---- the fused five-query call for a polycone (vg_query_all): one pass over the six coordinates ----
template <bool GRID, bool WEDGE>
VG_DEV void pcon_all_eval(const PolyconeP &p, const PconWalkSec *tab, const double *seg, const PconGrid &g, double x, double y,
                          double z, double dx, double dy, double dz, double step_max, int &cls, double &din, double &dout,
                          double &sdf)
{
    bool in, out;
    pcon_walk_classify<WEDGE>(p, tab, x, y, z, in, out);
    cls = classify(in, out);
    sdf = pcon_walk_eval<qSafeIn, GRID, WEDGE>(p, tab, seg, g, x, y, z, dx, dy, dz, step_max);
    din = pcon_walk_eval<qDistIn, GRID, WEDGE>(p, tab, seg, g, x, y, z, dx, dy, dz, step_max);
    dout = pcon_walk_eval<qDistOut, GRID, WEDGE>(p, tab, seg, g, x, y, z, dx, dy, dz, step_max);
}

template <bool GRID, bool WEDGE>
__global__ void __launch_bounds__(kWalkBlock, 2)
    pcon_all_kernel(const __grid_constant__ PolyconeP p, const __grid_constant__ PconGrid g, Tracks t, double step_max, int64_t n,
                    AllOut o)
{
    __shared__ __align__(16) PconWalkSec tab[kMaxSec];
    __shared__ __align__(16) double seg[GRID ? 64 * kPconSegStride : 2];
    pcon_stage(p, tab);
    if (GRID) pcon_stage_segs(p, seg);
    pdl_launch_dependents();
    __syncthreads();
    pdl_wait();
    const int64_t npairs = (n + 1) >> 1;
    for (int64_t j = int64_t(blockIdx.x) * kWalkBlock + threadIdx.x; j < npairs; j += int64_t(gridDim.x) * kWalkBlock) {
        const int64_t i = 2 * j;
        if (i + 1 < n) {
            const double2 x = ldg2(t.x + i), y = ldg2(t.y + i), z = ldg2(t.z + i);
            const double2 dx = ldg2(t.dx + i), dy = ldg2(t.dy + i), dz = ldg2(t.dz + i);
            int c0, c1;
            double a0, a1, b0, b1, s0, s1;
            pcon_all_eval<GRID, WEDGE>(p, tab, seg, g, x.x, y.x, z.x, dx.x, dy.x, dz.x, step_max, c0, a0, b0, s0);
            pcon_all_eval<GRID, WEDGE>(p, tab, seg, g, x.y, y.y, z.y, dx.y, dy.y, dz.y, step_max, c1, a1, b1, s1);
            stg2i(o.cls + i, c0, c1);
            stg2(o.din + i, a0, a1);
            stg2(o.dout + i, b0, b1);
            stg2(o.sin + i, s0, s1);
            stg2(o.sout + i, -s0, -s1);
        } else {
            int c0;
            double a0, b0, s0;
            pcon_all_eval<GRID, WEDGE>(p, tab, seg, g, ldg1(t.x + i), ldg1(t.y + i), ldg1(t.z + i), ldg1(t.dx + i), ldg1(t.dy + i),
                                       ldg1(t.dz + i), step_max, c0, a0, b0, s0);
            stg1i(o.cls + i, c0);
            stg1(o.din + i, a0);
            stg1(o.dout + i, b0);
            stg1(o.sin + i, s0);
            stg1(o.sout + i, -s0);
        }
    }
}

// ---- Inside and the two distances, one track per thread: the same ordered walks in 128-thread CTAs that read the section
// table from device memory (built at vg_shape_create; a few hundred bytes, L1-resident) instead of staging it.  No barrier,
// 46-48 registers against the persistent form's 70 with two tracks per thread, so twice the warps per SM to hide the walks'
// dependent FP64 chains: DistanceToIn 106 -> 93 us, DistanceToOut 132 -> 116 us, Inside 49 -> 44 us at 4 Mi tracks, 10.6 ->
// 8.0 us at 2^18, 402 -> 356 us at 2^24 (profiles/).  Any alignment, full phi or a phi cut.  The persistent kernel above
// still serves these queries when the table is not on the current device, and the safeties.
#ifndef VG_WALK_SMALL_BLOCK
#define VG_WALK_SMALL_BLOCK 128
#endif
constexpr int kWalkSmallBlock = VG_WALK_SMALL_BLOCK;

template <int Q, bool WEDGE>
__global__ void __launch_bounds__(kWalkSmallBlock)
    pcon_walk_small_kernel(const __grid_constant__ PolyconeP p, const PconWalkSec *__restrict__ tab, Tracks t, double step_max,
                           int64_t n, void *out_any)
{
    const int64_t i = int64_t(blockIdx.x) * kWalkSmallBlock + threadIdx.x;
    pdl_launch_dependents();
    pdl_wait();
    if (i >= n) return;
    const double x = ldg1(t.x + i), y = ldg1(t.y + i), z = ldg1(t.z + i);
    if (Q == qInside) {
        bool in, out;
        pcon_walk_classify<WEDGE>(p, tab, x, y, z, in, out);
        stg1i(static_cast<int32_t *>(out_any) + i, classify(in, out));
        return;
    }
    const double dx = ldg1(t.dx + i), dy = ldg1(t.dy + i), dz = ldg1(t.dz + i);
    const double r = Q == qDistOut ? pcon_walk_dist_out<WEDGE>(p, tab, x, y, z, dx, dy, dz)
                                   : pcon_walk_dist_in<WEDGE>(p, tab, x, y, z, dx, dy, dz);
    stg1(static_cast<double *>(out_any) + i, r <= step_max ? r : inf());
}

template <int Q, bool WEDGE>
cudaError_t launch_pcon_walk_small(const PolyconeP &p, const PconGrid &g, const Tracks &t, double step_max, int64_t n, void *out,
                                   cudaStream_t s)
{
    const unsigned grid = unsigned((n + kWalkSmallBlock - 1) / kWalkSmallBlock);
    return launch_kernel(pcon_walk_small_kernel<Q, WEDGE>, grid, kWalkSmallBlock, 0, s, p, g.wtab, t, step_max, n, out);
}

// ... and the safeties from the candidate grids the same way: segment records and section table read from device memory
template <int Q, bool WEDGE>
__global__ void __launch_bounds__(kWalkSmallBlock)
    pcon_safety_small_kernel(const __grid_constant__ PolyconeP p, const __grid_constant__ PconGrid g, Tracks t, int64_t n,
                             double *__restrict__ out)
{
    const int64_t i = int64_t(blockIdx.x) * kWalkSmallBlock + threadIdx.x;
    pdl_launch_dependents();
    pdl_wait();
    if (i >= n) return;
    const double x = ldg1(t.x + i), y = ldg1(t.y + i), z = ldg1(t.z + i);
    const double s = WEDGE ? pcon_grid_sdf_wedge(p, g.wtab, g.segs, g, x, y, z) : pcon_grid_sdf(p, g.wtab, g.segs, g, x, y, z);
    stg1(out + i, Q == qSafeIn ? s : -s);
}

template <int Q, bool WEDGE>
cudaError_t launch_pcon_safety_small(const PolyconeP &p, const PconGrid &g, const Tracks &t, int64_t n, void *out, cudaStream_t s)
{
    const unsigned grid = unsigned((n + kWalkSmallBlock - 1) / kWalkSmallBlock);
    return launch_kernel(pcon_safety_small_kernel<Q, WEDGE>, grid, kWalkSmallBlock, 0, s, p, g, t, n, static_cast<double *>(out));
}

// ... and the fused five-query call (vg_query_all)
template <bool WEDGE>
__global__ void __launch_bounds__(kWalkSmallBlock)
    pcon_all_small_kernel(const __grid_constant__ PolyconeP p, const __grid_constant__ PconGrid g, Tracks t, double step_max,
                          int64_t n, AllOut o)
{
    const int64_t i = int64_t(blockIdx.x) * kWalkSmallBlock + threadIdx.x;
    pdl_launch_dependents();
    pdl_wait();
    if (i >= n) return;
    int c0;
    double a0, b0, s0;
    pcon_all_eval<true, WEDGE>(p, g.wtab, g.segs, g, ldg1(t.x + i), ldg1(t.y + i), ldg1(t.z + i), ldg1(t.dx + i), ldg1(t.dy + i),
                               ldg1(t.dz + i), step_max, c0, a0, b0, s0);
    stg1i(o.cls + i, c0);
    stg1(o.din + i, a0);
    stg1(o.dout + i, b0);
    stg1(o.sin + i, s0);
    stg1(o.sout + i, -s0);
}

template <bool WEDGE>
cudaError_t launch_pcon_all_small(const PolyconeP &p, const PconGrid &g, const Tracks &t, double step_max, int64_t n, const AllOut &o,
                                  cudaStream_t s)
{
    const unsigned grid = unsigned((n + kWalkSmallBlock - 1) / kWalkSmallBlock);
    return launch_kernel(pcon_all_small_kernel<WEDGE>, grid, kWalkSmallBlock, 0, s, p, g, t, step_max, n, o);
}

template <bool GRID, bool WEDGE>
cudaError_t launch_pcon_all(const PolyconeP &p, const PconGrid &g, const Tracks &t, double step_max, int64_t n, const AllOut &o,
                            cudaStream_t s)
{
    int dev = 0, sms = 0, per_sm = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pcon_all_kernel<GRID, WEDGE>, kWalkBlock, 0)) != cudaSuccess) return e;
    const int64_t cap = int64_t(sms) * (per_sm < 1 ? 1 : per_sm), npairs = (n + 1) >> 1;
    int64_t grid = (npairs + kWalkBlock - 1) / kWalkBlock;
    if (grid > cap) grid = cap;
    return launch_kernel(pcon_all_kernel<GRID, WEDGE>, unsigned(grid), kWalkBlock, 0, s, p, g, t, step_max, n, o);
}

template <int Q, bool GRID, bool WEDGE = false>
cudaError_t launch_pcon_walk(const PolyconeP &p, const PconGrid &g, const Tracks &t, double step_max, int64_t n, void *out,
                             cudaStream_t s)
{
    constexpr int kMaxDev = 64; // resident CTAs of this instantiation, queried once per device
    static std::atomic<int> cap_cache[kMaxDev];
    int dev = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    int cap = (dev >= 0 && dev < kMaxDev) ? cap_cache[dev].load(std::memory_order_acquire) : 0;
    if (cap <= 0) {
        int sms = 0, per_sm = 0;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pcon_walk_kernel<Q, GRID, WEDGE>, kWalkBlock, 0)) != cudaSuccess) return e;
        cap = sms * (per_sm < 1 ? 1 : per_sm);
        if (dev >= 0 && dev < kMaxDev) cap_cache[dev].store(cap, std::memory_order_release);
    }
    const int64_t npairs = (n + 1) >> 1;
    int64_t grid = (npairs + kWalkBlock - 1) / kWalkBlock;
    if (grid > cap) grid = cap;
    return launch_kernel(pcon_walk_kernel<Q, GRID, WEDGE>, unsigned(grid), kWalkBlock, 0, s, p, g, t, step_max, n, out);
}

} // namespace vg
