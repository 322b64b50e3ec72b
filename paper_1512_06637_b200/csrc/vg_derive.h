// vg_derive.h -- host only: parameter validation and the derived constants of every solid (SURVEY.md sec. 8(a) A0:
// squared radii with the tolerance folded in, cos/sin of the phi planes, frustum generators, reciprocal edge
// lengths), computed once at vg_shape_create.  Included by vg_api.cu after its `fail(code, fmt, ...)` is defined.
#pragma once
#include "../../include/vg.h"
#include "vg_params.h"

#include <cmath>
#include <cstring>

using namespace vg;

struct vg_shape {
    int kind;
    union {
        BoxP box;
        OrbP orb;
        TubeP tube;
        ConeP cone;
        TrdP trd;
        PolyconeP pcon;
        BoolP boolean;
        CsgP csg;
    } u;
    // full-phi polycone only: the candidate grid of vg_pcon_grid.h in device memory of `grid_device` (masks == NULL if
    // no device was available at create; the safeties then run the ordered walk)
    PconGrid grid;
    int grid_device;
    // kBoolX only: the polycone operands' constants in device memory of `ext_device` (u.boolean's operand records point
    // into it); owned by the shape
    void *ext_blob;
    int ext_device;
    PolyconeP *ext_host; // ... and their host copies, in operand order (a world that places the boolean uploads its own)
};

// ------------------------------------------------------------------------------------------- derived constants

static const double kTwoPi = 2.0 * 3.14159265358979323846;

static Wedge make_wedge(double sphi, double dphi)
{
    Wedge w;
    w.full = dphi >= kTwoPi;
    w.wide = dphi > 0.5 * kTwoPi;
    w.e0x = std::cos(sphi);
    w.e0y = std::sin(sphi);
    w.e1x = std::cos(sphi + dphi);
    w.e1y = std::sin(sphi + dphi);
    return w;
}

static Frustum make_frustum(double z0, double r0, double z1, double r1)
{
    Frustum f;
    f.B = (r1 - r0) / (z1 - z0);
    f.A = r0 - f.B * z0;
    f.sec = std::sqrt(1.0 + f.B * f.B);
    f.r0 = r0;
    f.er = r1 - r0;
    f.inv_l2 = 1.0 / (f.er * f.er + (z1 - z0) * (z1 - z0));
    return f;
}

static bool all_finite(const double *p, int n)
{
    for (int i = 0; i < n; ++i)
        if (!std::isfinite(p[i])) return false;
    return true;
}

static int fill_shape(vg_shape *s, vg_kind kind, const double *p, int np)
{
    s->kind = kind;
    switch (kind) {
    case VG_BOX:
        if (np != 3) return fail(VG_ERR_PARAM, "box: 3 parameters expected, got %d", np);
        if (!(p[0] > 0 && p[1] > 0 && p[2] > 0)) return fail(VG_ERR_PARAM, "box: half-lengths must be > 0");
        s->u.box = BoxP{ p[0], p[1], p[2] };
        return VG_OK;
    case VG_ORB:
        if (np != 1) return fail(VG_ERR_PARAM, "orb: 1 parameter expected, got %d", np);
        if (!(p[0] > 0)) return fail(VG_ERR_PARAM, "orb: r must be > 0");
        s->u.orb.r = p[0];
        s->u.orb.r2 = p[0] * p[0];
        s->u.orb.rin2 = p[0] > kTol ? (p[0] - kTol) * (p[0] - kTol) : 0.0;
        s->u.orb.rout2 = (p[0] + kTol) * (p[0] + kTol);
        return VG_OK;
    case VG_TUBE: {
        if (np != 5) return fail(VG_ERR_PARAM, "tube: 5 parameters expected, got %d", np);
        double rmin = p[0], rmax = p[1], dz = p[2];
        if (!(rmin >= 0 && rmax > rmin && dz > 0 && p[4] > 0))
            return fail(VG_ERR_PARAM, "tube: need 0 <= rmin < rmax, dz > 0, dphi > 0");
        TubeP &t = s->u.tube;
        t.rmin = rmin;
        t.rmax = rmax;
        t.dz = dz;
        t.rmin2 = rmin * rmin;
        t.rmax2 = rmax * rmax;
        t.rmin_in2 = (rmin + kTol) * (rmin + kTol);
        t.rmax_in2 = (rmax - kTol) * (rmax - kTol);
        t.rmin_out2 = rmin > kTol ? (rmin - kTol) * (rmin - kTol) : 0.0;
        t.rmax_out2 = (rmax + kTol) * (rmax + kTol);
        t.rc = 0.5 * (rmin + rmax), t.rh = 0.5 * (rmax - rmin);
        t.w = make_wedge(p[3], p[4]);
        t.hollow = rmin > 0;
        return VG_OK;
    }
    case VG_CONE: {
        if (np != 7) return fail(VG_ERR_PARAM, "cone: 7 parameters expected, got %d", np);
        double rmin1 = p[0], rmax1 = p[1], rmin2 = p[2], rmax2 = p[3], dz = p[4];
        if (!(rmin1 >= 0 && rmax1 > rmin1 && rmin2 >= 0 && rmax2 > rmin2 && dz > 0 && p[6] > 0))
            return fail(VG_ERR_PARAM, "cone: need 0 <= rmin < rmax at both ends, dz > 0, dphi > 0");
        ConeP &c = s->u.cone;
        c.dz = dz;
        c.out = make_frustum(-dz, rmax1, dz, rmax2);
        c.in = make_frustum(-dz, rmin1, dz, rmin2);
        c.rmin1 = rmin1;
        c.rmax1 = rmax1;
        c.rmin2 = rmin2;
        c.rmax2 = rmax2;
        c.w = make_wedge(p[5], p[6]);
        c.hollow = rmin1 > 0 || rmin2 > 0;
        c.cap_c1 = 0.5 * (rmin1 + rmax1), c.cap_h1 = 0.5 * (rmax1 - rmin1);
        c.cap_c2 = 0.5 * (rmin2 + rmax2), c.cap_h2 = 0.5 * (rmax2 - rmin2);
        return VG_OK;
    }
    case VG_TRD: {
        if (np != 5) return fail(VG_ERR_PARAM, "trd: 5 parameters expected, got %d", np);
        for (int i = 0; i < 5; ++i)
            if (!(p[i] > 0)) return fail(VG_ERR_PARAM, "trd: half-lengths must be > 0");
        TrdP &t = s->u.trd;
        t.dx1 = p[0];
        t.dx2 = p[1];
        t.dy1 = p[2];
        t.dy2 = p[3];
        t.dz = p[4];
        t.fx = (t.dx2 - t.dx1) / (2 * t.dz);
        t.mx = (t.dx1 + t.dx2) / 2;
        t.cx = std::sqrt(1 + t.fx * t.fx);
        t.icx = 1 / t.cx;
        t.fy = (t.dy2 - t.dy1) / (2 * t.dz);
        t.my = (t.dy1 + t.dy2) / 2;
        t.cy = std::sqrt(1 + t.fy * t.fy);
        t.icy = 1 / t.cy;
        // slanted edge of the +x face: half-widths dy1 -> dy2 over the slant height 2 dz cx; likewise +y
        t.inv_kx = 1 / ((t.dy2 - t.dy1) * (t.dy2 - t.dy1) + 4 * t.dz * t.dz * t.cx * t.cx);
        t.inv_ky = 1 / ((t.dx2 - t.dx1) * (t.dx2 - t.dx1) + 4 * t.dz * t.dz * t.cy * t.cy);
        t.hex = t.dz * t.cx, t.hey = t.dz * t.cy;
        t.sfx = t.icx * t.fx, t.sfy = t.icy * t.fy;
        t.kxx = t.dy2 - t.dy1, t.kyx = 2.0 * t.hex, t.kxx_s = t.kxx * t.inv_kx, t.kyx_s = t.kyx * t.inv_kx;
        t.kxy = t.dx2 - t.dx1, t.kyy = 2.0 * t.hey, t.kxy_s = t.kxy * t.inv_ky, t.kyy_s = t.kyy * t.inv_ky;
        return VG_OK;
    }
    case VG_POLYCONE: {
        if (np < 3) return fail(VG_ERR_PARAM, "polycone: at least 3 parameters expected");
        int nz = int(p[2]);
        if (double(nz) != p[2] || nz < 2 || nz > VG_MAX_ZPLANES)
            return fail(VG_ERR_PARAM, "polycone: nz must be an integer in [2, %d]", VG_MAX_ZPLANES);
        if (np != 3 + 3 * nz) return fail(VG_ERR_PARAM, "polycone: %d parameters expected, got %d", 3 + 3 * nz, np);
        if (!(p[1] > 0)) return fail(VG_ERR_PARAM, "polycone: dphi must be > 0");
        const double *zp = p + 3;
        for (int i = 0; i < nz; ++i) {
            if (!(zp[3 * i + 1] >= 0 && zp[3 * i + 2] > zp[3 * i + 1]))
                return fail(VG_ERR_PARAM, "polycone: need 0 <= rmin < rmax at plane %d", i);
            if (i > 0 && !(zp[3 * i] >= zp[3 * (i - 1)]))
                return fail(VG_ERR_PARAM, "polycone: z must not decrease (plane %d)", i);
            if (i > 0 && zp[3 * i] == zp[3 * (i - 1)]) { // a z step (reading R26)
                if (i == 1 || i == nz - 1) return fail(VG_ERR_PARAM, "polycone: a z step at an end plane (plane %d)", i);
                if (zp[3 * i] == zp[3 * (i - 2)]) return fail(VG_ERR_PARAM, "polycone: three planes at one z (plane %d)", i);
                if (!(std::fmax(zp[3 * i + 1], zp[3 * i - 2]) < std::fmin(zp[3 * i + 2], zp[3 * i - 1])))
                    return fail(VG_ERR_PARAM, "polycone: radial ranges on the two sides of the z step at plane %d do not overlap", i);
            }
        }
        PolyconeP &c = s->u.pcon;
        std::memset(&c, 0, sizeof c);
        c.w = make_wedge(p[0], p[1]);
        c.zlo = zp[0];
        c.zhi = zp[3 * (nz - 1)];
        c.cap_lo_rmin = zp[1];
        c.cap_lo_rmax = zp[2];
        c.cap_hi_rmin = zp[3 * (nz - 1) + 1];
        c.cap_hi_rmax = zp[3 * (nz - 1) + 2];
        {
            double rb = 0;
            for (int i = 0; i < nz; ++i) rb = std::fmax(rb, zp[3 * i + 2]);
            c.rb2 = rb * rb * (1 + 2e-9);
        }
        int ns = 0;
        for (int k = 0; k < nz - 1; ++k) {
            const double *a = zp + 3 * k, *b = zp + 3 * (k + 1);
            if (b[0] == a[0]) { // the step between the section just stored and the next one
                PconStep &t = c.step[ns - 1];
                t.z = a[0];
                t.olo = std::fmin(a[2], b[2]), t.ohi = std::fmax(a[2], b[2]);
                t.ilo = std::fmin(a[1], b[1]), t.ihi = std::fmax(a[1], b[1]);
                t.oup = a[2] > b[2];
                t.iup = a[1] < b[1];
                if (!(t.ohi > t.olo)) t.olo = 1.0, t.ohi = -1.0; // no jump: an empty range no radius falls into
                if (!(t.ihi > t.ilo)) t.ilo = 1.0, t.ihi = -1.0;
                c.step_mask |= 1u << (ns - 1);
                ++c.nstep;
                continue;
            }
            c.sec[ns].z0 = a[0];
            c.sec[ns].z1 = b[0];
            c.sec[ns].out = make_frustum(a[0], a[2], b[0], b[2]);
            c.sec[ns].in = make_frustum(a[0], a[1], b[0], b[1]);
            if (a[1] > 0 || b[1] > 0) c.inner_mask |= 1u << ns;
            ++ns;
        }
        c.nsec = ns;
        return VG_OK;
    }
    }
    if (kind == VG_BOOLEAN) return fail(VG_ERR_ARG, "a boolean solid is made by vg_boolean_create");
    return fail(VG_ERR_PARAM, "unknown shape kind %d", int(kind));
}

