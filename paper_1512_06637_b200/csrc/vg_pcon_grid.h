// vg_pcon_grid.h -- host only: the candidate grid of a full-phi polycone, built once at vg_shape_create
// (SURVEY.md sec. 8(a) A0 "shape set-up"; the safeties are the exact signed distance of sec. 8(c) c.3).
//
// The exact distance from (rho, z) to the (r, z) outline is the minimum over its segments (outer and inner edge of
// every section, the two end caps, the annular faces of z steps).  For a CELL of a regular (rho, z) grid only a few segments can be that minimum
// for any point of the cell: segment s is a candidate iff
//     dmin_s(cell) <= min over s' of dmax_s'(cell)
// (the nearest segment s* of a point p of the cell has d(p, s*) <= d(p, s') <= dmax_s' for every s', and
// dmin_s* <= d(p, s*)).  dmax_s is the largest distance from a cell corner to s (the distance to a convex set is a
// convex function, so its maximum over a rectangle sits at a corner); dmin_s is 0 if s meets the cell, else the
// smaller of the corner-to-segment and endpoint-to-cell distances (two disjoint convex polygons in the plane are
// closest at a vertex of one of them).  Both are evaluated for the cell inflated by `margin`, and the comparison
// carries a slack, so a point that rounding bins into a neighbouring cell still finds its nearest segment.
// The kernel (vg_pcon_walk.cuh, pcon_grid_sdf) evaluates the candidates of the point's cell only: same minimum,
// same arithmetic per segment, a fraction of the work.  Points outside the grid take the ordered walk.
#pragma once
#include "vg_params.h"

#include <cmath>
#include <cstring>
#include <vector>

namespace vg {

struct PconSegH {
    double r0, z0, r1, z1;
    int bit;
};

// plain selects (std::fmax / std::fmin are libm calls without fast-math; no NaN can reach these)
static inline double pg_max(double a, double b) { return a > b ? a : b; }
static inline double pg_min(double a, double b) { return a < b ? a : b; }

// squared distances (the builder compares squares and takes one square root per cell)
static inline double pg_dist2_seg(double u, double v, const PconSegH &s, double inv_l2)
{
    double er = s.r1 - s.r0, ez = s.z1 - s.z0;
    double t = ((u - s.r0) * er + (v - s.z0) * ez) * inv_l2;
    t = t < 0 ? 0 : (t > 1 ? 1 : t);
    double du = u - s.r0 - t * er, dv = v - s.z0 - t * ez;
    return du * du + dv * dv;
}

static inline double pg_dist2_rect(double u, double v, double u0, double u1, double v0, double v1)
{
    double qu = pg_max(pg_max(u0 - u, u - u1), 0.0), qv = pg_max(pg_max(v0 - v, v - v1), 0.0);
    return qu * qu + qv * qv;
}

// does the segment meet the closed rectangle?  (Liang-Barsky clip of t in [0, 1])
static inline bool pg_seg_meets_rect(const PconSegH &s, double u0, double u1, double v0, double v1)
{
    double t0 = 0, t1 = 1;
    const double p[4] = { -(s.r1 - s.r0), s.r1 - s.r0, -(s.z1 - s.z0), s.z1 - s.z0 };
    const double q[4] = { s.r0 - u0, u1 - s.r0, s.z0 - v0, v1 - s.z0 };
    for (int i = 0; i < 4; ++i) {
        if (p[i] == 0) {
            if (q[i] < 0) return false;
        } else {
            double r = q[i] / p[i];
            if (p[i] < 0) t0 = pg_max(t0, r);
            else t1 = pg_min(t1, r);
        }
    }
    return t0 <= t1;
}

// segment numbering shared with the kernel (vg_params.h): bits 0 / 1 = the caps, 2 + 2k / 3 + 2k = outer / inner edge of
// section k, then two bits per z step
// `face` = false: the grid of the surface of revolution (rho in [0, R): kPconGridR columns, edges on the axis left out).
// `face` = true: the grid of a phi FACE (u in [-R, R): 2 kPconGridR columns, EVERY edge of the outline: on a face the
// edges on the axis bound the filled outline too, c.3), used for points outside the outline.
static inline void pcon_grid_build(const PolyconeP &c, bool face, PconGridGeom *geom, std::vector<unsigned long long> *masks,
                                   std::vector<unsigned char> *rows)
{
    std::vector<PconSegH> segs;
    double rmax = 0;
    const int ncol = face ? 2 * kPconGridR : kPconGridR;
    for (int k = 0; k < c.nsec; ++k) {
        const PconSec &s = c.sec[k];
        segs.push_back(PconSegH{ s.out.r0, s.z0, s.out.r0 + s.out.er, s.z1, kPconSecBit0 + 2 * k });
        if (face || ((c.inner_mask >> k) & 1u)) segs.push_back(PconSegH{ s.in.r0, s.z0, s.in.r0 + s.in.er, s.z1, kPconSecBit0 + 2 * k + 1 });
        rmax = pg_max(rmax, pg_max(s.out.r0, s.out.r0 + s.out.er));
    }
    for (int k = 0, j = 0; k + 1 < c.nsec; ++k) { // the annular faces of the z steps (R26), bits after the sections
        if (!((c.step_mask >> k) & 1u)) continue;
        const PconStep &t = c.step[k];
        const int bit = kPconSecBit0 + 2 * c.nsec + 2 * j++;
        if (t.ohi > t.olo) segs.push_back(PconSegH{ t.olo, t.z, t.ohi, t.z, bit });
        if (t.ihi > t.ilo) segs.push_back(PconSegH{ t.ilo, t.z, t.ihi, t.z, bit + 1 });
    }
    segs.push_back(PconSegH{ c.cap_lo_rmin, c.zlo, c.cap_lo_rmax, c.zlo, kPconCapLoBit });
    segs.push_back(PconSegH{ c.cap_hi_rmin, c.zhi, c.cap_hi_rmax, c.zhi, kPconCapHiBit });

    const double zl = c.zhi - c.zlo;
    const double R = 2.25 * rmax, zg0 = c.zlo - 0.5 * zl, zg1 = c.zhi + 0.5 * zl;
    const double cr = R / kPconGridR, cz = (zg1 - zg0) / kPconGridZ;
    geom->inv_cr = 1.0 / cr;
    geom->inv_cz = 1.0 / cz;
    geom->zg0 = zg0;
    const double margin = 1e-6 * pg_max(cr, cz); // dmin, dmax, thr below are SQUARED distances
    const size_t ns = segs.size();

    // corner lattice of squared distances, one layer per segment
    const int LR = ncol + 1, LZ = kPconGridZ + 1;
    const double umin = face ? -R : 0.0;
    std::vector<double> D(ns * size_t(LR) * LZ);
    for (size_t s = 0; s < ns; ++s) {
        const double er = segs[s].r1 - segs[s].r0, ez = segs[s].z1 - segs[s].z0, inv_l2 = 1.0 / (er * er + ez * ez);
        for (int j = 0; j < LZ; ++j)
            for (int i = 0; i < LR; ++i) D[(s * LZ + j) * LR + i] = pg_dist2_seg(umin + i * cr, zg0 + j * cz, segs[s], inv_l2);
    }

    masks->assign(size_t(ncol) * kPconGridZ, 0ull);
    std::vector<double> dmin(ns);
    for (int j = 0; j < kPconGridZ; ++j)
        for (int i = 0; i < ncol; ++i) {
            const double u0 = umin + i * cr, u1 = u0 + cr, v0 = zg0 + j * cz, v1 = v0 + cz;
            double thr = INFINITY;
            for (size_t s = 0; s < ns; ++s) {
                const double *L = &D[(s * LZ + j) * LR + i];
                const double d00 = L[0], d10 = L[1], d01 = L[LR], d11 = L[LR + 1];
                const double mx = pg_max(pg_max(d00, d10), pg_max(d01, d11));
                double mn = pg_min(pg_min(d00, d10), pg_min(d01, d11));
                mn = pg_min(mn, pg_dist2_rect(segs[s].r0, segs[s].z0, u0, u1, v0, v1));
                mn = pg_min(mn, pg_dist2_rect(segs[s].r1, segs[s].z1, u0, u1, v0, v1));
                const bool boxes_meet = pg_min(segs[s].r0, segs[s].r1) <= u1 + margin && pg_max(segs[s].r0, segs[s].r1) >= u0 - margin &&
                                        segs[s].z0 <= v1 + margin && segs[s].z1 >= v0 - margin;
                if (boxes_meet && pg_seg_meets_rect(segs[s], u0 - margin, u1 + margin, v0 - margin, v1 + margin)) mn = 0;
                dmin[s] = mn;
                thr = pg_min(thr, mx);
            }
            // inflation by `margin` moves either bound by at most sqrt(2) margin; relative slack for the FMA rounding
            thr = std::sqrt(thr) * (1 + 1e-9) + 4 * margin;
            thr *= thr;
            unsigned long long m = 0;
            for (size_t s = 0; s < ns; ++s)
                if (dmin[s] <= thr) m |= 1ull << segs[s].bit;
            (*masks)[size_t(j) * ncol + i] = m;
        }

    // section index at (slightly below) the lower edge of every z row: the kernel counts on from there
    rows->assign(kPconGridZ, 0);
    for (int j = 0; j < kPconGridZ; ++j) {
        const double zr = zg0 + j * cz - margin;
        int k = 0;
        for (int q = 1; q < c.nsec; ++q) k += (c.sec[q].z0 <= zr) ? 1 : 0;
        (*rows)[j] = (unsigned char)k;
    }
}

} // namespace vg
