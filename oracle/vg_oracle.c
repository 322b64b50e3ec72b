/*
 * vg_oracle.c -- ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, scalar CPU implementation of what the hot path computes:
 * the three geometry questions of the paper (sec. III.C:
 * "Is the particle inside or outside the solid?", "What is the minimal
 * distance between the particle and the border of the solid?", "What is the
 * maximal step length for a particle with a given velocity and direction?")
 * for box / orb / tube segment / cone segment / trd / polycone, the
 * one-level navigation step (distance to the geometric
 * border against the physics step; "coordinate transformations and distance
 * calculations"), and the same step in a tree of placed volumes with the
 * point location that goes with it ("hierarchical connections";
 * readings R22-R25 at the end of this file), and boolean solids of two
 * primitives (readings R27-R29 at the end of this file).
 *
 * The paper gives no formula for any solid.  Every query here is the PLAIN
 * DEFINITION written out as brute force over the boundary patches of the
 * solid, following the readings R1-R21 of SURVEY.md sec. 8(c) (listed again in
 * DESIGN.md):
 *   - solids as closed point sets ................ SURVEY.md 8(c) c.1
 *   - Inside / Safety / Cross / Distance / Step ... SURVEY.md 8(c) c.2
 *   - exact signed Euclidean distance per solid ... SURVEY.md 8(c) c.3
 *   - first boundary crossing per solid ........... SURVEY.md 8(c) c.4
 * No early-outs, no symmetry tricks, no direction filters, IEEE divides and
 * square roots, atan2 for the phi wedge.  Compile with -O2 -ffp-contract=off.
 *
 * Independence: this file shares NO code, header, table or constant
 * generator with paper_1512_06637_b200/csrc (the CUDA path) and includes
 * nothing from include/.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): closed forms and hand-worked
 * examples E1-E21 (tests/golden/worked_examples.txt), brute-force surface
 * sampling for every sdf, the eikonal property, sphere tracing and ray
 * marching for every first crossing, special-case reductions between solids
 * (trd==box, cone==tube, polycone==cone==tube, inserted collinear z-plane),
 * rigid-motion and permutation invariance of the navigation step, the world
 * queries against per-node membership / one-level steps composed in numpy and
 * against marching through orc_world_locate (tests/test_oracle_world.py), the
 * boolean solids against set-definition membership, ray marching, reductions
 * to one primitive and the never-over-estimating property of their composed
 * safety (tests/test_oracle_boolean.py), and
 * the 80-bit long-double build of this same file (-DORC_LONG_DOUBLE).
 * Start points INSIDE the kTol surface band follow reading R32 (stated above
 * surface_cross below; pins in tests/test_oracle_surface.py); it replaces R7.
 * Parity unpinned: nothing under readings R1-R32.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef ORC_LONG_DOUBLE
typedef long double real;
#define R_SQRT sqrtl
#define R_ATAN2 atan2l
#define R_FABS fabsl
#define R_FMOD fmodl
#define R_COS cosl
#define R_SIN sinl
#define R_PI 3.14159265358979323846264338327950288L
#else
typedef double real;
#define R_SQRT sqrt
#define R_ATAN2 atan2
#define R_FABS fabs
#define R_FMOD fmod
#define R_COS cos
#define R_SIN sin
#define R_PI 3.14159265358979323846
#endif

#define ORC_KTOL ((real)1e-9)      /* BASELINE.json: kTolerance = 1e-9; reading R6 */
#define ORC_INF ((real)INFINITY)   /* reading R5: a miss is IEEE +inf            */
#define ORC_MAXZ 32                /* polycone: at most 32 z-planes               */
#define ORC_MAXV (2 * ORC_MAXZ)

enum { ORC_BOX = 0, ORC_ORB = 1, ORC_TUBE = 2, ORC_CONE = 3, ORC_TRD = 4, ORC_POLYCONE = 5 };
enum { ORC_OUTSIDE = 0, ORC_SURFACE = 1, ORC_INSIDE = 2 };

typedef struct {
    int kind;
    real h[3];                 /* box half-lengths                                      */
    real r;                    /* orb radius                                            */
    real trd[5];               /* dx1 dx2 dy1 dy2 dz                                    */
    real pn[6][3], ph[6];      /* trd: six half-spaces n.p <= h, unit normals           */
    real fv[6][4][3];          /* trd: the four corners of each face, in order          */
    int nv;                    /* RZ polygon (tube, cone, polycone): vertex count       */
    real pr[ORC_MAXV], pz[ORC_MAXV];
    real sphi, dphi;
    int full;                  /* dphi >= 2 pi                                          */
    real e[2][2];              /* unit vectors of the two phi planes (cos, sin)         */
} orc_shape;

typedef struct {
    const orc_shape *mother;
    int nd;
    const orc_shape **daughter;
    real *xf;                  /* nd * 12, row-major [R | b], mother -> local (R12)     */
} orc_volume;

static real rmin2(real a, real b) { return a < b ? a : b; }
static real rmax2(real a, real b) { return a > b ? a : b; }

/* ------------------------------------------------------------------ create */

static int finite_all(const double *p, int n)
{
    for (int i = 0; i < n; ++i)
        if (!isfinite(p[i])) return 0;
    return 1;
}

static void set_wedge(orc_shape *s, real sphi, real dphi)
{
    s->sphi = sphi;
    s->dphi = dphi;
    /* "dphi >= 2 pi means full": 2 pi is the FP64 value in both builds */
    s->full = (dphi >= (real)(2.0 * 3.14159265358979323846));
    /* reading R11: cos/sin of the phi planes evaluated once at create */
    s->e[0][0] = R_COS(sphi);
    s->e[0][1] = R_SIN(sphi);
    s->e[1][0] = R_COS(sphi + dphi);
    s->e[1][1] = R_SIN(sphi + dphi);
}

static void trd_setup(orc_shape *s)
{
    /* SURVEY.md 8(c) c.3 "trd": six half-spaces with unit normals. */
    real dx1 = s->trd[0], dx2 = s->trd[1], dy1 = s->trd[2], dy2 = s->trd[3], dz = s->trd[4];
    real fx = (dx2 - dx1) / (2 * dz), mx = (dx1 + dx2) / 2, cx = R_SQRT(1 + fx * fx);
    real fy = (dy2 - dy1) / (2 * dz), my = (dy1 + dy2) / 2, cy = R_SQRT(1 + fy * fy);
    real n[6][3] = { { 0, 0, -1 }, { 0, 0, 1 }, { 1 / cx, 0, -fx / cx }, { -1 / cx, 0, -fx / cx },
                     { 0, 1 / cy, -fy / cy }, { 0, -1 / cy, -fy / cy } };
    real h[6] = { dz, dz, mx / cx, mx / cx, my / cy, my / cy };
    memcpy(s->pn, n, sizeof n);
    memcpy(s->ph, h, sizeof h);
    /* corners: (+-dx1, +-dy1, -dz), (+-dx2, +-dy2, +dz) */
    real f[6][4][3] = {
        { { -dx1, -dy1, -dz }, { dx1, -dy1, -dz }, { dx1, dy1, -dz }, { -dx1, dy1, -dz } },   /* -z */
        { { -dx2, -dy2, dz }, { dx2, -dy2, dz }, { dx2, dy2, dz }, { -dx2, dy2, dz } },       /* +z */
        { { dx1, -dy1, -dz }, { dx1, dy1, -dz }, { dx2, dy2, dz }, { dx2, -dy2, dz } },       /* +x */
        { { -dx1, -dy1, -dz }, { -dx1, dy1, -dz }, { -dx2, dy2, dz }, { -dx2, -dy2, dz } },   /* -x */
        { { -dx1, dy1, -dz }, { dx1, dy1, -dz }, { dx2, dy2, dz }, { -dx2, dy2, dz } },       /* +y */
        { { -dx1, -dy1, -dz }, { dx1, -dy1, -dz }, { dx2, -dy2, dz }, { -dx2, -dy2, dz } },   /* -y */
    };
    memcpy(s->fv, f, sizeof f);
}

/* Parameter layouts: SURVEY.md 8(b).  Returns NULL for invalid parameters. */
orc_shape *orc_shape_create(int kind, const double *par, int np)
{
    if (!par || np <= 0 || !finite_all(par, np)) return NULL;
    orc_shape *s = (orc_shape *)calloc(1, sizeof *s);
    if (!s) return NULL;
    s->kind = kind;
    s->full = 1;
    int ok = 0;
    switch (kind) {
    case ORC_BOX:
        if (np == 3 && par[0] > 0 && par[1] > 0 && par[2] > 0) {
            for (int i = 0; i < 3; ++i) s->h[i] = par[i];
            ok = 1;
        }
        break;
    case ORC_ORB:
        if (np == 1 && par[0] > 0) { s->r = par[0]; ok = 1; }
        break;
    case ORC_TUBE: /* rmin rmax dz sphi dphi : rectangle in (r, z), c.1 */
        if (np == 5 && par[0] >= 0 && par[1] > par[0] && par[2] > 0 && par[4] > 0) {
            real rmin = par[0], rmax = par[1], dz = par[2];
            s->nv = 4;
            s->pr[0] = rmin; s->pz[0] = -dz;
            s->pr[1] = rmax; s->pz[1] = -dz;
            s->pr[2] = rmax; s->pz[2] = dz;
            s->pr[3] = rmin; s->pz[3] = dz;
            set_wedge(s, par[3], par[4]);
            ok = 1;
        }
        break;
    case ORC_CONE: /* rmin1 rmax1 rmin2 rmax2 dz sphi dphi : quadrilateral, c.1 */
        if (np == 7 && par[0] >= 0 && par[1] > par[0] && par[2] >= 0 && par[3] > par[2] && par[4] > 0 &&
            par[6] > 0) {
            real dz = par[4];
            s->nv = 4;
            s->pr[0] = par[0]; s->pz[0] = -dz;
            s->pr[1] = par[1]; s->pz[1] = -dz;
            s->pr[2] = par[3]; s->pz[2] = dz;
            s->pr[3] = par[2]; s->pz[3] = dz;
            set_wedge(s, par[5], par[6]);
            ok = 1;
        }
        break;
    case ORC_TRD:
        if (np == 5 && par[0] > 0 && par[1] > 0 && par[2] > 0 && par[3] > 0 && par[4] > 0) {
            for (int i = 0; i < 5; ++i) s->trd[i] = par[i];
            trd_setup(s);
            ok = 1;
        }
        break;
    case ORC_POLYCONE: { /* sphi dphi nz (z rmin rmax)*nz : 2n-gon, c.1; readings R18, R26 */
        if (np < 3) break;
        int nz = (int)par[2];
        if ((double)nz != par[2] || nz < 2 || nz > ORC_MAXZ || np != 3 + 3 * nz || !(par[1] > 0)) break;
        ok = 1;
        for (int i = 0; i < nz; ++i) {
            double z = par[3 + 3 * i], rmin = par[4 + 3 * i], rmax = par[5 + 3 * i];
            if (rmin < 0 || rmax <= rmin) ok = 0;
            if (i > 0 && !(z >= par[3 + 3 * (i - 1)])) ok = 0;
            if (i > 0 && z == par[3 + 3 * (i - 1)]) {
                /* reading R26: two planes at the same z are a STEP, the radii jump there and the
                 * outline gets a horizontal edge (an annular face).  Not at either end, not three planes at one z, and
                 * the radial ranges on both sides must overlap, so that the outline stays a simple polygon. */
                double rmin_p = par[4 + 3 * (i - 1)], rmax_p = par[5 + 3 * (i - 1)];
                if (i == 1 || i == nz - 1) ok = 0;
                if (i >= 2 && z == par[3 + 3 * (i - 2)]) ok = 0;
                if (!((rmin_p > rmin ? rmin_p : rmin) < (rmax_p < rmax ? rmax_p : rmax))) ok = 0;
            }
            /* (rmin_0,z_0) ... (rmin_{n-1},z_{n-1}), (rmax_{n-1},z_{n-1}) ... (rmax_0,z_0) */
            s->pr[i] = rmin; s->pz[i] = z;
            s->pr[2 * nz - 1 - i] = rmax; s->pz[2 * nz - 1 - i] = z;
        }
        s->nv = 2 * nz;
        set_wedge(s, par[0], par[1]);
        break;
    }
    default:
        break;
    }
    if (!ok) { free(s); return NULL; }
    return s;
}

void orc_shape_destroy(orc_shape *s) { free(s); }

/* -------------------------------------------- RZ polygon + phi wedge (c.3) */

static int edge_on_axis(const orc_shape *s, int i)
{
    int j = (i + 1) % s->nv;
    return s->pr[i] == 0 && s->pr[j] == 0;
}

/* even-odd point-in-polygon in the (r, z) half plane */
static int in_poly(const orc_shape *s, real u, real v)
{
    int in = 0;
    for (int i = 0; i < s->nv; ++i) {
        int j = (i + 1) % s->nv;
        real ri = s->pr[i], zi = s->pz[i], rj = s->pr[j], zj = s->pz[j];
        if ((zi > v) != (zj > v)) {
            real ucross = ri + (v - zi) * (rj - ri) / (zj - zi);
            if (u < ucross) in = !in;
        }
    }
    return in;
}

static real seg_d2(real u, real v, real r0, real z0, real r1, real z1)
{
    real eu = r1 - r0, ev = z1 - z0, wu = u - r0, wv = v - z0;
    real L2 = eu * eu + ev * ev;
    real t = L2 > 0 ? (wu * eu + wv * ev) / L2 : 0;
    if (t < 0) t = 0;
    if (t > 1) t = 1;
    real du = wu - t * eu, dv = wv - t * ev;
    return du * du + dv * dv;
}

/* min squared distance to the polygon edges; axis edges are not a surface */
static real poly_d2(const orc_shape *s, real u, real v, int skip_axis)
{
    real best = ORC_INF;
    for (int i = 0; i < s->nv; ++i) {
        if (skip_axis && edge_on_axis(s, i)) continue;
        int j = (i + 1) % s->nv;
        best = rmin2(best, seg_d2(u, v, s->pr[i], s->pz[i], s->pr[j], s->pz[j]));
    }
    return best;
}

static int in_phi(const orc_shape *s, real x, real y)
{
    if (s->full) return 1;
    real phi = R_ATAN2(y, x);
    real d = R_FMOD(phi - s->sphi, 2 * R_PI);
    if (d < 0) d += 2 * R_PI;
    return d <= s->dphi;
}

static real sdf_rz(const orc_shape *s, real x, real y, real z)
{
    real rho = R_SQRT(x * x + y * y);
    int inphi = in_phi(s, x, y);
    int inside = inphi && in_poly(s, rho, z);
    real D2 = ORC_INF;
    if (inphi) D2 = poly_d2(s, rho, z, 1);
    if (!s->full) {
        for (int k = 0; k < 2; ++k) {
            real ex = s->e[k][0], ey = s->e[k][1];
            real u = x * ex + y * ey;
            real w = -x * ey + y * ex;
            real dF2 = in_poly(s, u, z) ? 0 : poly_d2(s, u, z, 0);
            D2 = rmin2(D2, w * w + dF2);
        }
    }
    real D = R_SQRT(D2);
    return inside ? -D : D;
}

/* --------------------------------------------------------------- trd (c.3) */

static real seg3_d2(const real p[3], const real a[3], const real b[3])
{
    real e[3], w[3], L2 = 0, we = 0;
    for (int i = 0; i < 3; ++i) { e[i] = b[i] - a[i]; w[i] = p[i] - a[i]; L2 += e[i] * e[i]; we += w[i] * e[i]; }
    real t = L2 > 0 ? we / L2 : 0;
    if (t < 0) t = 0;
    if (t > 1) t = 1;
    real d2 = 0;
    for (int i = 0; i < 3; ++i) { real d = w[i] - t * e[i]; d2 += d * d; }
    return d2;
}

/* exact distance from p to a planar convex quad (corners q[0..3] in order, unit normal n, offset h) */
static real quad_dist(const real p[3], const real q[4][3], const real n[3], real h)
{
    real dist = n[0] * p[0] + n[1] * p[1] + n[2] * p[2] - h;
    real f[3] = { p[0] - dist * n[0], p[1] - dist * n[1], p[2] - dist * n[2] };
    /* foot inside the quad <=> same side of all four edges */
    int pos = 0, neg = 0;
    for (int i = 0; i < 4; ++i) {
        int j = (i + 1) & 3;
        real e[3] = { q[j][0] - q[i][0], q[j][1] - q[i][1], q[j][2] - q[i][2] };
        real w[3] = { f[0] - q[i][0], f[1] - q[i][1], f[2] - q[i][2] };
        real c[3] = { e[1] * w[2] - e[2] * w[1], e[2] * w[0] - e[0] * w[2], e[0] * w[1] - e[1] * w[0] };
        real sgn = c[0] * n[0] + c[1] * n[1] + c[2] * n[2];
        if (sgn > 0) pos++;
        if (sgn < 0) neg++;
    }
    if (pos == 0 || neg == 0) return R_FABS(dist);
    real best = ORC_INF;
    for (int i = 0; i < 4; ++i) best = rmin2(best, seg3_d2(p, q[i], q[(i + 1) & 3]));
    return R_SQRT(best);
}

static real sdf_trd(const orc_shape *s, real x, real y, real z)
{
    real p[3] = { x, y, z };
    real g = -ORC_INF;
    for (int j = 0; j < 6; ++j)
        g = rmax2(g, s->pn[j][0] * x + s->pn[j][1] * y + s->pn[j][2] * z - s->ph[j]);
    if (g <= 0) return g; /* exact inside a convex polyhedron */
    real best = ORC_INF;
    for (int j = 0; j < 6; ++j) best = rmin2(best, quad_dist(p, s->fv[j], s->pn[j], s->ph[j]));
    return best;
}

/* -------------------------------------------------------------- sdf (c.3) */

static real sdf(const orc_shape *s, real x, real y, real z)
{
    switch (s->kind) {
    case ORC_BOX: {
        real qx = R_FABS(x) - s->h[0], qy = R_FABS(y) - s->h[1], qz = R_FABS(z) - s->h[2];
        real ax = rmax2(qx, 0), ay = rmax2(qy, 0), az = rmax2(qz, 0);
        return R_SQRT(ax * ax + ay * ay + az * az) + rmin2(rmax2(qx, rmax2(qy, qz)), 0);
    }
    case ORC_ORB:
        return R_SQRT(x * x + y * y + z * z) - s->r;
    case ORC_TRD:
        return sdf_trd(s, x, y, z);
    default:
        return sdf_rz(s, x, y, z);
    }
}

/* c.2: Inside */
static int inside(const orc_shape *s, real x, real y, real z)
{
    real d = sdf(s, x, y, z);
    if (d < -ORC_KTOL) return ORC_INSIDE;
    if (d > ORC_KTOL) return ORC_OUTSIDE;
    return ORC_SURFACE;
}

/* ------------------------------------------------- first crossing (c.4) */

/* a t^2 + 2 b t + c = 0; D = b^2 - a c; D <= 0 => no crossing (reading R8) */
static int quad_roots(real a, real b, real c, real t[2])
{
    real D = b * b - a * c;
    if (!(D > 0)) return 0;
    real sq = R_SQRT(D);
    real q = (b >= 0) ? -(b + sq) : -(b - sq); /* sgn(0) = +1, reading R9 */
    int n = 0;
    if (a != 0) t[n++] = q / a;
    if (q != 0) t[n++] = c / q;
    return n;
}

static real cross_box(const orc_shape *s, int is_inside, const real p[3], const real d[3])
{
    real tin = -ORC_INF, tout = ORC_INF;
    for (int i = 0; i < 3; ++i) {
        real h = s->h[i];
        if (d[i] != 0) {
            real sg = d[i] > 0 ? 1 : -1;
            real t1 = (-sg * h - p[i]) / d[i];
            real t2 = (sg * h - p[i]) / d[i];
            tin = rmax2(tin, t1);
            tout = rmin2(tout, t2);
        } else if (R_FABS(p[i]) >= h) {
            return ORC_INF;
        }
    }
    if (is_inside) return tout;
    return (tin < tout && tout > 0) ? tin : ORC_INF;
}

static real cross_convex(const orc_shape *s, int is_inside, const real p[3], const real d[3])
{
    real tin = -ORC_INF, tout = ORC_INF;
    for (int j = 0; j < 6; ++j) {
        real num = s->ph[j] - (s->pn[j][0] * p[0] + s->pn[j][1] * p[1] + s->pn[j][2] * p[2]);
        real den = s->pn[j][0] * d[0] + s->pn[j][1] * d[1] + s->pn[j][2] * d[2];
        if (den > 0) tout = rmin2(tout, num / den);
        else if (den < 0) tin = rmax2(tin, num / den);
        else if (num < 0) return ORC_INF;
    }
    if (is_inside) return tout;
    return (tin < tout && tout > 0) ? tin : ORC_INF;
}

static real cross_orb(const orc_shape *s, const real p[3], const real d[3])
{
    real t[2], best = ORC_INF;
    real b = p[0] * d[0] + p[1] * d[1] + p[2] * d[2];
    real c = p[0] * p[0] + p[1] * p[1] + p[2] * p[2] - s->r * s->r;
    int n = quad_roots(1, b, c, t);
    for (int i = 0; i < n; ++i)
        if (t[i] > 0) best = rmin2(best, t[i]);
    return best;
}

static real cross_rz(const orc_shape *s, const real p[3], const real d[3])
{
    real best = ORC_INF;
    real x = p[0], y = p[1], z = p[2], dx = d[0], dy = d[1], dz = d[2];
    for (int i = 0; i < s->nv; ++i) {
        if (edge_on_axis(s, i)) continue;
        int j = (i + 1) % s->nv;
        real r0 = s->pr[i], z0 = s->pz[i], r1 = s->pr[j], z1 = s->pz[j];
        if (z0 != z1) { /* frustum (cylinder if r0 == r1) */
            real B = (r1 - r0) / (z1 - z0), A = r0 - B * z0, k = A + B * z;
            real a = dx * dx + dy * dy - B * B * dz * dz;
            real b = x * dx + y * dy - B * dz * k;
            real c = x * x + y * y - k * k;
            real t[2];
            int n = quad_roots(a, b, c, t);
            for (int m = 0; m < n; ++m) {
                if (!(t[m] > 0)) continue;
                real zh = z + t[m] * dz;
                if (zh < rmin2(z0, z1) || zh > rmax2(z0, z1)) continue;
                if (!in_phi(s, x + t[m] * dx, y + t[m] * dy)) continue;
                best = rmin2(best, t[m]);
            }
        } else if (dz != 0) { /* cap annulus */
            real t = (z0 - z) / dz;
            if (!(t > 0)) continue;
            real hx = x + t * dx, hy = y + t * dy, rh2 = hx * hx + hy * hy;
            real rlo = rmin2(r0, r1), rhi = rmax2(r0, r1);
            if (rh2 < rlo * rlo || rh2 > rhi * rhi) continue;
            if (!in_phi(s, hx, hy)) continue;
            best = rmin2(best, t);
        }
    }
    if (!s->full) {
        for (int k = 0; k < 2; ++k) {
            real ex = s->e[k][0], ey = s->e[k][1];
            real nx = -ey, ny = ex;
            real nd = nx * dx + ny * dy;
            if (nd == 0) continue;
            real t = -(nx * x + ny * y) / nd;
            if (!(t > 0)) continue;
            real hx = x + t * dx, hy = y + t * dy;
            if (!in_poly(s, ex * hx + ey * hy, z + t * dz)) continue;
            best = rmin2(best, t);
        }
    }
    return best;
}

static real cross(const orc_shape *s, int is_inside, const real p[3], const real d[3])
{
    switch (s->kind) {
    case ORC_BOX: return cross_box(s, is_inside, p, d);
    case ORC_ORB: return cross_orb(s, p, d);
    case ORC_TRD: return cross_convex(s, is_inside, p, d);
    default: return cross_rz(s, p, d);
    }
}

/*
 * Reading R32 (SURVEY.md 8(c) R7 left start points in the surface band undefined; 8(f) f2 asks for them): a particle
 * whose geometric step won "is transported to the border" and starts its next step ON a surface.
 *   For a start point of class SURFACE the ray is read as starting on the crossing it sits on: let t_0 < t_1 < ... be
 *   ALL crossings of the whole line p + t d, t in (-inf, +inf), by the boundary (c.4 without the t > 0 filter, see
 *   line_crossings below); the solid is bounded, so along the line the even-numbered crossings enter it and the
 *   odd-numbered leave it.  Let t_s be the crossing nearest to t = 0 (the later one on a tie).
 *     DistanceToIn  = max(t_s, 0) if t_s is entering, else max(t_{s+1}, 0) (the next entry; +inf if there is none);
 *     DistanceToOut = max(t_s, 0) if t_s is leaving,  else max(t_{s+1}, 0) (the exit that follows the entry at t_s).
 *   A line that does not cross the boundary at all (a tangent start in the band): DistanceToIn = +inf, DistanceToOut = 0.
 * So a surface point moving inward has DistanceToIn 0 and DistanceToOut = its chord; moving outward DistanceToOut 0 and
 * DistanceToIn = the next entry.  For start points outside the band nothing changes (c.2).
 */
static int line_crossings(const orc_shape *s, const real p[3], const real d[3], real *out);

static real surface_cross(const orc_shape *s, const real p[3], const real d[3], int want_leaving)
{
    real t[4 * ORC_MAXV + 8];
    int n = line_crossings(s, p, d, t); /* t[0], t[2], ... enter, t[1], t[3], ... leave */
    if (n == 0) return want_leaving ? (real)0 : ORC_INF;
    int k = 0;
    for (int i = 1; i < n; ++i)
        if (R_FABS(t[i]) <= R_FABS(t[k])) k = i;
    int leaving = k & 1;
    if (leaving != want_leaving) ++k; /* the next crossing has the wanted sense */
    if (k >= n) return ORC_INF;
    return rmax2(t[k], 0);
}

/* c.2: DistanceToIn / DistanceToOut (readings R4, R5; R32 in the surface band) */
static real distance_to_in(const orc_shape *s, const real p[3], const real d[3], real step_max)
{
    int cls = inside(s, p[0], p[1], p[2]);
    if (cls == ORC_INSIDE) return -1;
    real t = cls == ORC_SURFACE ? surface_cross(s, p, d, 0) : cross(s, 0, p, d);
    return t <= step_max ? t : ORC_INF;
}

static real distance_to_out(const orc_shape *s, const real p[3], const real d[3], real step_max)
{
    int cls = inside(s, p[0], p[1], p[2]);
    if (cls == ORC_OUTSIDE) return -1;
    real t = cls == ORC_SURFACE ? surface_cross(s, p, d, 1) : cross(s, 1, p, d);
    return t <= step_max ? t : ORC_INF;
}

/* ------------------------------------------------------------ batch entry */

double orc_ktol(void) { return 1e-9; }

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

void orc_sdf(const orc_shape *s, const double *x, const double *y, const double *z, int64_t n, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) out[i] = (double)sdf(s, x[i], y[i], z[i]);
}

void orc_inside(const orc_shape *s, const double *x, const double *y, const double *z, int64_t n, int32_t *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) out[i] = inside(s, x[i], y[i], z[i]);
}

/* c.2: SafetyToIn = +sdf, SafetyToOut = -sdf; exact and signed (readings R2, R3) */
void orc_safety_to_in(const orc_shape *s, const double *x, const double *y, const double *z, int64_t n, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) out[i] = (double)sdf(s, x[i], y[i], z[i]);
}

void orc_safety_to_out(const orc_shape *s, const double *x, const double *y, const double *z, int64_t n, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) out[i] = (double)(-sdf(s, x[i], y[i], z[i]));
}

void orc_distance_to_in(const orc_shape *s, const double *x, const double *y, const double *z, const double *dx,
                        const double *dy, const double *dz, double step_max, int64_t n, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        real p[3] = { x[i], y[i], z[i] }, d[3] = { dx[i], dy[i], dz[i] };
        out[i] = (double)distance_to_in(s, p, d, step_max);
    }
}

void orc_distance_to_out(const orc_shape *s, const double *x, const double *y, const double *z, const double *dx,
                         const double *dy, const double *dz, double step_max, int64_t n, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        real p[3] = { x[i], y[i], z[i] }, d[3] = { dx[i], dy[i], dz[i] };
        out[i] = (double)distance_to_out(s, p, d, step_max);
    }
}

/* the raw first crossing Cross(p, d) of c.2, exposed for the pins */
void orc_cross(const orc_shape *s, const double *x, const double *y, const double *z, const double *dx,
               const double *dy, const double *dz, int64_t n, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        real p[3] = { x[i], y[i], z[i] }, d[3] = { dx[i], dy[i], dz[i] };
        int in = inside(s, p[0], p[1], p[2]) != ORC_OUTSIDE;
        out[i] = (double)cross(s, in, p, d);
    }
}

/* ---------------------------------------------------------- navigation */

orc_volume *orc_volume_create(const orc_shape *mother, int nd, const orc_shape *const *daughters, const double *xf)
{
    if (!mother || nd < 0 || (nd > 0 && (!daughters || !xf))) return NULL;
    orc_volume *v = (orc_volume *)calloc(1, sizeof *v);
    if (!v) return NULL;
    v->mother = mother;
    v->nd = nd;
    v->daughter = (const orc_shape **)calloc((size_t)(nd > 0 ? nd : 1), sizeof *v->daughter);
    v->xf = (real *)calloc((size_t)(nd > 0 ? nd : 1) * 12, sizeof *v->xf);
    for (int i = 0; i < nd; ++i) {
        v->daughter[i] = daughters[i];
        for (int k = 0; k < 12; ++k) v->xf[12 * i + k] = xf[12 * i + k];
    }
    return v;
}

void orc_volume_destroy(orc_volume *v)
{
    if (!v) return;
    free((void *)v->daughter);
    free(v->xf);
    free(v);
}

static void to_local(const real *m, const real p[3], const real d[3], real pl[3], real dl[3])
{
    /* reading R12: p_loc = R p + b, d_loc = R d, row-major [R | b] */
    for (int r = 0; r < 3; ++r) {
        pl[r] = m[4 * r + 0] * p[0] + m[4 * r + 1] * p[1] + m[4 * r + 2] * p[2] + m[4 * r + 3];
        dl[r] = m[4 * r + 0] * d[0] + m[4 * r + 1] * d[1] + m[4 * r + 2] * d[2];
    }
}

/* c.2 ComputeStep; tie-break reading R13; (stepMax, -2) when the physics step wins */
void orc_compute_step(const orc_volume *v, const double *x, const double *y, const double *z, const double *dx,
                      const double *dy, const double *dz, double step_max, int64_t n, double *step, int32_t *hit)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        real p[3] = { x[i], y[i], z[i] }, d[3] = { dx[i], dy[i], dz[i] };
        real best = distance_to_out(v->mother, p, d, ORC_INF);
        int32_t who = -1;
        for (int k = 0; k < v->nd; ++k) {
            real pl[3], dl[3];
            to_local(v->xf + 12 * k, p, d, pl, dl);
            real t = distance_to_in(v->daughter[k], pl, dl, ORC_INF);
            if (t >= 0 && t < best) { best = t; who = k; }
        }
        if (best > step_max) { best = step_max; who = -2; }
        step[i] = (double)best;
        hit[i] = who;
    }
}

/*
 * Isotropic safety of the navigation state (widening of PAPER.md:113 to the
 * placed-volume level): min( SafetyToOut_mother(p), min_i SafetyToIn_i(R_i p + b_i) ).
 * Positive for a point inside the mother and outside every daughter.
 */
void orc_volume_safety(const orc_volume *v, const double *x, const double *y, const double *z, int64_t n, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        real p[3] = { x[i], y[i], z[i] }, d0[3] = { 0, 0, 0 };
        real best = -sdf(v->mother, p[0], p[1], p[2]);
        for (int k = 0; k < v->nd; ++k) {
            real pl[3], dl[3];
            to_local(v->xf + 12 * k, p, d0, pl, dl);
            best = rmin2(best, sdf(v->daughter[k], pl[0], pl[1], pl[2]));
        }
        out[i] = (double)best;
    }
}

/* ------------------------------------------------- hierarchy of volumes */
/*
 * Widening SURVEY.md 8(f) f3: "with hierarchical connections one can build
 * the whole detector"; a particle whose geometric step wins
 * "is transported to the border" and changes volume.  The paper
 * gives no data structure or algorithm; readings R22-R25 of DESIGN.md:
 *   R22  a world is a tree of placed solids ("nodes"): node 0 is the root,
 *        parent[i] < i, xf[i] = row-major 3x4 [R | b] from the PARENT's local
 *        frame to node i's local frame (for the root: from the world frame);
 *        the children of a node are the nodes naming it as parent, in index
 *        order; siblings do not overlap and lie inside their parent.
 *   R23  Locate(p): -1 if p is not strictly inside the root (Inside != INSIDE);
 *        else descend from the root: the first child (index order) that holds
 *        p strictly inside becomes the current node; stop when no child does.
 *   R24  Step(node, p, d): p, d given in the WORLD frame and mapped down the
 *        chain root -> node one transform at a time; the one-level ComputeStep
 *        of c.2 in that node (its solid as mother, its children as daughters,
 *        R13 tie-break); `next` is the child entered, the parent (-1 above the
 *        root) when the node's own exit wins, the node itself when step_max
 *        wins (the physics step is shorter).
 *   R25  Safety(node, p): min(SafetyToOut_node, SafetyToIn of every child),
 *        i.e. orc_volume_safety in that node.
 */

/* boolean solids are defined further down (R27-R29); a node may be one (R30: a node is any solid of this file, a
 * primitive, a polycone or a boolean; with a boolean among a node and its children the node's safety inherits R29's
 * "never over-estimates" in place of "exact") */
typedef struct orc_boolean_s orc_boolean;
static int bool_inside(const orc_boolean *c, const real p[3]);
static real bool_sdf(const orc_boolean *c, const real p[3]);
static real bool_cross(const orc_boolean *c, int cls, int want_leaving, const real p[3], const real d[3]);

typedef struct {
    int nn;
    const orc_shape **shape;     /* NULL where the node is a boolean */
    const orc_boolean **boolean; /* NULL where the node is a plain solid */
    int32_t *parent;
    real *xf; /* nn * 12 */
} orc_world;

static int node_inside(const orc_world *w, int i, const real p[3])
{
    return w->boolean[i] ? bool_inside(w->boolean[i], p) : inside(w->shape[i], p[0], p[1], p[2]);
}

static real node_sdf(const orc_world *w, int i, const real p[3])
{
    return w->boolean[i] ? bool_sdf(w->boolean[i], p) : sdf(w->shape[i], p[0], p[1], p[2]);
}

static real node_distance_to_in(const orc_world *w, int i, const real p[3], const real d[3])
{
    if (!w->boolean[i]) return distance_to_in(w->shape[i], p, d, ORC_INF);
    int cls = bool_inside(w->boolean[i], p);
    return cls == ORC_INSIDE ? (real)-1 : bool_cross(w->boolean[i], cls, 0, p, d);
}

static real node_distance_to_out(const orc_world *w, int i, const real p[3], const real d[3])
{
    if (!w->boolean[i]) return distance_to_out(w->shape[i], p, d, ORC_INF);
    int cls = bool_inside(w->boolean[i], p);
    return cls == ORC_OUTSIDE ? (real)-1 : bool_cross(w->boolean[i], cls, 1, p, d);
}

/* exactly one of shapes[i], booleans[i] is given per node (booleans may be NULL: no boolean nodes) */
orc_world *orc_world_create_mixed(int nn, const orc_shape *const *shapes, const orc_boolean *const *booleans,
                                  const int32_t *parent, const double *xf)
{
    if (nn < 1 || !shapes || !parent || !xf || parent[0] != -1) return NULL;
    for (int i = 0; i < nn; ++i) {
        int nb = booleans && booleans[i];
        if ((shapes[i] != NULL) == nb) return NULL;
        if (i > 0 && (parent[i] < 0 || parent[i] >= i)) return NULL;
    }
    if (!finite_all(xf, 12 * nn)) return NULL;
    orc_world *w = (orc_world *)calloc(1, sizeof *w);
    if (!w) return NULL;
    w->nn = nn;
    w->shape = (const orc_shape **)calloc((size_t)nn, sizeof *w->shape);
    w->boolean = (const orc_boolean **)calloc((size_t)nn, sizeof *w->boolean);
    w->parent = (int32_t *)calloc((size_t)nn, sizeof *w->parent);
    w->xf = (real *)calloc((size_t)nn * 12, sizeof *w->xf);
    for (int i = 0; i < nn; ++i) {
        w->shape[i] = shapes[i];
        w->boolean[i] = booleans ? booleans[i] : NULL;
        w->parent[i] = parent[i];
        for (int k = 0; k < 12; ++k) w->xf[12 * i + k] = xf[12 * i + k];
    }
    return w;
}

orc_world *orc_world_create(int nn, const orc_shape *const *shapes, const int32_t *parent, const double *xf)
{
    return orc_world_create_mixed(nn, shapes, NULL, parent, xf);
}

void orc_world_destroy(orc_world *w)
{
    if (!w) return;
    free((void *)w->shape);
    free((void *)w->boolean);
    free(w->parent);
    free(w->xf);
    free(w);
}

/* world frame -> local frame of `node`, one transform at a time from the root down (R24) */
static void world_to_node(const orc_world *w, int node, const real p[3], const real d[3], real pl[3], real dl[3])
{
    real pp[3], dp[3];
    if (w->parent[node] >= 0) world_to_node(w, w->parent[node], p, d, pp, dp);
    else { for (int k = 0; k < 3; ++k) { pp[k] = p[k]; dp[k] = d[k]; } }
    to_local(w->xf + 12 * node, pp, dp, pl, dl);
}

/* R23 */
void orc_world_locate(const orc_world *w, const double *x, const double *y, const double *z, int64_t n, int32_t *node)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        real p[3] = { x[i], y[i], z[i] }, d0[3] = { 0, 0, 0 }, pl[3], dl[3];
        to_local(w->xf, p, d0, pl, dl);
        if (node_inside(w, 0, pl) != ORC_INSIDE) { node[i] = -1; continue; }
        int cur = 0, moved = 1;
        while (moved) {
            moved = 0;
            for (int c = cur + 1; c < w->nn; ++c) {
                if (w->parent[c] != cur) continue;
                real pc[3];
                to_local(w->xf + 12 * c, pl, d0, pc, dl);
                if (node_inside(w, c, pc) == ORC_INSIDE) {
                    cur = c;
                    pl[0] = pc[0]; pl[1] = pc[1]; pl[2] = pc[2];
                    moved = 1;
                    break;
                }
            }
        }
        node[i] = cur;
    }
}

/* R24 */
void orc_world_step(const orc_world *w, const int32_t *node, const double *x, const double *y, const double *z,
                    const double *dx, const double *dy, const double *dz, double step_max, int64_t n, double *step,
                    int32_t *next)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        int nd = node[i];
        if (nd < 0 || nd >= w->nn) { step[i] = -1; next[i] = -1; continue; }
        real p[3] = { x[i], y[i], z[i] }, d[3] = { dx[i], dy[i], dz[i] }, pl[3], dl[3];
        world_to_node(w, nd, p, d, pl, dl);
        real best = node_distance_to_out(w, nd, pl, dl);
        int32_t who = w->parent[nd];
        for (int c = nd + 1; c < w->nn; ++c) {
            if (w->parent[c] != nd) continue;
            real pc[3], dc[3];
            to_local(w->xf + 12 * c, pl, dl, pc, dc);
            real t = node_distance_to_in(w, c, pc, dc);
            if (t >= 0 && t < best) { best = t; who = c; }
        }
        if (best > step_max) { best = step_max; who = nd; }
        step[i] = (double)best;
        next[i] = who;
    }
}

/* R25 */
void orc_world_safety(const orc_world *w, const int32_t *node, const double *x, const double *y, const double *z,
                      int64_t n, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        int nd = node[i];
        if (nd < 0 || nd >= w->nn) { out[i] = -1; continue; }
        real p[3] = { x[i], y[i], z[i] }, d0[3] = { 0, 0, 0 }, pl[3], dl[3];
        world_to_node(w, nd, p, d0, pl, dl);
        real best = -node_sdf(w, nd, pl);
        for (int c = nd + 1; c < w->nn; ++c) {
            if (w->parent[c] != nd) continue;
            real pc[3];
            to_local(w->xf + 12 * c, pl, d0, pc, dl);
            best = rmin2(best, node_sdf(w, c, pc));
        }
        out[i] = (double)best;
    }
}

/* ------------------------------------------------------- boolean solids */
/*
 * Widening SURVEY.md 8(f) f2: the paper's geometry holds "rotations, translations, logical operations, and distance
 * calculations" and builds solids by "boolean operations"; it defines none of them.
 * Readings R27-R29 of DESIGN.md:
 *   R27  C = A op B, op in {union, intersection, subtraction (A minus B)}; A, B primitive solids, A in the frame of
 *        C, B placed by a row-major 3x4 [R | b] from the frame of C to the frame of B.  Membership is the set
 *        operation on the closed sets.  Inside(p) combines the two classes: union: INSIDE if either is INSIDE,
 *        OUTSIDE if both are OUTSIDE; intersection: INSIDE if both, OUTSIDE if either is OUTSIDE; subtraction:
 *        INSIDE if A INSIDE and B OUTSIDE, OUTSIDE if A OUTSIDE or B INSIDE; SURFACE otherwise.
 *   R28  Distances: along the WHOLE line each solid is a union of intervals bounded by its crossings (ALL crossings of
 *        c.4, not only the first, t of either sign); C's membership along the line is the set operation on the two
 *        interval sets (outside both far behind the start point); DistanceToIn / DistanceToOut is the first t > 0 at
 *        which C's membership flips, +inf if it never does; -1 on the wrong side as R4; R32 for a start of class SURFACE.
 *   R29  Safeties: the usual composition sdf_C = min(sdfA, sdfB) / max(sdfA, sdfB) / max(sdfA, -sdfB).  This is
 *        NOT the exact distance of R2: it never over-estimates the distance to the surface of C, is exact where
 *        only one operand matters, and has the sign of the membership (pinned as such).
 */

enum { ORC_UNION = 0, ORC_INTERSECTION = 1, ORC_SUBTRACTION = 2 };

/* R31: an operand may itself be a boolean (a CSG tree); R27-R29 apply unchanged with "operand" read recursively: the
 * class, the composed sdf and the membership intervals of an operand that is a boolean are those of that boolean.
 * At most ORC_MAXLEAF primitives per tree. */
#define ORC_MAXLEAF 8

struct orc_boolean_s {
    int op;
    const orc_shape *a, *b;    /* operand is a primitive ... */
    const orc_boolean *ca, *cb; /* ... or a boolean: exactly one of (a, ca) and one of (b, cb) is given */
    int nleaf;
    real xf[12];
};

orc_boolean *orc_boolean_create_nested(int op, const orc_shape *a, const orc_boolean *ca, const orc_shape *b,
                                       const orc_boolean *cb, const double *xf)
{
    if (op < 0 || op > 2 || ((a != NULL) == (ca != NULL)) || ((b != NULL) == (cb != NULL)) || !xf || !finite_all(xf, 12)) return NULL;
    int nleaf = (a ? 1 : ca->nleaf) + (b ? 1 : cb->nleaf);
    if (nleaf > ORC_MAXLEAF) return NULL;
    orc_boolean *c = (orc_boolean *)calloc(1, sizeof *c);
    if (!c) return NULL;
    c->op = op;
    c->a = a;
    c->b = b;
    c->ca = ca;
    c->cb = cb;
    c->nleaf = nleaf;
    for (int k = 0; k < 12; ++k) c->xf[k] = xf[k];
    return c;
}

orc_boolean *orc_boolean_create(int op, const orc_shape *a, const orc_shape *b, const double *xf)
{
    return orc_boolean_create_nested(op, a, NULL, b, NULL, xf);
}

void orc_boolean_destroy(orc_boolean *c) { free(c); }

#define ORC_MAXX (4 * ORC_MAXV + 8)

/* every crossing of the boundary of one solid by the ray, ascending (c.4 with "collect" in place of "min"):
 * whole = 0: the crossings t > 0; whole = 1: those of the whole line, t of either sign (R32, R28) */
static int crossings(const orc_shape *s, const real p[3], const real d[3], real *out, int whole)
{
    int n = 0;
    if (s->kind == ORC_BOX || s->kind == ORC_TRD) { /* convex: the interval [tin, tout] of the clip */
        real tin = -ORC_INF, tout = ORC_INF;
        if (s->kind == ORC_BOX) {
            for (int i = 0; i < 3; ++i) {
                real h = s->h[i];
                if (d[i] != 0) {
                    real sg = d[i] > 0 ? 1 : -1;
                    tin = rmax2(tin, (-sg * h - p[i]) / d[i]);
                    tout = rmin2(tout, (sg * h - p[i]) / d[i]);
                } else if (R_FABS(p[i]) >= h) {
                    return 0;
                }
            }
        } else {
            for (int j = 0; j < 6; ++j) {
                real num = s->ph[j] - (s->pn[j][0] * p[0] + s->pn[j][1] * p[1] + s->pn[j][2] * p[2]);
                real den = s->pn[j][0] * d[0] + s->pn[j][1] * d[1] + s->pn[j][2] * d[2];
                if (den > 0) tout = rmin2(tout, num / den);
                else if (den < 0) tin = rmax2(tin, num / den);
                else if (num < 0) return 0;
            }
        }
        if (!(tin < tout)) return 0;
        if (whole || tin > 0) out[n++] = tin;
        if (whole || tout > 0) out[n++] = tout;
        return n;
    }
    if (s->kind == ORC_ORB) {
        real t[2];
        real b = p[0] * d[0] + p[1] * d[1] + p[2] * d[2];
        real c = p[0] * p[0] + p[1] * p[1] + p[2] * p[2] - s->r * s->r;
        int m = quad_roots(1, b, c, t);
        for (int i = 0; i < m; ++i)
            if (whole || t[i] > 0) out[n++] = t[i];
    } else { /* RZ polygon + phi wedge: the candidate loops of cross_rz */
        real x = p[0], y = p[1], z = p[2], dx = d[0], dy = d[1], dz = d[2];
        for (int i = 0; i < s->nv; ++i) {
            if (edge_on_axis(s, i)) continue;
            int j = (i + 1) % s->nv;
            real r0 = s->pr[i], z0 = s->pz[i], r1 = s->pr[j], z1 = s->pz[j];
            if (z0 != z1) {
                real B = (r1 - r0) / (z1 - z0), A = r0 - B * z0, k = A + B * z;
                real t[2];
                int m = quad_roots(dx * dx + dy * dy - B * B * dz * dz, x * dx + y * dy - B * dz * k, x * x + y * y - k * k, t);
                for (int q = 0; q < m; ++q) {
                    if (!whole && !(t[q] > 0)) continue;
                    real zh = z + t[q] * dz;
                    if (zh < rmin2(z0, z1) || zh > rmax2(z0, z1)) continue;
                    if (!in_phi(s, x + t[q] * dx, y + t[q] * dy)) continue;
                    out[n++] = t[q];
                }
            } else if (dz != 0) {
                real t = (z0 - z) / dz;
                if (!whole && !(t > 0)) continue;
                real hx = x + t * dx, hy = y + t * dy, rh2 = hx * hx + hy * hy;
                real rlo = rmin2(r0, r1), rhi = rmax2(r0, r1);
                if (rh2 < rlo * rlo || rh2 > rhi * rhi) continue;
                if (!in_phi(s, hx, hy)) continue;
                out[n++] = t;
            }
        }
        if (!s->full) {
            for (int k = 0; k < 2; ++k) {
                real ex = s->e[k][0], ey = s->e[k][1], nx = -ey, ny = ex;
                real nd = nx * dx + ny * dy;
                if (nd == 0) continue;
                real t = -(nx * x + ny * y) / nd;
                if (!whole && !(t > 0)) continue;
                real hx = x + t * dx, hy = y + t * dy;
                if (!in_poly(s, ex * hx + ey * hy, z + t * dz)) continue;
                out[n++] = t;
            }
        }
    }
    for (int i = 1; i < n; ++i) { /* insertion sort */
        real v = out[i];
        int j = i - 1;
        while (j >= 0 && out[j] > v) { out[j + 1] = out[j]; --j; }
        out[j + 1] = v;
    }
    return n;
}

static int all_crossings(const orc_shape *s, const real p[3], const real d[3], real *out) { return crossings(s, p, d, out, 0); }

/* The crossings of the WHOLE line at which the membership of the solid really flips, ascending (R32, R28).  The patch
 * loops above deliver every intersection with a boundary patch; a line through an edge of the solid meets two patches
 * at one point, and one that clips an edge by less than the tolerance meets them within kTol of each other, so raw
 * values within kTol of the first of their cluster are ONE candidate.  A candidate is a crossing iff the sign of the
 * exact sdf differs between the midpoints of the gaps before and after it (outside before the first candidate and
 * after the last: the solid is bounded).  So out[0], out[2], ... enter the solid and out[1], out[3], ... leave it. */
static int line_crossings(const orc_shape *s, const real p[3], const real d[3], real *out)
{
    real raw[ORC_MAXX], c[ORC_MAXX];
    int n = crossings(s, p, d, raw, 1), m = 0, k = 0;
    for (int i = 0; i < n; ++i)
        if (m == 0 || raw[i] - c[m - 1] > ORC_KTOL) c[m++] = raw[i];
    int prev_in = 0;
    for (int j = 0; j < m; ++j) {
        int next_in = 0;
        if (j + 1 < m) {
            real tm = (c[j] + c[j + 1]) / 2;
            next_in = sdf(s, p[0] + tm * d[0], p[1] + tm * d[1], p[2] + tm * d[2]) < 0;
        }
        if (next_in != prev_in) out[k++] = c[j];
        prev_in = next_in;
    }
    return k;
}

static int bool_member(int op, int ina, int inb)
{
    if (op == ORC_UNION) return ina || inb;
    if (op == ORC_INTERSECTION) return ina && inb;
    return ina && !inb;
}

/* an operand's answers: the primitive's, or (R31) the nested boolean's */
static int operand_inside(const orc_shape *s, const orc_boolean *c, const real p[3])
{
    return s ? inside(s, p[0], p[1], p[2]) : bool_inside(c, p);
}

static real operand_sdf(const orc_shape *s, const orc_boolean *c, const real p[3])
{
    return s ? sdf(s, p[0], p[1], p[2]) : bool_sdf(c, p);
}

static int bool_events(const orc_boolean *c, const real p[3], const real d[3], real *out);

/* every t (either sign) at which the operand's membership flips along the whole line, ascending */
static int operand_events(const orc_shape *s, const orc_boolean *c, const real p[3], const real d[3], real *out)
{
    return s ? line_crossings(s, p, d, out) : bool_events(c, p, d, out);
}

/* R27 */
static int bool_inside(const orc_boolean *c, const real p[3])
{
    real d0[3] = { 0, 0, 0 }, pb[3], db[3];
    to_local(c->xf, p, d0, pb, db);
    int ca = operand_inside(c->a, c->ca, p), cb = operand_inside(c->b, c->cb, pb);
    int ain = ca == ORC_INSIDE, aout = ca == ORC_OUTSIDE, bin = cb == ORC_INSIDE, bout = cb == ORC_OUTSIDE;
    int in, out;
    if (c->op == ORC_UNION) { in = ain || bin; out = aout && bout; }
    else if (c->op == ORC_INTERSECTION) { in = ain && bin; out = aout || bout; }
    else { in = ain && bout; out = aout || bin; }
    return in ? ORC_INSIDE : (out ? ORC_OUTSIDE : ORC_SURFACE);
}

/* R29 */
static real bool_sdf(const orc_boolean *c, const real p[3])
{
    real d0[3] = { 0, 0, 0 }, pb[3], db[3];
    to_local(c->xf, p, d0, pb, db);
    real sa = operand_sdf(c->a, c->ca, p), sb = operand_sdf(c->b, c->cb, pb);
    if (c->op == ORC_UNION) return rmin2(sa, sb);
    if (c->op == ORC_INTERSECTION) return rmax2(sa, sb);
    return rmax2(sa, -sb);
}

/* R28: every t, of either sign, at which the membership of C along the WHOLE line flips, ascending: the merge of the
 * operands' flips (a tie goes to A).  Both operands are bounded, so far behind the start point the line is outside
 * both and the memberships are counted on from there; no class of the start point enters (a start point in the
 * surface band of an operand would make that class ambiguous). */
static int bool_events(const orc_boolean *c, const real p[3], const real d[3], real *out)
{
    real pb[3], db[3];
    real *ta = (real *)malloc(sizeof(real) * 2 * ORC_MAXLEAF * ORC_MAXX), *tb = ta + ORC_MAXLEAF * ORC_MAXX;
    to_local(c->xf, p, d, pb, db);
    int na = operand_events(c->a, c->ca, p, d, ta), nb = operand_events(c->b, c->cb, pb, db, tb);
    int ina = 0, inb = 0, cur = 0;
    int i = 0, j = 0, n = 0;
    while (i < na || j < nb) {
        real t;
        if (j >= nb || (i < na && ta[i] <= tb[j])) { t = ta[i++]; ina = !ina; }
        else { t = tb[j++]; inb = !inb; }
        int now = bool_member(c->op, ina, inb);
        if (now != cur) { out[n++] = t; cur = now; }
    }
    free(ta);
    return n;
}

/* R28: the first flip ahead of a start point of class INSIDE or OUTSIDE; R32 (read with "crossing" = flip of C's
 * membership) for a start point of class SURFACE: want_leaving = 0 DistanceToIn, 1 DistanceToOut */
static real bool_cross(const orc_boolean *c, int cls, int want_leaving, const real p[3], const real d[3])
{
    real *t = (real *)malloc(sizeof(real) * ORC_MAXLEAF * ORC_MAXX);
    int n = bool_events(c, p, d, t);
    real r = ORC_INF;
    if (cls != ORC_SURFACE) {
        for (int i = 0; i < n; ++i)
            if (t[i] > 0) { r = t[i]; break; }
    } else if (n == 0) {
        r = want_leaving ? (real)0 : ORC_INF;
    } else {
        int k = 0;
        for (int i = 1; i < n; ++i)
            if (R_FABS(t[i]) <= R_FABS(t[k])) k = i;
        if ((k & 1) != want_leaving) ++k;
        if (k < n) r = rmax2(t[k], 0);
    }
    free(t);
    return r;
}

void orc_boolean_inside(const orc_boolean *c, const double *x, const double *y, const double *z, int64_t n, int32_t *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        real p[3] = { x[i], y[i], z[i] };
        out[i] = bool_inside(c, p);
    }
}

void orc_boolean_sdf(const orc_boolean *c, const double *x, const double *y, const double *z, int64_t n, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        real p[3] = { x[i], y[i], z[i] };
        out[i] = (double)bool_sdf(c, p);
    }
}

/* which = 0: DistanceToIn, 1: DistanceToOut (R4, R5 as for the primitives) */
void orc_boolean_distance(const orc_boolean *c, int which, const double *x, const double *y, const double *z,
                          const double *dx, const double *dy, const double *dz, double step_max, int64_t n, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        real p[3] = { x[i], y[i], z[i] }, d[3] = { dx[i], dy[i], dz[i] };
        int cls = bool_inside(c, p);
        if ((which == 0 && cls == ORC_INSIDE) || (which == 1 && cls == ORC_OUTSIDE)) { out[i] = -1; continue; }
        real t = bool_cross(c, cls, which, p, d);
        out[i] = (double)(t <= step_max ? t : ORC_INF);
    }
}

/* the crossings of one primitive, exposed for the pins: writes up to `max` ascending values, returns the count */
int orc_all_crossings(const orc_shape *s, double x, double y, double z, double dx, double dy, double dz, double *out, int max)
{
    real p[3] = { x, y, z }, d[3] = { dx, dy, dz }, t[ORC_MAXX];
    int n = all_crossings(s, p, d, t);
    for (int i = 0; i < n && i < max; ++i) out[i] = (double)t[i];
    return n;
}

/* the crossings of the whole line (t of either sign, R32), exposed for the pins */
int orc_line_crossings(const orc_shape *s, double x, double y, double z, double dx, double dy, double dz, double *out, int max)
{
    real p[3] = { x, y, z }, d[3] = { dx, dy, dz }, t[ORC_MAXX];
    int n = line_crossings(s, p, d, t);
    for (int i = 0; i < n && i < max; ++i) out[i] = (double)t[i];
    return n;
}

/* the membership flips of a boolean along the whole line (R28), exposed for the pins */
int orc_boolean_events(const orc_boolean *c, double x, double y, double z, double dx, double dy, double dz, double *out, int max)
{
    real p[3] = { x, y, z }, d[3] = { dx, dy, dz };
    real *t = (real *)malloc(sizeof(real) * ORC_MAXLEAF * ORC_MAXX);
    int n = bool_events(c, p, d, t);
    for (int i = 0; i < n && i < max; ++i) out[i] = (double)t[i];
    free(t);
    return n;
}
