// vg_nav_cull.h -- which daughters of a volume can a ray touch?  (ComputeStep)
//
// ComputeStep is "every placed daughter" (BASELINE.json): DistanceToIn of each of the nd daughters and the lexicographic
// minimum.  A daughter the ray cannot touch has DistanceToIn = +inf and never wins, so the kernel may skip it as long as
// the skip is CONSERVATIVE: it may keep a daughter the ray misses, it must never drop one the ray touches.  This header
// holds that predicate, in one place and compiled for BOTH sides: the device code of nav_kernel (vg_nav.cu) and the
// host-only debug export vg_debug_nav_cull (vg_api.cu), which tests/test_nav_cull.py runs on the CPU over adversarial
// rays against the oracle's DistanceToIn.  Every operation is written with an explicit rounding (fma / fmaf, IEEE
// reciprocal), so host and device evaluate it bit for bit the same.
//
// Two stages per track:
//  1. FP64 walk of a coarse uniform grid laid over the bounding box of all daughter spheres in the mother frame (3-D
//     DDA).  Each cell holds the bit mask of the daughters whose bounding sphere, inflated by `pad`, meets the closed
//     cell; the candidate mask of the ray is the OR over the cells it crosses between the start point and t_lim (the
//     mother's exit or the physics step, whichever is nearer: a daughter crossed later cannot win).  Rounding can make
//     the walk cut a corner the exact ray passes (or the other way round) only within ~1e-13 of the grid's size from a
//     cell edge; `pad` = 1e-6 of the grid diagonal, so a sphere that meets the exact ray inside the skipped cell also
//     meets a visited neighbour.
//  2. FP32 test of the ray against the bounding sphere of each remaining candidate.  With S >= |c - p| + r the FP32
//     evaluation of |c - p|^2 - ((c - p).d)^2 is off by < 30 u S^2 (u = 2^-24); the squared radius in the table is
//     inflated by 64 u S^2 + 1e-6 relative and rounded up (vg_volume_create), S taken for p anywhere in the mother's
//     bounding sphere.  Start points outside that sphere (contract violations) skip both stages and keep every daughter.
#pragma once
#include "vg_params.h"

#if defined(__CUDA_ARCH__)
#define VG_HD __host__ __device__ __forceinline__
#ifdef VG_NAV_FAST_RCP
#define VG_RCP_RN(a) vg::rcp(a)
#else
#define VG_RCP_RN(a) __drcp_rn(a)
#endif
#define VG_CLZ32(m) __clz(int(m))
#elif defined(__CUDACC__)
#define VG_HD __host__ __device__ inline
#define VG_RCP_RN(a) (1.0 / (a))
#define VG_CLZ32(m) __builtin_clz(m)
#else
#define VG_HD inline
#define VG_RCP_RN(a) (1.0 / (a))
#define VG_CLZ32(m) __builtin_clz(m)
#endif

#include <math.h>

namespace vg {

// one axis of the walk: clip [t0, t1] to the slab [0, L] of the grid
VG_HD bool nav_axis_clip(double p, double d, double L, double &t0, double &t1, double &inv)
{
    if (fabs(d) < 1e-300) { // parallel to the slab: inside it for all t or never
        inv = 0.0;
        return p >= 0.0 && p <= L;
    }
    inv = VG_RCP_RN(d);
    double ta = -p * inv, tb = (L - p) * inv;
    double tn = ta < tb ? ta : tb, tf = ta < tb ? tb : ta;
    t0 = tn > t0 ? tn : t0;
    t1 = tf < t1 ? tf : t1;
    return true;
}

// ... and set up the stepping: ray parameter of the next cell border on this axis (tmax), its increment per cell
// (tdelta), the cell index
VG_HD void nav_axis_init(double p, double d, double inv, double t0, double cs, double ics, int g, double &tmax,
                         double &tdelta, int &i)
{
    double e = fma(t0, d, p); // entry coordinate relative to the grid origin
    i = int(floor(e * ics));
    i = i < 0 ? 0 : (i > g - 1 ? g - 1 : i);
    const bool up = d > 0.0, still = inv == 0.0;
    tmax = still ? INFINITY : fma(double(i + (up ? 1 : 0)), cs, -p) * inv;
    tdelta = still ? 0.0 : cs * fabs(inv);
}

// Stage 2: the ray against the inflated bounding sphere {cx, cy, cz, r2} of one daughter, in FP32.
VG_HD bool nav_sphere_keep(const float4 s, float xf, float yf, float zf, float dxf, float dyf, float dzf)
{
    float vx = s.x - xf, vy = s.y - yf, vz = s.z - zf;
    float vv = fmaf(vx, vx, fmaf(vy, vy, vz * vz));
    float tca = fmaf(vx, dxf, fmaf(vy, dyf, vz * dzf));
    float d2 = fmaf(-tca, tca, vv);
    return d2 <= s.w && (tca >= 0.f || vv <= s.w);
}

// Stage 1.  m[c] |= candidates of chunk c (64 daughters per chunk).  `cells`: [gz + 2][gy + 2][gx + 2][NC] masks: the grid
// with a ring of EMPTY cells around it, so the walk needs no bounds test -- it stops when the next border lies beyond
// t1 <= (the ray's exit from the grid) + slack, i.e. at the latest one step per axis into the ring.  The loop body is
// branch-free (selects), so the lanes of a warp stay converged while they walk different cells.
// FUSED: a cell that lists exactly ONE daughter (`prim[cell]` >= 0: the usual case when the grid has about one cell per
// daughter) has that daughter's sphere tested right here and the verdict goes to hit[]; only cells with several daughters
// add their mask to m[] for the loop of stage 2.  Same predicate, same outcome, without a second per-lane loop.
template <int NC, bool FUSED>
VG_HD void nav_grid_walk(const NavGrid &G, const unsigned long long *cells, const int *prim, const float4 *cull, double x,
                         double y, double z, double dx, double dy, double dz, double t_lim, unsigned long long (&m)[NC],
                         unsigned long long (&hit)[NC])
{
#pragma unroll
    for (int c = 0; c < NC; ++c) m[c] = 0ull, hit[c] = 0ull;
    const float xf = float(x), yf = float(y), zf = float(z), dxf = float(dx), dyf = float(dy), dzf = float(dz);
    const double px = x - G.o[0], py = y - G.o[1], pz = z - G.o[2];
    double t0 = 0.0, t1 = fma(t_lim, 1e-9, t_lim) + G.tpad; // a crossing at t_lim itself still counts
    double ivx, ivy, ivz;
    bool ok = nav_axis_clip(px, dx, G.len[0], t0, t1, ivx);
    ok = nav_axis_clip(py, dy, G.len[1], t0, t1, ivy) && ok;
    ok = nav_axis_clip(pz, dz, G.len[2], t0, t1, ivz) && ok;
    if (!ok || !(t0 <= t1)) return;
    double tmx, tmy, tmz, tdx, tdy, tdz;
    int ix, iy, iz;
    nav_axis_init(px, dx, ivx, t0, G.cs[0], G.ics[0], G.g[0], tmx, tdx, ix);
    nav_axis_init(py, dy, ivy, t0, G.cs[1], G.ics[1], G.g[1], tmy, tdy, iy);
    nav_axis_init(pz, dz, ivz, t0, G.cs[2], G.ics[2], G.g[2], tmz, tdz, iz);
    const int sy_ = G.g[0] + 2, sz_ = sy_ * (G.g[1] + 2); // strides of the ringed array
    int idx = (ix + 1) + sy_ * (iy + 1) + sz_ * (iz + 1);
    const int stx = dx > 0.0 ? 1 : -1, sty = dy > 0.0 ? sy_ : -sy_, stz = dz > 0.0 ? sz_ : -sz_;
    const int max_cells = G.g[0] + G.g[1] + G.g[2] + 3; // a straight line crosses at most gx + gy + gz - 2 cells (+ the ring)
    for (int it = 0; it < max_cells; ++it) {
        const int pj = FUSED ? prim[idx] : -1;
        if (pj >= 0) {
            const unsigned long long bit = (unsigned long long)nav_sphere_keep(cull[pj], xf, yf, zf, dxf, dyf, dzf) << (pj & 63);
#pragma unroll
            for (int c = 0; c < NC; ++c) hit[c] |= (NC == 1 || (pj >> 6) == c) ? bit : 0ull;
        } else {
#pragma unroll
            for (int c = 0; c < NC; ++c) m[c] |= cells[idx * NC + c];
        }
        const bool sx = tmx <= tmy && tmx <= tmz, sy = !sx && tmy <= tmz, sz = !sx && !sy;
        const double tsel = sx ? tmx : (sy ? tmy : tmz);
        if (tsel >= t1) break; // (>= also ends a ray that moves along no axis: inf >= inf)
        idx += sx ? stx : (sy ? sty : stz);
        tmx += sx ? tdx : 0.0, tmy += sy ? tdy : 0.0, tmz += sz ? tdz : 0.0;
    }
}

// ... for every candidate of one chunk.  The 64-bit mask is walked as two 32-bit words inside ONE loop (a 64-bit
// find-first-set costs three times a 32-bit one, and two loops would each run to the slowest lane of the warp).
template <int NC>
VG_HD void nav_sphere_refine(const float4 *cull, double x, double y, double z, double dx, double dy, double dz,
                             unsigned long long (&m)[NC])
{
    const float xf = float(x), yf = float(y), zf = float(z), dxf = float(dx), dyf = float(dy), dzf = float(dz);
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        unsigned lo = unsigned(m[c]), hi = unsigned(m[c] >> 32), olo = 0u, ohi = 0u;
        while (lo | hi) {
            const bool in_lo = lo != 0u;
            const unsigned w = in_lo ? lo : hi, low = w & (0u - w);
            lo = in_lo ? lo ^ low : lo;
            hi = in_lo ? hi : hi ^ low;
            const int j = (in_lo ? 31 : 63) - VG_CLZ32(low);
            const bool keep = nav_sphere_keep(cull[64 * c + j], xf, yf, zf, dxf, dyf, dzf);
            olo |= (keep && in_lo) ? low : 0u;
            ohi |= (keep && !in_lo) ? low : 0u;
        }
        m[c] = (unsigned long long)ohi << 32 | olo;
    }
}

// The candidates of a POINT (Locate in a tree of volumes): the mask of the cell that holds it; empty outside the grid's
// box, which holds every sphere.  A point that rounding puts into the neighbouring cell is within ~1e-13 of the border,
// and a sphere that holds it reaches across the border by its pad.
// (nchunks mask words per cell; NULL outside the box)
VG_HD const unsigned long long *nav_point_cell_masks(const NavGrid &G, const unsigned long long *cells, int nchunks, double x,
                                                     double y, double z)
{
    const double px = x - G.o[0], py = y - G.o[1], pz = z - G.o[2];
    if (!(px >= 0.0 && px <= G.len[0] && py >= 0.0 && py <= G.len[1] && pz >= 0.0 && pz <= G.len[2])) return nullptr;
    int ix = int(floor(px * G.ics[0])), iy = int(floor(py * G.ics[1])), iz = int(floor(pz * G.ics[2]));
    ix = ix > G.g[0] - 1 ? G.g[0] - 1 : ix, iy = iy > G.g[1] - 1 ? G.g[1] - 1 : iy, iz = iz > G.g[2] - 1 ? G.g[2] - 1 : iz;
    const int sy_ = G.g[0] + 2, sz_ = sy_ * (G.g[1] + 2);
    return cells + size_t((ix + 1) + sy_ * (iy + 1) + sz_ * (iz + 1)) * size_t(nchunks);
}

// ... of a grid with one word per cell (at most 64 daughters)
VG_HD unsigned long long nav_point_cell(const NavGrid &G, const unsigned long long *cells, double x, double y, double z)
{
    const unsigned long long *c = nav_point_cell_masks(G, cells, 1, x, y, z);
    return c ? *c : 0ull;
}

// The candidates of a point's SAFETY (min over the daughters of SafetyToIn): the mask of the safety grid's cell that
// holds it.  A daughter lies inside its bounding sphere (c, r), so for every point p of a cell
//   |p - c| - r  <=  SafetyToIn(daughter)  <=  |p - c| + r,
// and with U = min over the daughters of (farthest distance from the cell to c) + r, a daughter whose
// (nearest distance from the cell to c) - r exceeds U is strictly farther than some other daughter everywhere in the
// cell: it is never the minimum, and the cell's mask leaves it out (vg_volume_create / vg_world_create; a solid that can
// be empty -- a boolean -- gives no upper bound and does not enter U).  The cells are taken `spad` larger than they
// are, so a point that rounding puts into the neighbouring cell still finds its nearest daughter.  Returns the cell's
// nchunks mask words -- followed by one more word: the daughter that attains U, which the kernels evaluate first (any
// choice gives the same minimum; ~0 if no daughter bounds the cell) -- or NULL outside the grid's box -- the mother's bounding box: such a point is outside the mother --
// or without a grid: the caller then keeps every daughter.
VG_HD const unsigned long long *nav_safety_cell(const NavGrid &G, const unsigned long long *scells, int nchunks, double x,
                                                double y, double z)
{
    const double px = x - G.so[0], py = y - G.so[1], pz = z - G.so[2];
    if (G.gs <= 0 || !(px >= 0.0 && px <= G.slen[0] && py >= 0.0 && py <= G.slen[1] && pz >= 0.0 && pz <= G.slen[2])) return nullptr;
    int ix = int(floor(px * G.sics[0])), iy = int(floor(py * G.sics[1])), iz = int(floor(pz * G.sics[2]));
    ix = ix > G.gs - 1 ? G.gs - 1 : ix, iy = iy > G.gs - 1 ? G.gs - 1 : iy, iz = iz > G.gs - 1 ? G.gs - 1 : iz;
    return scells + size_t((iz * G.gs + iy) * G.gs + ix) * size_t(nchunks + 1);
}

// Both stages.  `all[c]` = every daughter of chunk c (what a start point outside the mother's bounding sphere keeps).
template <int NC>
VG_HD void nav_cull(const NavGrid &G, const float4 *cull, const unsigned long long *cells, const int *prim,
                    const unsigned long long *all, double x, double y, double z, double dx, double dy, double dz, double t_lim,
                    unsigned long long (&m)[NC])
{
    const double pp = fma(x, x, fma(y, y, z * z));
    if (!(pp <= G.rm2)) { // outside the mother's bounding sphere (or NaN): the error bounds above do not cover it
#pragma unroll
        for (int c = 0; c < NC; ++c) m[c] = all[c];
        return;
    }
    unsigned long long hit[NC];
    nav_grid_walk<NC, true>(G, cells, prim, cull, x, y, z, dx, dy, dz, t_lim, m, hit);
    nav_sphere_refine<NC>(cull, x, y, z, dx, dy, dz, m);
#pragma unroll
    for (int c = 0; c < NC; ++c) m[c] |= hit[c];
}

} // namespace vg
