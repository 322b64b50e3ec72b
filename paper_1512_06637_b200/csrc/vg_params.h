// vg_params.h -- plain-data device constants of every solid, derived once on the host at vg_shape_create
// and handed to the kernels by value in kernel-parameter space (constant bank:
// warp-uniform operands cost no instruction and no register).
#pragma once
#include <stdint.h>
#include <vector_types.h> // float4

namespace vg {

constexpr int kMaxZ = 32;       // polycone z-planes
constexpr int kMaxSec = kMaxZ - 1;

enum Kind : int { kBox = 0, kOrb = 1, kTube = 2, kCone = 3, kTrd = 4, kPolycone = 5, kBoolean = 6,
                  kCsg = 7 /* internal: a boolean whose operands include booleans (reading R31); reported as VG_BOOLEAN */,
                  kBoolX = 8 /* internal: a boolean of two solids of which at least one is a polycone; reported as VG_BOOLEAN */ };
enum Query : int { qInside = 0, qDistIn = 1, qDistOut = 2, qSafeIn = 3, qSafeOut = 4 };

// phi segment [sphi, sphi + dphi]; e0, e1 = unit vectors of the two bounding half-planes (reading R11)
struct Wedge {
    double e0x, e0y, e1x, e1y;
    int full; // dphi >= 2 pi: no cut
    int wide; // dphi > pi: the segment is the union of two half-planes, else their intersection
};

struct BoxP {
    double hx, hy, hz;
};

struct OrbP {
    double r, r2;
    double rin2, rout2; // (r - kTol)^2, (r + kTol)^2
};

struct TubeP {
    double rmin, rmax, dz;
    double rmin2, rmax2;
    double rmin_in2, rmax_in2;   // (rmin + kTol)^2, (rmax - kTol)^2 : strictly-inside tests
    double rmin_out2, rmax_out2; // (rmin - kTol)^2 (0 if rmin <= kTol), (rmax + kTol)^2
    double rc, rh;               // (rmin + rmax) / 2, (rmax - rmin) / 2: distance to [rmin, rmax] = max(|rho - rc| - rh, 0)
    Wedge w;
    int hollow; // rmin > 0
};

// one conical (or cylindrical) patch r = A + B z over [z0, z1] plus its (r, z) edge for the exact distance
struct Frustum {
    double A, B;       // generator
    double sec;        // sqrt(1 + B^2): radial width of a band of unit normal distance
    double r0, er;     // radius at z0, r(z1) - r(z0)
    double inv_l2;     // 1 / (er^2 + (z1 - z0)^2)
};

struct ConeP {
    double dz;
    Frustum out, in;
    double rmin1, rmax1, rmin2, rmax2;
    double cap_c1, cap_h1, cap_c2, cap_h2; // centre (rmin + rmax) / 2 and half-width (rmax - rmin) / 2 of the two cap annuli
    Wedge w;
    int hollow; // rmin1 > 0 || rmin2 > 0 : the inner patch is a surface
};

struct TrdP {
    double dx1, dx2, dy1, dy2, dz;
    double fx, mx, icx, cx; // X(z) = mx + fx z; cx = sqrt(1 + fx^2)
    double fy, my, icy, cy;
    double inv_kx, inv_ky;  // 1 / ((d2 - d1)^2 + (2 dz c)^2) for the slanted edge of the +x / +y face
    double hex, hey;        // dz cx, dz cy: half-heights of the +x / +y face along its slant
    double sfx, sfy;        // icx fx, icy fy: z shift of the foot of the perpendicular per unit plane distance
    double kxx, kyx, kxx_s, kyx_s; // +x face: edge vector of its slanted side (dy2 - dy1, 2 hex), and the same / |edge|^2
    double kxy, kyy, kxy_s, kyy_s; // +y face: (dx2 - dx1, 2 hey), and the same / |edge|^2
};

struct PconSec {
    double z0, z1;
    Frustum out, in;
};

// A z step (reading R26: two planes at one z): the radii jump between section k and section k + 1 and the outline has
// a horizontal edge there, i.e. up to two annular faces at z: [olo, ohi] where the outer radius jumps and [ilo, ihi]
// where the inner one does (an empty range, lo > hi, if that radius does not jump).  `oup` / `iup`: the material lies
// BELOW the face (its outward normal is +z): rmax falls across the step / rmin rises across it.
struct PconStep {
    double z;
    double olo, ohi, ilo, ihi;
    int oup, iup;
};

struct PolyconeP {
    int nsec;            // sections of non-zero length, in z order; consecutive sections share their boundary plane
    unsigned inner_mask; // bit k: section k has an inner surface (rmin_k > 0 || rmin_{k+1} > 0)
    unsigned step_mask;  // bit k: the radii jump at the plane between section k and section k + 1 (step[k] is valid)
    int nstep;
    Wedge w;
    double zlo, zhi;
    double cap_lo_rmin, cap_lo_rmax, cap_hi_rmin, cap_hi_rmax;
    double rb2; // square of the largest rmax, inflated by 1e-9 relative: bounding cylinder of the ordered walk
    PconSec sec[kMaxSec];
    PconStep step[kMaxSec - 1];
};

// Candidate grid of a full-phi polycone (vg_pcon_grid.h): kPconGridZ x kPconGridR cells over
// rho in [0, kPconGridR / inv_cr), z in [zg0, zg0 + kPconGridZ / inv_cz); one 64-bit mask of candidate segments per
// cell (bit 0 / 1 = lower / upper cap, bit 2 + 2k = outer edge of section k, 3 + 2k = inner edge: up to 15 sections fit
// the low word; the faces of the j-th z step follow the sections at bits 2 + 2 nsec + 2j (outer) and + 1 (inner);
// sections + steps <= 31, so 64 bits suffice), one byte per z row with the section index at the row's lower edge.
// Device memory owned by the vg_shape.
#ifndef VG_PCON_GRID_R
#define VG_PCON_GRID_R 64
#endif
#ifndef VG_PCON_GRID_Z
#define VG_PCON_GRID_Z 128
#endif
constexpr int kPconGridR = VG_PCON_GRID_R, kPconGridZ = VG_PCON_GRID_Z;
constexpr int kPconCapLoBit = 0, kPconCapHiBit = 1, kPconSecBit0 = 2;

struct PconGridGeom {
    double inv_cr, inv_cz, zg0;
};

// One record per section for the lanes-per-track kernels (vg_pcon_coop.cuh), in device memory: a lane reads the record of
// ITS section, so the table cannot live in the constant bank (divergent indices serialise there).  20 doubles.
struct alignas(16) PconCoopSec {
    double z0, z1, Ao, Bo, Ai, Bi, seco, seci; // slab, generators r = A + B z of the outer / inner patch, sqrt(1 + B^2)
    double ro0, ero, ilo, ri0, eri, ili;       // outline edges: (r0, z0) -> (r0 + er, z1), 1 / |edge|^2
    double sz, solo, sohi, silo, sihi;         // the z step on top of this section (flags & 2): PconStep z, olo, ohi, ilo, ihi
    int flags, pad;                            // 1: inner surface, 2: step above, 4: step.oup, 8: step.iup
};

// One compact record per section for the ordered walks (vg_pcon_walk.cuh): staged in shared memory by the persistent
// kernels, read from device memory by the medium-batch kernel.  14 doubles, 16-byte aligned.
struct alignas(16) PconWalkSec {
    double z0, z1;
    double Ao, Bo, Ai, Bi;    // generators r = A + B z of the outer / inner patch
    double ro0, ero, ilo;     // outer edge (r0, z0) -> (r0 + er, z1), 1 / |edge|^2
    double ri0, eri, ili;     // inner edge
    double seco, seci;        // sqrt(1 + B^2) of both patches (tolerance band of the Inside test)
};

struct PconGrid {
    const PconWalkSec *wtab;         // [nsec] in device memory; NULL: not uploaded
    const double *segs;              // [64][6] segment records of the candidate grids (vg_pcon_walk.cuh), device memory
    const PconCoopSec *coop;         // [nsec]; NULL: not uploaded, the thread-per-track kernels serve every batch size
    const unsigned long long *masks; // [kPconGridZ][kPconGridR]; NULL: no grid, the ordered walk serves the safeties
    const unsigned long long *face_masks; // phi cut only: [kPconGridZ][2 kPconGridR] over u in [-R, R), every outline edge
    const unsigned char *rows;       // [kPconGridZ]
    PconGridGeom g;
};

// One record per segment of the polycone's (r, z) outline, numbered like the mask bits of the candidate grids: start point,
// edge vector, edge vector / |edge|^2 (six doubles, 16-byte aligned).  Staged in shared memory by the persistent safety
// kernel, read from device memory by the one-track-per-thread one.
constexpr int kPconSegStride = 6;
#ifdef __CUDACC__
#define VG_PARAMS_HD __host__ __device__
#else
#define VG_PARAMS_HD
#endif
// record s of the table (bit s of the grid masks); plain arithmetic, compiled for the host too (vg_api.cu uploads the table
// the one-track-per-thread safety kernel reads from device memory)
VG_PARAMS_HD inline void pcon_seg_record(const PolyconeP &p, int s, double *o)
{
    double r0 = 0, z0 = 0, er = 0, ez = 0, il = 0;
    const int k = (s - kPconSecBit0) >> 1;
    if (s >= kPconSecBit0 && k < p.nsec) {
        const PconSec &c = p.sec[k];
        const Frustum &f = (s & 1) ? c.in : c.out;
        r0 = f.r0, z0 = c.z0, er = f.er, ez = c.z1 - c.z0, il = f.inv_l2;
    }
    const int js = s - kPconSecBit0 - 2 * p.nsec; // >= 0: face (js & 1 ? inner : outer) of the (js >> 1)-th z step
    if (js >= 0 && (js >> 1) < p.nstep) {
        int kk = -1;
        for (int q = 0, seen = 0; q + 1 < p.nsec; ++q)
            if ((p.step_mask >> q) & 1u) {
                if (seen++ == (js >> 1)) kk = q;
            }
        const PconStep &t = p.step[kk];
        const double lo = (js & 1) ? t.ilo : t.olo, hi = (js & 1) ? t.ihi : t.ohi;
        if (hi > lo) r0 = lo, z0 = t.z, er = hi - lo, ez = 0.0, il = 1.0 / (er * er);
    }
    if (s == kPconCapLoBit) r0 = p.cap_lo_rmin, z0 = p.zlo, er = p.cap_lo_rmax - p.cap_lo_rmin, il = 1.0 / (er * er);
    if (s == kPconCapHiBit) r0 = p.cap_hi_rmin, z0 = p.zhi, er = p.cap_hi_rmax - p.cap_hi_rmin, il = 1.0 / (er * er);
    o[0] = r0, o[1] = z0, o[2] = er, o[3] = ez, o[4] = er * il, o[5] = ez * il;
}

// a solid that may be a mother or a daughter of a volume (every kind except the polycone), or an operand of a boolean
// (there a polycone too: kind == kPolycone and u.pcon points at its constants in device memory, vg_boolx.cu)
struct PolyconeP;
struct SolidU {
    int kind;
    int pad;
    union {
        BoxP box;
        OrbP orb;
        TubeP tube;
        ConeP cone;
        TrdP trd;
        const PolyconeP *pcon;
    } u;
};

// boolean solid C = A op B of two primitives (readings R27-R29): A in the frame of C, B placed by X (frame of C -> frame of B)
enum BoolOp : int { kUnion = 0, kIntersection = 1, kSubtraction = 2 };
struct BoolP {
    int op;
    int pad;
    double X[12];
    SolidU a, b;
};

// A CSG tree flattened at vg_boolean_create (reading R31): up to kCsgMaxLeaf primitives, each with the transform from the
// frame of the tree to its own frame, and the tree as a postfix program over them (token < 0x80: push that leaf,
// 0x80 | op: combine the two on top, left operand below).  Leaves appear in tree order, so "lowest leaf first" is the
// oracle's "a tie goes to the left operand".
constexpr int kCsgMaxLeaf = 8, kCsgMaxProg = 2 * kCsgMaxLeaf;
struct CsgP {
    int nleaf, nprog;
    unsigned char prog[kCsgMaxProg];
    double X[kCsgMaxLeaf][12];
    SolidU leaf[kCsgMaxLeaf];
};

// navigation: one placed daughter
struct Daughter {
    double m[12]; // row-major [R | b], mother -> local (reading R12)
    SolidU s;
};

// The daughter table is ONE blob in device memory that a CTA stages into shared memory with a single TMA bulk copy:
//   [0, 16 ndp)                float4 {cx, cy, cz, r2}: bounding sphere of daughter k in the MOTHER frame, in FP32 with
//                              the radius inflated by the FP32 error bound (conservative cull, see vg_nav.cu);
//                              ndp = nd rounded up to a multiple of kCullUnroll, padding entries have r2 = -1
//   [off_d, off_d + nd stride) the Daughter records, stride = sizeof(Daughter) rounded up to an ODD number of 8-byte
//                              words so that lanes reading different daughters spread over the shared-memory banks
//   [off_g, off_g + 8 ncell nchunks)  candidate masks of the grid cells (NavGrid below), off_g a multiple of 16
//   [off_p, off_p + 4 ncell)          the only daughter of each cell or -1
//   total (NavMeta::bytes) rounded up to a multiple of 16 bytes (bulk-copy granularity)
//   [off_s, off_s + 8 gs^3 (nchunks + 1))  behind the staged part, read from device memory: the safety grid's cells
//                                     (nchunks masks + the daughter to evaluate first)
constexpr int kCullUnroll = 8;
constexpr int kDaughterStride = int(sizeof(Daughter)) + (((sizeof(Daughter) / 8) % 2 == 0) ? 8 : 0);
constexpr int kNavChunks = 4; // 64 daughters per chunk, VG_MAX_DAUGHTERS = 256
constexpr int kNavKinds = 5;  // every kind except the polycone

// Uniform grid over the bounding box of all daughter spheres in the mother frame (vg_nav_cull.h): g[0] x g[1] x g[2]
// cells of size cs, each with one 64-bit candidate mask per chunk at blob offset off_g, stored with a ring of empty cells
// around the grid ([gz + 2][gy + 2][gx + 2][nchunks]).
constexpr int kNavGridMax = 8; // cells per axis
// The safety grid (vg_nav_cull.h, nav_safety_cell): a finer grid over the mother's own bounding box (every point with a
// positive SafetyToOut lies in it) whose cells list the daughters that can be the NEAREST one of a point of the cell
// (bounding-sphere bounds, taken at create time).
#ifndef VG_NAV_SAFE_MAX
#define VG_NAV_SAFE_MAX 32
#endif
constexpr int kNavSafeGridMax = VG_NAV_SAFE_MAX;
constexpr int kNavSafeGridMin = 8; // daughters from which the grid is built
struct NavGrid {
    double o[3], len[3], cs[3], ics[3]; // origin, extent, cell size and its inverse per axis
    double tpad;                        // absolute slack added to the ray-parameter limit of the walk
    double rm2;                         // squared radius of the mother's bounding sphere about its origin, inflated
    int g[3];
    unsigned off_g;
    unsigned off_p; // int32 per cell (same ringed layout): the cell's only daughter, -1 if it lists none or several
    int gs;         // the SAFETY grid: gs^3 cells (no ring) over the bounding box of the MOTHER, 0 = none
    double so[3], slen[3], sics[3]; // its origin, extent and inverse cell size per axis
    double spad;    // how far outside its cell a point may sit and still find its nearest daughter in the cell's list
    unsigned off_s; // its masks (nchunks words per cell): daughters that can be the nearest one of a point of the cell
    unsigned pad;
};

struct NavMeta {
    int nd, nchunks;
    int dense, pad; // the grid's cells list many daughters each (vg_volume_create): phase 2 of ComputeStep pools the warp's work
    unsigned off_d, bytes;
    unsigned long long kmask[kNavKinds][kNavChunks]; // bit j of kmask[kind][c]: daughter 64 c + j is of that kind
    unsigned long long all[kNavChunks];              // every daughter of the chunk
    NavGrid grid;
};

// hierarchy of volumes (vg_world.cu): one record per node, plus the child lists as one int32 array
struct alignas(16) WorldNode {
    double G[12];   // world frame -> local frame, composed at create from the chain of placements
    double X[12];   // parent's local frame -> local frame (the placement itself)
    double bs[4];   // bounding sphere in the PARENT's local frame: centre, squared radius inflated by the rounding bound
    double br;      // its radius (inflated), for the safety cull
    SolidU s;
    int parent, child0, nchild; // children: child_list[child0 .. child0 + nchild), ascending node index
    int ext;                    // s.kind == kPolycone / kBoolean: index into the world's polycone / boolean array
    int grid;                   // >= 0: index of the node's candidate grid over its children (WorldGrid), -1: none
    int pad_[3];
};

// Candidate grid of a node with kWorldGridMin..64 children (vg_nav_cull.h; bit j = the j-th child of the node's list): Step
// walks it along the ray and Locate looks the point's cell up instead of testing every child's bounding sphere.
constexpr int kWorldGridMin = 12;
struct WorldGrid {
    NavGrid g;
    unsigned cells0, prim0; // first element of the node's cells / prim arrays in the world's pools (safety cells: g.off_s,
                            // an element index into the cells pool)
    unsigned long long all; // every child of the node
};

// everything a world kernel needs, by value in kernel-parameter space
struct WorldTab {
    const WorldNode *nodes;
    const int32_t *kids;          // the child lists
    const float4 *cull;           // FP32 bounding spheres in child-list order
    const struct PolyconeP *pcons; // nodes that are polycones (reading R30)
    const struct BoolP *bools;     // nodes that are booleans of two primitives
    const struct CsgP *csgs;       // nodes that are nested booleans (reading R31)
    const WorldGrid *grids;        // candidate grids of the nodes with many children
    const unsigned long long *gcells; // their cells' masks (one 64-bit word per cell, ringed layout)
    const int *gprim;              // ... and the only child of each cell or -1
    int nnodes;
    int has_ext;                   // any polycone / boolean node: the kernels with their code are launched
};

} // namespace vg
