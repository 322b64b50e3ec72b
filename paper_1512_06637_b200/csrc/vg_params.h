// vg_params.h -- plain-data device constants of every solid, derived once on the host at vg_shape_create
// and handed to the kernels by value in kernel-parameter space (constant bank:
// warp-uniform operands cost no instruction and no register).
#pragma once
#include <stdint.h>

namespace vg {

constexpr int kMaxZ = 32;       // polycone z-planes
constexpr int kMaxSec = kMaxZ - 1;

enum Kind : int { kBox = 0, kOrb = 1, kTube = 2, kCone = 3, kTrd = 4, kPolycone = 5 };
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
    Wedge w;
    int hollow; // rmin1 > 0 || rmin2 > 0 : the inner patch is a surface
};

struct TrdP {
    double dx1, dx2, dy1, dy2, dz;
    double fx, mx, icx, cx; // X(z) = mx + fx z; cx = sqrt(1 + fx^2)
    double fy, my, icy, cy;
    double inv_kx, inv_ky;  // 1 / ((d2 - d1)^2 + (2 dz c)^2) for the slanted edge of the +x / +y face
};

struct PconSec {
    double z0, z1;
    Frustum out, in;
};

struct PolyconeP {
    int nsec;
    unsigned inner_mask; // bit k: section k has an inner surface (rmin_k > 0 || rmin_{k+1} > 0)
    Wedge w;
    double zlo, zhi;
    double cap_lo_rmin, cap_lo_rmax, cap_hi_rmin, cap_hi_rmax;
    PconSec sec[kMaxSec];
};

// a solid that may be a mother or a daughter of a volume (every kind except the polycone)
struct SolidU {
    int kind;
    int pad;
    union {
        BoxP box;
        OrbP orb;
        TubeP tube;
        ConeP cone;
        TrdP trd;
    } u;
};

// navigation: one placed daughter; sizeof is a multiple of 16 so that the table moves by one TMA bulk copy
struct alignas(16) Daughter {
    double m[12]; // row-major [R | b], mother -> local (reading R12)
    SolidU s;
};
static_assert(sizeof(Daughter) % 16 == 0, "daughter table entries must be 16-byte multiples");

} // namespace vg
