// vg_solid.cuh -- run-time dispatch over the solid kinds a placed volume may have (every kind but the polycone):
// the navigator (vg_nav.cu) and the world kernels (vg_world.cu) hold their solids as SolidU records.
#pragma once
#include "vg_shapes.cuh"

namespace vg {

VG_DEV double solid_dist_in(const SolidU &s, double x, double y, double z, double dx, double dy, double dz)
{
    switch (s.kind) { // warp-uniform
    case kBox: return Box::dist_in(s.u.box, x, y, z, dx, dy, dz);
    case kOrb: return Orb::dist_in(s.u.orb, x, y, z, dx, dy, dz);
    case kTube: return Tube::dist_in(s.u.tube, x, y, z, dx, dy, dz);
    case kCone: return Cone::dist_in(s.u.cone, x, y, z, dx, dy, dz);
    default: return Trd::dist_in(s.u.trd, x, y, z, dx, dy, dz);
    }
}

VG_DEV double solid_dist_out(const SolidU &s, double x, double y, double z, double dx, double dy, double dz)
{
    switch (s.kind) {
    case kBox: return Box::dist_out(s.u.box, x, y, z, dx, dy, dz);
    case kOrb: return Orb::dist_out(s.u.orb, x, y, z, dx, dy, dz);
    case kTube: return Tube::dist_out(s.u.tube, x, y, z, dx, dy, dz);
    case kCone: return Cone::dist_out(s.u.cone, x, y, z, dx, dy, dz);
    default: return Trd::dist_out(s.u.trd, x, y, z, dx, dy, dz);
    }
}

VG_DEV double solid_sdf(const SolidU &s, double x, double y, double z)
{
    switch (s.kind) {
    case kBox: return Box::safety(s.u.box, x, y, z);
    case kOrb: return Orb::safety(s.u.orb, x, y, z);
    case kTube: return Tube::safety(s.u.tube, x, y, z);
    case kCone: return Cone::safety(s.u.cone, x, y, z);
    default: return Trd::safety(s.u.trd, x, y, z);
    }
}

VG_DEV int solid_inside(const SolidU &s, double x, double y, double z)
{
    switch (s.kind) {
    case kBox: return Box::inside(s.u.box, x, y, z);
    case kOrb: return Orb::inside(s.u.orb, x, y, z);
    case kTube: return Tube::inside(s.u.tube, x, y, z);
    case kCone: return Cone::inside(s.u.cone, x, y, z);
    default: return Trd::inside(s.u.trd, x, y, z);
    }
}

} // namespace vg
