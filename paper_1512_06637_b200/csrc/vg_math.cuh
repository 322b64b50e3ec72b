// vg_math.cuh -- FP64 building blocks of the sm_100a kernels.
//
// Why not plain `/` and `sqrt`: on sm_100a an IEEE FP64 divide is MUFU.RCP64H + 8 FP64-pipe instructions
// (+ a slow-path branch), a sqrt MUFU.RSQ64H + 8.  The parity contract is
// |gpu - oracle| <= max(1e-9, 1e-12 |oracle|) (BASELINE.json north_star), not correct rounding, so the
// kernels use a third-order (cubic) refinement of the 20-bit MUFU seed: 3 FP64 instructions for a reciprocal,
// 5 for a square root, relative error ~1e-16 (seed error e ~ 2^-18.5, the refinements leave O(e^3)).
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

namespace vg {

constexpr double kTol = 1e-9;   // BASELINE.json kTolerance, SURVEY.md 8(c) R6
constexpr double kTiny = 1e-300; // stands in for an exactly-zero direction component / denominator
// Reading R32 ("transported to the border"): a start point in the surface band is read as
// starting ON the crossing it sits on.  The kernels take every crossing of the wanted sense with t > -kRayTol and clamp
// the result at 0.  For a start point >= 1e-6 from every surface (the parity generators) no crossing lies within 1e-6
// of t = 0, so nothing changes there; for a band point the crossing it sits on is within kTol / |n.d| <= kRayTol of
// t = 0 unless the ray grazes the surface at |n.d| < 2e-3.
constexpr double kRayTol = 5e-7;

#define VG_DEV __device__ __forceinline__

VG_DEV double inf() { return __longlong_as_double(0x7ff0000000000000LL); }

VG_DEV double sel(bool c, double a, double b) { return c ? a : b; }

// R32: is a crossing at ray parameter t ahead of, or at, the start point?  (NaN: no)
VG_DEV bool ahead(double t) { return t > -kRayTol; }

// max / min that compile to one DSETP + selects; NaN in `b` keeps `a`
VG_DEV double dmax(double a, double b) { return b > a ? b : a; }
VG_DEV double dmin(double a, double b) { return b < a ? b : a; }

VG_DEV double copysign_bits(double mag, double sgn)
{
    // integer-pipe copysign (LOP3 on the high word), keeps the FP64 pipe free
    int hi_m = __double2hiint(mag), hi_s = __double2hiint(sgn);
    return __hiloint2double((hi_m & 0x7fffffff) | (hi_s & 0x80000000), __double2loint(mag));
}

VG_DEV double flipsign_bits(double v, double sgn)
{
    // v * sign(sgn) without FP64 work
    return __hiloint2double(__double2hiint(v) ^ (__double2hiint(sgn) & 0x80000000), __double2loint(v));
}

// Sign tests on the integer pipe: one ISETP on the high word instead of a DSETP, which would take an FP64-pipe
// slot (the FP64 pipe is the scarce unit of these kernels).  They differ from the IEEE
// compares only off the normal range: a +-NaN tests like a number of its sign (every caller ANDs in a real
// compare or a discriminant test that a NaN fails), -0.0 tests negative, and denormals below 2^-1042 test as 0.
VG_DEV bool is_pos(double x) { return __double2hiint(x) > 0; }                        // x > 0
VG_DEV bool is_neg(double x) { return (unsigned)__double2hiint(x) > 0x80000000u; }    // x < 0
VG_DEV bool not_neg(double x) { return __double2hiint(x) >= 0; }                      // x >= 0 (sign bit clear)
VG_DEV bool sign_differs(double a, double b) { return (__double2hiint(a) ^ __double2hiint(b)) < 0; }

// |a| < kTiny (incl. +-0)  ->  +-kTiny, so that 1/a and num/a stay finite-or-inf with the right sign and the
// slab / plane formulas need no special case for rays parallel to a surface.
VG_DEV double nonzero(double a) { return fabs(a) < kTiny ? copysign_bits(kTiny, a) : a; }

#ifndef VG_IEEE_MATH
// 1/a for normal, non-zero a.  r0 = MUFU.RCP64H seed; e = 1 - a r0; r = r0 (1 + e + e^2).
VG_DEV double rcp(double a)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));
    double e = fma(-a, r, 1.0);
    e = fma(e, e, e);
    return fma(r, e, r);
}

// sqrt(a) for a > 0 (normal).  y = MUFU.RSQ64H seed; g = a y; r = 1 - a y^2; sqrt = g (1 + r/2 + 3 r^2/8):
// five FP64 instructions.
VG_DEV double sqrt_pos(double a)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double g = a * y;
    double r = fma(-g, y, 1.0);
    double q = fma(r, 0.375, 0.5);
    return fma(g * r, q, g);
}
#else
VG_DEV double rcp(double a) { return 1.0 / a; }
VG_DEV double sqrt_pos(double a) { return sqrt(a); }
#endif

// sqrt(a) for a >= 0 including exactly 0
VG_DEV double sqrt_nn(double a) { return a > 0.0 ? sqrt_pos(a) : 0.0; }

// 128-bit streaming loads / stores: every track is touched once
VG_DEV double2 ldg2(const double *p)
{
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
VG_DEV double ldg1(const double *p)
{
    double v;
    asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
VG_DEV void stg2(double *p, double a, double b)
{
    asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(a), "d"(b) : "memory");
}
VG_DEV void stg1(double *p, double a) { asm volatile("st.global.cs.f64 [%0], %1;" ::"l"(p), "d"(a) : "memory"); }
VG_DEV void stg2i(int32_t *p, int a, int b)
{
    asm volatile("st.global.cs.v2.s32 [%0], {%1, %2};" ::"l"(p), "r"(a), "r"(b) : "memory");
}
VG_DEV void stg1i(int32_t *p, int a) { asm volatile("st.global.cs.s32 [%0], %1;" ::"l"(p), "r"(a) : "memory"); }

} // namespace vg
