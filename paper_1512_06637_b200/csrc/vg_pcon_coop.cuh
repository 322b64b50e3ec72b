// vg_pcon_coop.cuh -- the small-batch form of the full-phi polycone queries: a GROUP OF LANES per track.
//
// the GPU only pays off at large N.  At N <= 2^14 the thread-per-track walk (vg_pcon_walk.cuh) keeps two
// to thirty-two CTAs busy while each lane walks up to nsec sections one after the other behind a staged table and a
// barrier: the launch is pure latency (4.7 us for 1,024 tracks of configs[3]; an orb at the same N takes 1.2 us).
// Here G = 4..32 lanes share one track (BASELINE.json north_star: "a warp cooperates"): lane g evaluates section g
// (and g + G, ...) -- the two conical patches, the section's share of the Inside test, the z step above it, or its two
// outline edges for the safety -- and the group folds its candidates with log2(G) shuffle steps (min of the
// distances, OR of the class bits).  The critical path is ONE section instead of nsec, there is no shared-memory
// table and no barrier: each lane reads its section's record straight from global memory (built once at
// vg_shape_create, L2-resident), and that read overlaps the track loads.  Same candidates and validity tests as
// PolyconeT (vg_shapes.cuh), so the same results as every other form of the query.
#pragma once
#include "vg_kernels.cuh"

namespace vg {

constexpr int kCoopBlock = 128;

VG_DEV double2 ldg2c(const double *p) { return __ldg(reinterpret_cast<const double2 *>(p)); }

// min over the G lanes of a group (G a power of two, groups aligned in the warp; every lane of the warp takes part)
template <int G> VG_DEV double group_min(double v)
{
#pragma unroll
    for (int o = G >> 1; o > 0; o >>= 1) v = dmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// OR over the group of a predicate: one vote for the whole warp, then the group's bits
template <int G> VG_DEV bool group_any(bool f)
{
    const unsigned b = __ballot_sync(0xffffffffu, f);
    const unsigned lane = threadIdx.x & 31u;
    const unsigned gm = (G == 32 ? 0xffffffffu : ((1u << G) - 1u)) << (lane & ~unsigned(G - 1));
    return (b & gm) != 0u;
}

// the fields of a section record one query needs, in registers
struct CoopRec {
    double2 zz, ob, ib, sc, e0, e1, e2, s0, s1;
    double sihi;
    int flags;
};

template <int Q> VG_DEV void coop_load(CoopRec &c, const PconCoopSec *rec, bool steps)
{
    constexpr bool kDir = (Q == qDistIn || Q == qDistOut);
    const double *q = reinterpret_cast<const double *>(rec);
    c.zz = ldg2c(q), c.ob = ldg2c(q + 2), c.ib = ldg2c(q + 4); // z0 z1 | Ao Bo | Ai Bi
    c.flags = __ldg(&rec->flags);
    if (kDir || Q == qInside) c.sc = ldg2c(q + 6); // seco seci
    if (Q == qSafeIn || Q == qSafeOut) c.e0 = ldg2c(q + 8), c.e1 = ldg2c(q + 10), c.e2 = ldg2c(q + 12); // ro0 ero | ilo ri0 | eri ili
    if (steps) c.s0 = ldg2c(q + 14), c.s1 = ldg2c(q + 16), c.sihi = __ldg(q + 18); // z olo | ohi ilo | ihi
}

template <int Q, int G>
__global__ void __launch_bounds__(kCoopBlock)
    pcon_coop_kernel(const __grid_constant__ PolyconeP p, const PconCoopSec *__restrict__ tab, Tracks t, double step_max,
                     int64_t n, void *out_any)
{
    constexpr bool kDir = (Q == qDistIn || Q == qDistOut);
    constexpr bool kLeaving = (Q == qDistOut);
    const int64_t tid = int64_t(blockIdx.x) * kCoopBlock + threadIdx.x;
    const int64_t i_raw = tid / G;
    const int g = int(threadIdx.x) & (G - 1);
    const bool valid = i_raw < n;
    const int64_t i = valid ? i_raw : n - 1; // the lanes past the end redo the last track: every shuffle stays full-warp
    // The lane's first section record is requested before anything else -- the table is a constant of the shape, not a
    // product of the previous kernel, so the read may even precede griddepcontrol.wait -- and the track loads follow
    // at once: issue is in order, and the first use of a track coordinate would otherwise hold the record loads back.
    CoopRec c = {};
    const bool steps = p.step_mask != 0u; // uniform: no load waits for another one
    if (g < p.nsec) coop_load<Q>(c, tab + g, steps);
    pdl_launch_dependents();
    pdl_wait();
    const double x = ldg1(t.x + i), y = ldg1(t.y + i), z = ldg1(t.z + i);
    double dx = 0, dy = 0, dz = 0;
    if (kDir) dx = ldg1(t.dx + i), dy = ldg1(t.dy + i), dz = ldg1(t.dz + i);

    const double rho2 = fma(x, x, y * y);
    RayRZ r;
    r.rho2 = rho2, r.a_xy = fma(dx, dx, dy * dy), r.b_xy = fma(x, dx, y * dy);
    const double rho = sqrt_nn(rho2);
    const double idz = kDir ? rcp(dz) : 0.0; // NaN for dz = 0: caps and step faces rejected
    const bool up = dz > 0.0;

    double best = inf();   // distances: nearest crossing of the wanted sense; safeties: smallest squared distance
    bool any_in = false, any_near = false, near_face = false, in2d = false;
#pragma unroll 1
    for (int k = g; k < p.nsec; k += G) {
        const double2 zz = c.zz, ob = c.ob, ib = c.ib;
        const int flags = c.flags;
        const bool inner = flags & 1, has_step = flags & 2;
        const double ro = fma(ob.y, z, ob.x), ri = fma(ib.y, z, ib.x);
        if (kDir || Q == qInside) { // Inside, per section (PolyconeT::classify_pt)
            const double2 sc = c.sc;
            const double to = kTol * sc.x, ti = kTol * sc.y;
            const bool zin = z >= zz.x && z <= zz.y, znear = z >= zz.x - kTol && z <= zz.y + kTol;
            any_in = any_in || (zin && rho < ro - to && (!inner || rho > ri + ti));
            any_near = any_near || (znear && rho <= ro + to && (!inner || rho >= ri - ti));
        }
        if (kDir) { // crossings of the two patches (PolyconeT::cross)
            Frustum f;
            bool ok;
            f.A = ob.x, f.B = ob.y;
            double tt = frustum_root(f, r, z, dz, kLeaving, ok);
            double zh = fma(tt, dz, z);
            ok = ok && zh >= zz.x && zh <= zz.y;
            best = (ok && tt < best) ? tt : best;
            f.A = ib.x, f.B = ib.y;
            tt = frustum_root(f, r, z, dz, !kLeaving, ok);
            zh = fma(tt, dz, z);
            ok = ok && inner && zh >= zz.x && zh <= zz.y;
            best = (ok && tt < best) ? tt : best;
        }
        if (Q == qSafeIn || Q == qSafeOut) { // the two outline edges of the section (PolyconeT::outline_d2)
            const double2 e0 = c.e0, e1 = c.e1, e2 = c.e2;
            const double ez = zz.y - zz.x;
            best = dmin(best, seg_d2(rho, z, e0.x, zz.x, e0.y, ez, e1.x));
            const double di = seg_d2(rho, z, e1.y, zz.x, e2.x, ez, e2.y);
            best = inner ? dmin(best, di) : best;
            in2d = in2d || (z >= zz.x && z <= zz.y && rho <= ro && rho >= ri);
        }
        if (has_step) { // the annular faces of the z step on top of this section (reading R26)
            const double2 s0 = c.s0, s1 = c.s1;
            const double sihi = c.sihi;
            const double sz = s0.x, olo = s0.y, ohi = s1.x, ilo = s1.y, ihi = sihi;
            const bool oup = flags & 4, iup = flags & 8;
            if (kDir || Q == qInside)
                near_face = near_face || (fabs(z - sz) <= kTol && ((rho >= olo - kTol && rho <= ohi + kTol) ||
                                                                   (rho >= ilo - kTol && rho <= ihi + kTol)));
            if (kDir) {
                const double tt = (sz - z) * idz;
                const double rh2 = fma(tt, fma(tt, r.a_xy, r.b_xy + r.b_xy), rho2);
                const bool on_o = rh2 >= olo * olo && rh2 <= ohi * ohi && ohi > olo && (kLeaving ? oup == up : oup != up);
                const bool on_i = rh2 >= ilo * ilo && rh2 <= ihi * ihi && ihi > ilo && (kLeaving ? iup == up : iup != up);
                const bool ok = ahead(tt) && (on_o || on_i);
                best = (ok && tt < best) ? tt : best;
            }
            if (Q == qSafeIn || Q == qSafeOut) {
                const double vz = z - sz, vz2 = vz * vz;
                const double bo = dmax(dmax(olo - rho, rho - ohi), 0.0), bi = dmax(dmax(ilo - rho, rho - ihi), 0.0);
                best = ohi > olo ? dmin(best, fma(bo, bo, vz2)) : best;
                best = ihi > ilo ? dmin(best, fma(bi, bi, vz2)) : best;
            }
        }
        if (k + G < p.nsec) coop_load<Q>(c, tab + k + G, steps);
    }
    // the end caps: every lane (the arithmetic is independent of the section loop and overlaps it)
    if (kDir) {
        {
            const double tt = (p.zlo - z) * idz;
            const double rh2 = fma(tt, fma(tt, r.a_xy, r.b_xy + r.b_xy), rho2);
            const bool sense = kLeaving ? dz < 0.0 : dz > 0.0;
            const bool ok = sense && ahead(tt) && rh2 >= p.cap_lo_rmin * p.cap_lo_rmin && rh2 <= p.cap_lo_rmax * p.cap_lo_rmax;
            best = (ok && tt < best) ? tt : best;
        }
        {
            const double tt = (p.zhi - z) * idz;
            const double rh2 = fma(tt, fma(tt, r.a_xy, r.b_xy + r.b_xy), rho2);
            const bool sense = kLeaving ? dz > 0.0 : dz < 0.0;
            const bool ok = sense && ahead(tt) && rh2 >= p.cap_hi_rmin * p.cap_hi_rmin && rh2 <= p.cap_hi_rmax * p.cap_hi_rmax;
            best = (ok && tt < best) ? tt : best;
        }
    }
    if (Q == qSafeIn || Q == qSafeOut) {
        const double b1 = dmax(dmax(p.cap_lo_rmin - rho, rho - p.cap_lo_rmax), 0.0), v1 = z - p.zlo;
        const double b2 = dmax(dmax(p.cap_hi_rmin - rho, rho - p.cap_hi_rmax), 0.0), v2 = z - p.zhi;
        best = dmin(best, dmin(fma(b1, b1, v1 * v1), fma(b2, b2, v2 * v2)));
    }

    // fold the group
    if (Q != qInside) best = group_min<G>(best);
    bool in = false, outside = false;
    if (kDir || Q == qInside) {
        in = group_any<G>(any_in) && z > p.zlo + kTol && z < p.zhi - kTol;
        if (p.step_mask) in = in && !group_any<G>(near_face);
        if (Q != qDistIn) outside = !group_any<G>(any_near);
    }
    if (Q == qSafeIn || Q == qSafeOut) in2d = group_any<G>(in2d);
    if (!valid || g != 0) return;
    if (Q == qInside) {
        stg1i(static_cast<int32_t *>(out_any) + i, classify(in, outside));
    } else if (kDir) {
        const double tt = (kLeaving ? outside : in) ? -1.0 : dmax(best, 0.0);
        stg1(static_cast<double *>(out_any) + i, tt <= step_max ? tt : inf());
    } else {
        const double d = sqrt_nn(best), s = in2d ? -d : d;
        stg1(static_cast<double *>(out_any) + i, Q == qSafeIn ? s : -s);
    }
}

extern std::atomic<int64_t> g_coop_max_n; // vg_set_option(VG_OPT_COOP_MAX_N)

template <int Q, int G>
cudaError_t launch_pcon_coop_g(const PolyconeP &p, const PconGrid &g, const Tracks &t, double step_max, int64_t n, void *out,
                               cudaStream_t s)
{
    const int64_t threads = n * G;
    const unsigned grid = unsigned((threads + kCoopBlock - 1) / kCoopBlock);
    return launch_kernel(pcon_coop_kernel<Q, G>, grid, kCoopBlock, 0, s, p, g.coop, t, step_max, n, out);
}

// Lanes per track.  Up to kCoopWideN tracks the launch is pure latency and every section gets its own lane (the smallest
// power of two >= nsec, at least 4); above it the idle lanes of that layout cost throughput, so a group is half as
// wide and each lane takes two sections in turn.
#ifndef VG_COOP_WIDE_N
#define VG_COOP_WIDE_N 4096
#endif
#ifndef VG_COOP_SHIFT
#define VG_COOP_SHIFT 1
#endif
template <int Q>
cudaError_t launch_pcon_coop(const PolyconeP &p, const PconGrid &g, const Tracks &t, double step_max, int64_t n, void *out,
                             cudaStream_t s)
{
    int G = 4;
    while (G < p.nsec && G < 32) G <<= 1;
    if (n > VG_COOP_WIDE_N) G = (G >> VG_COOP_SHIFT) < 4 ? 4 : (G >> VG_COOP_SHIFT);
    switch (G) {
    case 4: return launch_pcon_coop_g<Q, 4>(p, g, t, step_max, n, out, s);
    case 8: return launch_pcon_coop_g<Q, 8>(p, g, t, step_max, n, out, s);
    case 16: return launch_pcon_coop_g<Q, 16>(p, g, t, step_max, n, out, s);
    }
    return launch_pcon_coop_g<Q, 32>(p, g, t, step_max, n, out, s);
}

} // namespace vg
