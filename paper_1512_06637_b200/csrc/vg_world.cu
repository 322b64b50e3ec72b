// vg_world.cu -- queries over a tree of placed solids ("with hierarchical connections one can build the
// whole detector"; PAPER.md:98 the particle "is transported to the border" and changes volume; SURVEY.md sec. 8(f) f3;
// readings R22-R25, R30 in DESIGN.md): Locate, Step (one-level ComputeStep in each track's own node + the node entered)
// and the per-node safety.
//
// Design: one thread per track; the node table (vg_params.h WorldNode, ~0.5 KiB per node) stays in global memory and
// is read through L1 (tracks of a warp sit in different nodes, so there is no table to share per CTA as in
// vg_nav.cu).  Every child is first tested against its bounding sphere in the parent's frame -- a point test for
// Locate, a ray test for Step, a lower bound |p - c| - r for the safety -- and only the survivors pay for the 3x4
// transform and the solid's own code.  Locate and Step run the test as in vg_nav.cu: phase 1 on the FP32 pipe over a
// compact float4 array laid out like the child lists (64 children per 64-bit mask), phase 2 walks the mask in FP64.
// The spheres are inflated by the rounding bound of the test, so the cull can only keep too many children: a culled
// child's DistanceToIn is +inf, its Inside is OUTSIDE and its SafetyToIn exceeds the running minimum, i.e. results
// are identical to visiting every child.  Children are visited in ascending node index, so the strict `<` scan is
// the tie-break of R13.
#include "vg_csg.cuh"
#include "vg_nav_cull.h"

namespace vg {

constexpr int kWorldBlock = 128;

VG_DEV void xf_point(const double *m, double x, double y, double z, double &lx, double &ly, double &lz)
{
    lx = fma(m[0], x, fma(m[1], y, fma(m[2], z, m[3])));
    ly = fma(m[4], x, fma(m[5], y, fma(m[6], z, m[7])));
    lz = fma(m[8], x, fma(m[9], y, fma(m[10], z, m[11])));
}

VG_DEV void xf_dir(const double *m, double dx, double dy, double dz, double &lx, double &ly, double &lz)
{
    lx = fma(m[0], dx, fma(m[1], dy, m[2] * dz));
    ly = fma(m[4], dx, fma(m[5], dy, m[6] * dz));
    lz = fma(m[8], dx, fma(m[9], dy, m[10] * dz));
}

// ---- a node's solid: the five placeable primitives inline; polycones and booleans (reading R30) live in side arrays and
// are reached through calls that are NOT inlined, so that the common path keeps its registers ----

__device__ __noinline__ int ext_inside(const WorldTab &w, const WorldNode &N, double x, double y, double z)
{
    if (N.s.kind == kCsg) {
        unsigned in, out;
        csg_classes(w.csgs[N.ext], x, y, z, in, out);
        return csg_classify(w.csgs[N.ext], in, out);
    }
    if (N.s.kind == kBoolX) return bool_inside_pt<true>(w.bools[N.ext], x, y, z); // a polycone operand: constants in w.pcons
    return N.s.kind == kPolycone ? Polycone::inside(w.pcons[N.ext], x, y, z) : bool_inside_pt(w.bools[N.ext], x, y, z);
}

__device__ __noinline__ double ext_sdf(const WorldTab &w, const WorldNode &N, double x, double y, double z)
{
    if (N.s.kind == kCsg) return csg_sdf(w.csgs[N.ext], x, y, z);
    if (N.s.kind == kBoolX) return bool_sdf_pt<true>(w.bools[N.ext], x, y, z);
    return N.s.kind == kPolycone ? Polycone::safety(w.pcons[N.ext], x, y, z) : bool_sdf_pt(w.bools[N.ext], x, y, z);
}

__device__ __noinline__ double ext_distance(const WorldTab &w, const WorldNode &N, bool to_out, double x, double y, double z,
                                            double dx, double dy, double dz)
{
    if (N.s.kind == kPolycone)
        return to_out ? Polycone::dist_out(w.pcons[N.ext], x, y, z, dx, dy, dz) : Polycone::dist_in(w.pcons[N.ext], x, y, z, dx, dy, dz);
    if (N.s.kind == kCsg) return csg_distance(w.csgs[N.ext], to_out, x, y, z, dx, dy, dz);
    if (N.s.kind == kBoolX) return bool_distance<-1, -1, true>(w.bools[N.ext], to_out, x, y, z, dx, dy, dz);
    return bool_distance<-1, -1>(w.bools[N.ext], to_out, x, y, z, dx, dy, dz);
}

template <bool EXT> VG_DEV int node_inside(const WorldTab &w, const WorldNode &N, double x, double y, double z)
{
    return (!EXT || N.s.kind < kPolycone) ? solid_inside(N.s, x, y, z) : ext_inside(w, N, x, y, z);
}

template <bool EXT> VG_DEV double node_sdf(const WorldTab &w, const WorldNode &N, double x, double y, double z)
{
    return (!EXT || N.s.kind < kPolycone) ? solid_sdf(N.s, x, y, z) : ext_sdf(w, N, x, y, z);
}

template <bool EXT> VG_DEV double node_dist_in(const WorldTab &w, const WorldNode &N, double x, double y, double z, double dx, double dy, double dz)
{
    return (!EXT || N.s.kind < kPolycone) ? solid_dist_in(N.s, x, y, z, dx, dy, dz) : ext_distance(w, N, false, x, y, z, dx, dy, dz);
}

template <bool EXT> VG_DEV double node_dist_out(const WorldTab &w, const WorldNode &N, double x, double y, double z, double dx, double dy, double dz)
{
    return (!EXT || N.s.kind < kPolycone) ? solid_dist_out(N.s, x, y, z, dx, dy, dz) : ext_distance(w, N, true, x, y, z, dx, dy, dz);
}

// EXT: the world holds polycone / boolean nodes (their code costs registers: primitive-only worlds run the lean instantiation)
template <bool EXT>
__global__ void __launch_bounds__(kWorldBlock)
    world_locate_kernel(const __grid_constant__ WorldTab w, Tracks t, int64_t n, int32_t *__restrict__ out)
{
    const WorldNode *__restrict__ nodes = w.nodes;
    const int32_t *__restrict__ kids = w.kids;
    const float4 *__restrict__ cull = w.cull;
    pdl_launch_dependents();
    pdl_wait();
    const int64_t i = int64_t(blockIdx.x) * kWorldBlock + threadIdx.x;
    if (i >= n) return;
    double x, y, z;
    xf_point(nodes[0].X, ldg1(t.x + i), ldg1(t.y + i), ldg1(t.z + i), x, y, z);
    int cur = -1;
    if (node_inside<EXT>(w, nodes[0], x, y, z) == cInside) {
        cur = 0;
        bool moved = true;
        while (moved) {
            moved = false;
            const int c0 = nodes[cur].child0, nc = nodes[cur].nchild, gi = nodes[cur].grid;
            const float xf = float(x), yf = float(y), zf = float(z);
            for (int base = 0; base < nc && !moved; base += 64) {
                const int lim = min(64, nc - base);
                unsigned long long m = 0;
                if (gi >= 0) { // a node with many children: the candidates of the point's grid cell (vg_nav_cull.h)
                    const WorldGrid &G = w.grids[gi];
                    m = nav_point_cell(G.g, w.gcells + G.cells0, x, y, z);
                } else {
#pragma unroll 4
                    for (int j = 0; j < lim; ++j) { // phase 1, FP32: inside the child's bounding sphere?
                        const float4 sp = __ldg(cull + c0 + base + j);
                        const float vx = xf - sp.x, vy = yf - sp.y, vz = zf - sp.z;
                        m |= (unsigned long long)(fmaf(vx, vx, fmaf(vy, vy, vz * vz)) <= sp.w) << j;
                    }
                }
                while (m) { // phase 2, FP64, ascending child index
                    const int c = kids[c0 + base + __ffsll((long long)m) - 1];
                    m &= m - 1;
                    const WorldNode &C = nodes[c];
                    double lx, ly, lz;
                    xf_point(C.X, x, y, z, lx, ly, lz);
                    if (node_inside<EXT>(w, C, lx, ly, lz) == cInside) {
                        cur = c;
                        x = lx, y = ly, z = lz;
                        moved = true;
                        break;
                    }
                }
            }
        }
    }
    stg1i(out + i, cur);
}

// kStep: Step (R24); else the per-node safety (R25)
template <bool kStep, bool EXT>
__global__ void __launch_bounds__(kWorldBlock)
    world_node_kernel(const __grid_constant__ WorldTab w, const int32_t *__restrict__ node, Tracks t, double step_max,
                      int64_t n, double *__restrict__ out, int32_t *__restrict__ next)
{
    const WorldNode *__restrict__ nodes = w.nodes;
    const int32_t *__restrict__ kids = w.kids;
    const float4 *__restrict__ cull = w.cull;
    const int nnodes = w.nnodes;
    pdl_launch_dependents();
    pdl_wait();
    const int64_t i = int64_t(blockIdx.x) * kWorldBlock + threadIdx.x;
    if (i >= n) return;
    // node == NULL: a one-level volume held as a world (vg_volume with polycone / boolean solids): every track is in node 0
    // and the result follows vg_compute_step's convention (hit = daughter index, -1 mother exit, -2 physics step)
    const bool vol = node == nullptr;
    const int nd = vol ? 0 : node[i];
    if (nd < 0 || nd >= nnodes) {
        stg1(out + i, -1.0);
        if (kStep) stg1i(next + i, -1);
        return;
    }
    const WorldNode &N = nodes[nd];
    double x, y, z, dx = 0, dy = 0, dz = 0;
    xf_point(N.G, ldg1(t.x + i), ldg1(t.y + i), ldg1(t.z + i), x, y, z);
    if (kStep) xf_dir(N.G, ldg1(t.dx + i), ldg1(t.dy + i), ldg1(t.dz + i), dx, dy, dz);
    const int c0 = N.child0, nc = N.nchild;
    if (kStep) {
        double best = node_dist_out<EXT>(w, N, x, y, z, dx, dy, dz);
        int who = N.parent;
        const float xf = float(x), yf = float(y), zf = float(z), dxf = float(dx), dyf = float(dy), dzf = float(dz);
        for (int base = 0; base < nc; base += 64) {
            const int lim = min(64, nc - base);
            unsigned long long m = 0;
            if (N.grid >= 0) { // a node with many children: ComputeStep's cull (grid walk + sphere test, vg_nav_cull.h)
                const WorldGrid &G = w.grids[N.grid];
                unsigned long long mm[1];
                nav_cull<1>(G.g, cull + c0, w.gcells + G.cells0, w.gprim + G.prim0, &G.all, x, y, z, dx, dy, dz,
                            best < step_max ? best : step_max, mm);
                m = mm[0];
            } else {
#pragma unroll 4
                for (int j = 0; j < lim; ++j) {
                    // phase 1, FP32: ray against the bounding sphere (closest approach of the line; sphere not behind the start)
                    // (the predicate of ComputeStep's cull, vg_nav_cull.h: pinned on the CPU by tests/test_nav_cull.py, stage 2)
                    const float4 sp = __ldg(cull + c0 + base + j);
                    m |= (unsigned long long)nav_sphere_keep(sp, xf, yf, zf, dxf, dyf, dzf) << j;
                }
            }
            while (m) { // phase 2, FP64, ascending child index: the strict < is R13's tie-break
                const int c = kids[c0 + base + __ffsll((long long)m) - 1];
                m &= m - 1;
                const WorldNode &C = nodes[c];
                double lx, ly, lz, ldx, ldy, ldz;
                xf_point(C.X, x, y, z, lx, ly, lz);
                xf_dir(C.X, dx, dy, dz, ldx, ldy, ldz);
                const double tk = node_dist_in<EXT>(w, C, lx, ly, lz, ldx, ldy, ldz);
                const bool take = tk >= 0.0 && tk < best;
                best = take ? tk : best;
                who = take ? c : who;
            }
        }
        const bool phys = best > step_max; // the physics step is shorter than the geometric one
        stg1(out + i, phys ? step_max : best);
        stg1i(next + i, vol ? (phys ? -2 : (who < 0 ? -1 : who - 1)) : (phys ? nd : who));
    } else {
        double best = -node_sdf<EXT>(w, N, x, y, z);
        // SafetyToIn of a child >= |p - c| - r: a child whose bound is not below the running minimum is skipped (valid for
        // a minimum of either sign, so trees whose children overlap or stick out of their parent get the plain minimum too).
        // The candidates: for a node with a safety grid, the children that can be nearest to a point of its cell
        // (vg_nav_cull.h, nav_safety_cell), else every child.  One child is evaluated first -- the one with the smallest
        // upper bound over the cell, stored with the cell, else the one whose sphere looks nearest in FP32; a heuristic
        // with no bearing on the result, the minimum is order-independent -- so that the bound, taken in FP64 against
        // the running minimum, leaves few of the others.
        const float xf = float(x), yf = float(y), zf = float(z);
        for (int base = 0; base < nc; base += 64) { // (every chunk whatever the sign so far: the result is the plain minimum)
            const int lim = min(64, nc - base);
            unsigned long long m = lim == 64 ? ~0ull : ((1ull << lim) - 1ull);
            int probe = -1;
            const unsigned long long *cell = nullptr;
            if (N.grid >= 0) {
                const WorldGrid &G = w.grids[N.grid];
                cell = nav_safety_cell(G.g, w.gcells + G.g.off_s, 1, x, y, z);
            }
            if (cell) { // the cell's list, and the child with the smallest upper bound over the cell
                m = cell[0];
                probe = int(cell[1]);
            } else {
                float key = 3.0e38f;
                for (unsigned long long mm = m; mm; mm &= mm - 1) {
                    const int j = __ffsll((long long)mm) - 1;
                    const float4 sp = __ldg(cull + c0 + base + j);
                    const float vx = xf - sp.x, vy = yf - sp.y, vz = zf - sp.z;
                    const float k = fmaf(vx, vx, fmaf(vy, vy, fmaf(vz, vz, -sp.w)));
                    probe = k < key ? j : probe;
                    key = fminf(k, key);
                }
            }
            if (probe >= 0) {
                const WorldNode &C = nodes[kids[c0 + base + probe]];
                double lx, ly, lz;
                xf_point(C.X, x, y, z, lx, ly, lz);
                best = dmin(best, node_sdf<EXT>(w, C, lx, ly, lz));
                m &= ~(1ull << probe);
            }
            while (m) {
                const int c = kids[c0 + base + __ffsll((long long)m) - 1];
                m &= m - 1;
                const WorldNode &C = nodes[c];
                const double vx = x - C.bs[0], vy = y - C.bs[1], vz = z - C.bs[2];
                const double vv = fma(vx, vx, fma(vy, vy, vz * vz));
                const double reach = best + C.br;
                if (vv > reach * reach * (1.0 + 1e-9)) continue;
                double lx, ly, lz;
                xf_point(C.X, x, y, z, lx, ly, lz);
                best = dmin(best, node_sdf<EXT>(w, C, lx, ly, lz));
            }
        }
        stg1(out + i, best);
    }
}

cudaError_t launch_world_locate(const WorldTab &w, const Tracks &t, int64_t n, int32_t *out, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    const unsigned grid = unsigned((n + kWorldBlock - 1) / kWorldBlock);
    return w.has_ext ? launch_kernel(world_locate_kernel<true>, grid, kWorldBlock, 0, s, w, t, n, out)
                     : launch_kernel(world_locate_kernel<false>, grid, kWorldBlock, 0, s, w, t, n, out);
}

cudaError_t launch_world_step(const WorldTab &w, const int32_t *node, const Tracks &t, double step_max, int64_t n, double *step,
                              int32_t *next, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    const unsigned grid = unsigned((n + kWorldBlock - 1) / kWorldBlock);
    return w.has_ext ? launch_kernel(world_node_kernel<true, true>, grid, kWorldBlock, 0, s, w, node, t, step_max, n, step, next)
                     : launch_kernel(world_node_kernel<true, false>, grid, kWorldBlock, 0, s, w, node, t, step_max, n, step, next);
}

cudaError_t launch_world_safety(const WorldTab &w, const int32_t *node, const Tracks &t, int64_t n, double *safety, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    const unsigned grid = unsigned((n + kWorldBlock - 1) / kWorldBlock);
    int32_t *none = nullptr;
    return w.has_ext ? launch_kernel(world_node_kernel<false, true>, grid, kWorldBlock, 0, s, w, node, t, 0.0, n, safety, none)
                     : launch_kernel(world_node_kernel<false, false>, grid, kWorldBlock, 0, s, w, node, t, 0.0, n, safety, none);
}

} // namespace vg
