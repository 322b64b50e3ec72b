// vg_nav.cu -- ComputeStep and the volume safety (sec. 8(c) c.2, R12, R13;
// the distance to the geometric border against the physics step, "coordinate
// transformations and distance calculations").
//
// Design: persistent CTAs (a multiple of the SM count), each stages the volume's blob (vg_params.h: FP32 bounding
// spheres, daughter records, candidate grid) into shared memory ONCE with a TMA bulk copy (cp.async.bulk.shared::cluster
// .global + mbarrier complete_tx) and then strides over track tiles, one thread per track.  Per track:
//   phase 1 (per lane; vg_nav_cull.h): FP64 walk of the candidate grid along the ray up to the mother's exit, then an
//           FP32 ray / bounding-sphere test of the few daughters listed in the cells crossed -> a 64-bit candidate
//           mask per chunk of 64 daughters.  Both tests only ever keep too many daughters: a culled daughter's
//           DistanceToIn is +inf by construction, the result is bit-identical to evaluating all daughters.
//   phase 2 (per warp): the candidates of the warp's 32 tracks, pooled per solid kind, are evaluated as one dense work
//           list -- transform p, d with the daughter's 3x4 matrix, DistanceToIn -- and every owner lane takes the
//           lexicographic min of (distance, index) over its own.
// The tie-break of R13 (lowest index, mother first) is kept by comparing (t, k) pairs explicitly.
#include "vg_kernels.cuh"
#include "vg_nav_cull.h"
#include "vg_solid.cuh"
#include "vg_tma.cuh"

#include <mutex>

namespace vg {

#ifndef VG_NAV_BLOCK
#define VG_NAV_BLOCK 256
#endif
#ifndef VG_NAV_MINB
#define VG_NAV_MINB 3
#endif
constexpr int kNavBlock = VG_NAV_BLOCK;
#ifndef VG_NAV_SMALL_N
#define VG_NAV_SMALL_N (148 * 64)
#endif
constexpr int kNavSmallBlock = 64;          // CTA size of ComputeStep for batches below kNavSmallN tracks
constexpr int64_t kNavSmallN = VG_NAV_SMALL_N;

// one elected thread: arm the barrier with the byte count and issue the bulk copy global -> shared
VG_DEV void tma_load_table(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    mbar_expect_tx(bar, bytes);
    bulk_g2s(dst_smem, src_gmem, bytes, bar);
}

template <class S> struct Pick;
template <> struct Pick<Box> { VG_DEV static const BoxP &of(const SolidU &s) { return s.u.box; } };
template <> struct Pick<Orb> { VG_DEV static const OrbP &of(const SolidU &s) { return s.u.orb; } };
template <> struct Pick<Tube> { VG_DEV static const TubeP &of(const SolidU &s) { return s.u.tube; } };
template <> struct Pick<Cone> { VG_DEV static const ConeP &of(const SolidU &s) { return s.u.cone; } };
template <> struct Pick<Trd> { VG_DEV static const TrdP &of(const SolidU &s) { return s.u.trd; } };

VG_DEV const Daughter &daughter_at(const unsigned char *dtab, int k)
{
    return *reinterpret_cast<const Daughter *>(dtab + size_t(k) * kDaughterStride);
}

// ---- phase 2, per lane: every lane walks ITS OWN candidates, one loop per solid kind so that the lanes of a warp run the
// same DistanceToIn code on different daughters.  The form for sparse volumes (a ray meets the bounding sphere of 0-2
// daughters: configs[4]), where pooling the work costs more than the idle lanes it saves (A/B in DESIGN.md sec. 6.4).
template <class S>
VG_DEV void lane_candidates(unsigned long long mk, int base, const unsigned char *dtab, double x, double y, double z,
                            double dx, double dy, double dz, double &best, int &who)
{
    unsigned lo = unsigned(mk), hi = unsigned(mk >> 32);
    while (lo | hi) {
        const bool in_lo = lo != 0u;
        const unsigned w = in_lo ? lo : hi;
        const int k = base + (in_lo ? 0 : 32) + __ffs(int(w)) - 1;
        lo = in_lo ? (lo & (lo - 1u)) : lo;
        hi = in_lo ? hi : (hi & (hi - 1u));
        const Daughter &D = daughter_at(dtab, k);
        double lx = fma(D.m[0], x, fma(D.m[1], y, fma(D.m[2], z, D.m[3])));
        double ly = fma(D.m[4], x, fma(D.m[5], y, fma(D.m[6], z, D.m[7])));
        double lz = fma(D.m[8], x, fma(D.m[9], y, fma(D.m[10], z, D.m[11])));
        double ldx = fma(D.m[0], dx, fma(D.m[1], dy, D.m[2] * dz));
        double ldy = fma(D.m[4], dx, fma(D.m[5], dy, D.m[6] * dz));
        double ldz = fma(D.m[8], dx, fma(D.m[9], dy, D.m[10] * dz));
        double tk = S::dist_in(Pick<S>::of(D.s), lx, ly, lz, ldx, ldy, ldz);
        // R13: lexicographic min of (distance, index); a daughter the track is inside of (-1) is skipped
        bool take = tk >= 0.0 && (tk < best || (tk == best && k < who));
        best = take ? tk : best;
        who = take ? k : who;
    }
}

// ---- phase 2, warp-cooperative: the candidates of the 32 tracks of a warp are evaluated as one dense work list ----
//
// After the cull a lane holds 0-3 candidates and most lanes hold none (22 % of the tracks of configs[4] hit anything):
// with every lane walking its own list the warp runs max-over-lanes iterations at 1-2 active lanes each.  Here the
// lanes pool their candidates of one solid kind in a shared-memory queue (one (lane, daughter) code per entry, places
// from a warp prefix sum), then ALL lanes take one entry each, fetch the owner's track with shuffles, transform it
// into the daughter's frame and run that kind's DistanceToIn -- the same code on 32 different (track, daughter) pairs.
// The distances go back through shared memory; every owner folds its own, in ascending daughter order, into the
// lexicographic minimum of R13.  (BASELINE.json north_star: "warp-level ... where a warp cooperates over daughters".)
constexpr int kCoopPerLane = 2;               // candidates a lane may enqueue per pass (unrolled: no per-lane loops)
constexpr int kCoopQueue = 32 * kCoopPerLane; // entries per warp
constexpr unsigned kFullWarp = 0xffffffffu;

// lowest set bit of the 64-bit mask held as two words, removed from it; 64 if the mask is empty
VG_DEV int pop_lowest(unsigned &lo, unsigned &hi)
{
    const bool in_lo = lo != 0u;
    const unsigned w = in_lo ? lo : hi;
    const int b = (in_lo ? 0 : 32) + __ffs(int(w)) - 1;
    lo = in_lo ? (lo & (lo - 1u)) : lo;
    hi = in_lo ? hi : (hi & (hi - 1u));
    return w ? b : 64;
}

template <class S>
VG_DEV void coop_candidates(unsigned long long mk, int base, const unsigned char *dtab, double x, double y, double z,
                            double dx, double dy, double dz, double &best, int &who, int *q, double *res)
{
    const unsigned lane = threadIdx.x & 31u, lt = (1u << lane) - 1u;
    unsigned lo = unsigned(mk), hi = unsigned(mk >> 32);
    while (true) {
        const int b0 = pop_lowest(lo, hi), b1 = pop_lowest(lo, hi);
        const unsigned B0 = __ballot_sync(kFullWarp, b0 < 64), B1 = __ballot_sync(kFullWarp, b1 < 64);
        if (B0 == 0u) break;
        const int n0 = __popc(B0), total = n0 + __popc(B1);
        const int off0 = __popc(B0 & lt), off1 = n0 + __popc(B1 & lt);
        if (b0 < 64) q[off0] = int(lane << 6) | b0;
        if (b1 < 64) q[off1] = int(lane << 6) | b1;
        __syncwarp();
        for (int r0 = 0; r0 < total; r0 += 32) {
            const int it = r0 + int(lane);
            const bool act = it < total;
            const int code = act ? q[it] : int(lane << 6);
            const int src = code >> 6, k = base + (code & 63);
            const double sx = __shfl_sync(kFullWarp, x, src), sy = __shfl_sync(kFullWarp, y, src),
                         sz = __shfl_sync(kFullWarp, z, src), sdx = __shfl_sync(kFullWarp, dx, src),
                         sdy = __shfl_sync(kFullWarp, dy, src), sdz = __shfl_sync(kFullWarp, dz, src);
            if (act) {
                const Daughter &D = daughter_at(dtab, k);
                double lx = fma(D.m[0], sx, fma(D.m[1], sy, fma(D.m[2], sz, D.m[3])));
                double ly = fma(D.m[4], sx, fma(D.m[5], sy, fma(D.m[6], sz, D.m[7])));
                double lz = fma(D.m[8], sx, fma(D.m[9], sy, fma(D.m[10], sz, D.m[11])));
                double ldx = fma(D.m[0], sdx, fma(D.m[1], sdy, D.m[2] * sdz));
                double ldy = fma(D.m[4], sdx, fma(D.m[5], sdy, D.m[6] * sdz));
                double ldz = fma(D.m[8], sdx, fma(D.m[9], sdy, D.m[10] * sdz));
                res[it] = S::dist_in(Pick<S>::of(D.s), lx, ly, lz, ldx, ldy, ldz);
            }
        }
        __syncwarp();
        // R13: lexicographic min of (distance, index), own candidates in ascending index order; a daughter the track
        // is inside of (-1) is skipped
        const double t0 = b0 < 64 ? res[off0] : -1.0, t1 = b1 < 64 ? res[off1] : -1.0;
        const int k0 = base + b0, k1 = base + b1;
        const bool take0 = t0 >= 0.0 && (t0 < best || (t0 == best && k0 < who));
        best = take0 ? t0 : best;
        who = take0 ? k0 : who;
        const bool take1 = t1 >= 0.0 && (t1 < best || (t1 == best && k1 < who));
        best = take1 ? t1 : best;
        who = take1 ? k1 : who;
        if (!__any_sync(kFullWarp, (lo | hi) != 0u)) break;
        __syncwarp(); // the next pass reuses q and res
    }
}

// ComputeStep; NC = chunks of 64 daughters (1, 2 or 4); COOP = phase 2 pooled over the warp, else per lane; BLOCK = CTA
// size: kNavBlock for batches that fill the GPU, kNavSmallBlock for small ones (four times the CTAs: a 1,024-track call
// runs on 16 SMs instead of 4)
template <int NC, bool COOP, int BLOCK>
__global__ void __launch_bounds__(BLOCK, BLOCK == kNavBlock ? VG_NAV_MINB : 1) nav_step_kernel(const __grid_constant__ SolidU mother,
                                                             const __grid_constant__ NavMeta meta,
                                                             const unsigned char *__restrict__ table, Tracks t,
                                                             double step_max, int64_t n, double *__restrict__ out,
                                                             int32_t *__restrict__ hit)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar;
    __shared__ int q_all[BLOCK / 32][kCoopQueue];
    __shared__ double res_all[BLOCK / 32][kCoopQueue];
    const float4 *cull = reinterpret_cast<const float4 *>(smem_raw);
    const unsigned char *dtab = smem_raw + meta.off_d;
    const unsigned long long *cells = reinterpret_cast<const unsigned long long *>(smem_raw + meta.grid.off_g);
    const int *prim = reinterpret_cast<const int *>(smem_raw + meta.grid.off_p);
    const int nd = meta.nd;
    int *q = q_all[threadIdx.x >> 5];
    double *res = res_all[threadIdx.x >> 5];

    if (threadIdx.x == 0) {
        mbar_init(&bar, 1);
        mbar_fence_init();
    }
    pdl_launch_dependents();
    __syncthreads();
    pdl_wait();
    if (threadIdx.x == 0 && nd > 0) tma_load_table(smem_raw, table, meta.bytes, &bar);
    bool waited = (nd == 0);

    // warp-uniform trip count: the lanes past n take part in the warp's collectives with an empty candidate list
    for (int64_t tile = int64_t(blockIdx.x) * BLOCK; tile < n; tile += int64_t(gridDim.x) * BLOCK) {
        const int64_t i = tile + threadIdx.x;
        const bool valid = i < n;
        double x = 0, y = 0, z = 0, dx = 0, dy = 0, dz = 1;
        if (valid) {
            x = ldg1(t.x + i), y = ldg1(t.y + i), z = ldg1(t.z + i);
            dx = ldg1(t.dx + i), dy = ldg1(t.dy + i), dz = ldg1(t.dz + i);
        }
        if (!waited) { // the track loads above are already in flight while the table lands
            mbar_wait(&bar, 0);
            waited = true;
        }
        double best = solid_dist_out(mother, x, y, z, dx, dy, dz);
        int who = -1;
        if (nd > 0) {
            unsigned long long m[NC];
            nav_cull<NC>(meta.grid, cull, cells, prim, meta.all, x, y, z, dx, dy, dz, best < step_max ? best : step_max, m);
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                const unsigned long long mc = valid ? m[c] : 0ull;
                if (meta.kmask[kBox][c]) { if (COOP) coop_candidates<Box>(mc & meta.kmask[kBox][c], 64 * c, dtab, x, y, z, dx, dy, dz, best, who, q, res); else lane_candidates<Box>(mc & meta.kmask[kBox][c], 64 * c, dtab, x, y, z, dx, dy, dz, best, who); }
                if (meta.kmask[kTube][c]) { if (COOP) coop_candidates<Tube>(mc & meta.kmask[kTube][c], 64 * c, dtab, x, y, z, dx, dy, dz, best, who, q, res); else lane_candidates<Tube>(mc & meta.kmask[kTube][c], 64 * c, dtab, x, y, z, dx, dy, dz, best, who); }
                if (meta.kmask[kOrb][c]) { if (COOP) coop_candidates<Orb>(mc & meta.kmask[kOrb][c], 64 * c, dtab, x, y, z, dx, dy, dz, best, who, q, res); else lane_candidates<Orb>(mc & meta.kmask[kOrb][c], 64 * c, dtab, x, y, z, dx, dy, dz, best, who); }
                if (meta.kmask[kCone][c]) { if (COOP) coop_candidates<Cone>(mc & meta.kmask[kCone][c], 64 * c, dtab, x, y, z, dx, dy, dz, best, who, q, res); else lane_candidates<Cone>(mc & meta.kmask[kCone][c], 64 * c, dtab, x, y, z, dx, dy, dz, best, who); }
                if (meta.kmask[kTrd][c]) { if (COOP) coop_candidates<Trd>(mc & meta.kmask[kTrd][c], 64 * c, dtab, x, y, z, dx, dy, dz, best, who, q, res); else lane_candidates<Trd>(mc & meta.kmask[kTrd][c], 64 * c, dtab, x, y, z, dx, dy, dz, best, who); }
            }
        }
        if (valid) {
            bool phys = best > step_max; // the physics step is shorter than the geometric one
            stg1(out + i, phys ? step_max : best);
            stg1i(hit + i, phys ? -2 : who);
        }
    }
}

// volume safety: min over the mother and every daughter of the exact distance
__global__ void __launch_bounds__(kNavBlock) nav_safety_kernel(const __grid_constant__ SolidU mother,
                                                               const __grid_constant__ NavMeta meta,
                                                               const unsigned char *__restrict__ table, Tracks t,
                                                               int64_t n, double *__restrict__ out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar;
    const float4 *cull = reinterpret_cast<const float4 *>(smem_raw);
    const unsigned char *dtab = smem_raw + meta.off_d;
    const int nd = meta.nd;

    if (threadIdx.x == 0) {
        mbar_init(&bar, 1);
        mbar_fence_init();
    }
    pdl_launch_dependents();
    __syncthreads();
    pdl_wait();
    if (threadIdx.x == 0 && nd > 0) tma_load_table(smem_raw, table, meta.bytes, &bar);
    bool waited = (nd == 0);

    for (int64_t i = int64_t(blockIdx.x) * kNavBlock + threadIdx.x; i < n; i += int64_t(gridDim.x) * kNavBlock) {
        double x = ldg1(t.x + i), y = ldg1(t.y + i), z = ldg1(t.z + i);
        if (!waited) {
            mbar_wait(&bar, 0);
            waited = true;
        }
        double best = -solid_sdf(mother, x, y, z);
        // A daughter lies inside the sphere of radius r about its local origin (the table's FP32 sphere, centre in the
        // mother's frame, r^2 inflated by the rounding bound of the FP32 test: vg_volume_create), so its
        // SafetyToIn >= |p - c| - r and a daughter whose bound is not below the running minimum is skipped.  The
        // candidates: the daughters that can be nearest to a point of the safety grid's cell (vg_nav_cull.h,
        // nav_safety_cell; read from device memory: 64 cells per daughter are too many to stage), else every daughter.
        // One daughter is evaluated first, exactly -- the one with the smallest upper bound over the cell, stored behind
        // the cell's masks; a heuristic with no bearing on the result, the minimum is order-independent -- and the
        // others meet the bound against that value in FP32, then -- after the FP64 transform only they pay for -- in
        // FP64 against the running minimum.
        if (best > 0.0 && nd > 0) {
            const float xf = float(x), yf = float(y), zf = float(z);
            const unsigned long long *cell =
                nav_safety_cell(meta.grid, reinterpret_cast<const unsigned long long *>(table + meta.grid.off_s), meta.nchunks, x, y, z);
            const unsigned long long *cand = cell ? cell : meta.all;
            int probe = -1;
            if (cell) { // the daughter with the smallest upper bound over the cell (vg_volume_create)
                probe = int(cell[meta.nchunks]);
            } else {    // no grid (fewer than 8 daughters): the one whose sphere looks nearest to the point
                float key = 3.0e38f;
                for (int c = 0; c < meta.nchunks; ++c)
                    for (unsigned long long mm = cand[c]; mm; mm &= mm - 1) {
                        const int k = 64 * c + __ffsll((long long)mm) - 1;
                        const float4 sp = cull[k];
                        const float vx = xf - sp.x, vy = yf - sp.y, vz = zf - sp.z;
                        const float q = fmaf(vx, vx, fmaf(vy, vy, fmaf(vz, vz, -sp.w)));
                        probe = q < key ? k : probe;
                        key = fminf(q, key);
                    }
            }
            if (probe >= 0) {
                const Daughter &D = daughter_at(dtab, probe);
                const double lx = fma(D.m[0], x, fma(D.m[1], y, fma(D.m[2], z, D.m[3])));
                const double ly = fma(D.m[4], x, fma(D.m[5], y, fma(D.m[6], z, D.m[7])));
                const double lz = fma(D.m[8], x, fma(D.m[9], y, fma(D.m[10], z, D.m[11])));
                best = dmin(best, solid_sdf(D.s, lx, ly, lz));
            }
            const float bf = float(best);
            for (int c = 0; c < meta.nchunks && best > 0.0; ++c) { // (best <= 0: inside the probe, the branch below)
                unsigned long long m = cand[c];
                if ((probe >> 6) == c) m &= ~(1ull << (probe & 63)); // already counted
                while (m) {
                    const int k = 64 * c + __ffsll((long long)m) - 1;
                    m &= m - 1;
                    const float4 sp = cull[k];
                    const float vx = xf - sp.x, vy = yf - sp.y, vz = zf - sp.z;
                    const float rf = sqrtf(sp.w), reachf = bf + rf;
                    if (!(fmaf(vx, vx, fmaf(vy, vy, vz * vz)) <= reachf * reachf)) continue;
                    const Daughter &D = daughter_at(dtab, k);
                    const double lx = fma(D.m[0], x, fma(D.m[1], y, fma(D.m[2], z, D.m[3])));
                    const double ly = fma(D.m[4], x, fma(D.m[5], y, fma(D.m[6], z, D.m[7])));
                    const double lz = fma(D.m[8], x, fma(D.m[9], y, fma(D.m[10], z, D.m[11])));
                    // the slack keeps the comparison on the safe side of its own rounding
                    const double reach = best + double(rf) * (1.0 + 1e-6);
                    const double l2 = fma(lx, lx, fma(ly, ly, lz * lz));
                    if (best > 0.0 && l2 >= reach * reach * (1.0 + 1e-12)) continue;
                    best = dmin(best, solid_sdf(D.s, lx, ly, lz));
                }
            }
        }
        if (best <= 0.0 && nd > 0) {
            // Outside the mother, on a surface or inside a daughter: only a daughter that HOLDS the point (SafetyToIn
            // < 0) can lower a minimum that is not positive, and its bounding sphere then holds the point too: the
            // candidates are the daughters listed in the point's cell of the candidate grid (vg_nav_cull.h,
            // nav_point_cell; none outside the grid's box, which holds every sphere).  For volumes that keep the
            // containment contract this is at most the daughter the point is in; for the others the result stays the
            // plain minimum over every daughter.
            const unsigned long long *cell =
                nav_point_cell_masks(meta.grid, reinterpret_cast<const unsigned long long *>(smem_raw + meta.grid.off_g), meta.nchunks, x, y, z);
            for (int c = 0; cell && c < meta.nchunks; ++c)
                for (unsigned long long m = cell[c]; m; m &= m - 1) {
                    const Daughter &D = daughter_at(dtab, 64 * c + __ffsll((long long)m) - 1);
                    const double lx = fma(D.m[0], x, fma(D.m[1], y, fma(D.m[2], z, D.m[3])));
                    const double ly = fma(D.m[4], x, fma(D.m[5], y, fma(D.m[6], z, D.m[7])));
                    const double lz = fma(D.m[8], x, fma(D.m[9], y, fma(D.m[10], z, D.m[11])));
                    best = dmin(best, solid_sdf(D.s, lx, ly, lz));
                }
        }
        stg1(out + i, best);
    }
}

// Per-device launch state, process-wide: the shared-memory opt-in of a kernel is a per-device attribute that
// cudaFuncSetAttribute SETS (it does not max), so it is only ever raised, under a lock, and the occupancy is cached
// for the size it was computed for.
struct NavDevState {
    std::mutex mu;
    int sm_count = 0;
    size_t granted = 32 * 1024; // the kernels also hold static shared memory: opt in early
    size_t occ_smem = size_t(-1);
    int per_sm = 0;
};

template <class Kern>
static cudaError_t nav_grid_size(Kern kern, NavDevState *states, size_t smem, int64_t n, unsigned *grid, int block = kNavBlock)
{
    constexpr int kMaxDev = 64;
    int dev = 0;
    cudaError_t err;
    if ((err = cudaGetDevice(&dev)) != cudaSuccess) return err;
    if (dev < 0 || dev >= kMaxDev) return cudaErrorInvalidDevice;
    NavDevState &st = states[dev];
    std::lock_guard<std::mutex> lock(st.mu);
    if (st.sm_count == 0 &&
        (err = cudaDeviceGetAttribute(&st.sm_count, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess)
        return err;
    if (smem > st.granted) {
        if ((err = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem))) != cudaSuccess)
            return err;
        st.granted = smem;
    }
    if (smem != st.occ_smem) {
        if ((err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&st.per_sm, kern, block, smem)) != cudaSuccess) return err;
        if (st.per_sm < 1) st.per_sm = 1;
        st.occ_smem = smem;
    }
    const int64_t want = (n + block - 1) / block;
    const int64_t cap = int64_t(st.sm_count) * st.per_sm; // persistent: one resident wave, a multiple of the SM count
    *grid = unsigned(want < cap ? want : cap);
    return cudaSuccess;
}

template <int NC, bool COOP, int BLOCK>
static cudaError_t launch_step_nc_b(const SolidU &mother, const unsigned char *table_dev, const NavMeta &meta, const Tracks &t,
                                    double step_max, int64_t n, double *step, int32_t *hit, cudaStream_t s)
{
    static NavDevState states[64];
    unsigned grid = 0;
    cudaError_t err = nav_grid_size(nav_step_kernel<NC, COOP, BLOCK>, states, meta.bytes, n, &grid, BLOCK);
    if (err != cudaSuccess) return err;
    return launch_kernel(nav_step_kernel<NC, COOP, BLOCK>, grid, BLOCK, meta.bytes, s, mother, meta, table_dev, t, step_max, n, step, hit);
}

template <int NC, bool COOP>
static cudaError_t launch_step_nc(const SolidU &mother, const unsigned char *table_dev, const NavMeta &meta, const Tracks &t,
                                  double step_max, int64_t n, double *step, int32_t *hit, cudaStream_t s)
{
    if (n < kNavSmallN) return launch_step_nc_b<NC, COOP, kNavSmallBlock>(mother, table_dev, meta, t, step_max, n, step, hit, s);
    return launch_step_nc_b<NC, COOP, kNavBlock>(mother, table_dev, meta, t, step_max, n, step, hit, s);
}

template <bool COOP>
static cudaError_t launch_step_form(const SolidU &mother, const unsigned char *table_dev, const NavMeta &meta, const Tracks &t,
                                    double step_max, int64_t n, double *step, int32_t *hit, cudaStream_t s)
{
    if (meta.nchunks <= 1) return launch_step_nc<1, COOP>(mother, table_dev, meta, t, step_max, n, step, hit, s);
    if (meta.nchunks == 2) return launch_step_nc<2, COOP>(mother, table_dev, meta, t, step_max, n, step, hit, s);
    return launch_step_nc<4, COOP>(mother, table_dev, meta, t, step_max, n, step, hit, s);
}

cudaError_t launch_compute_step(const SolidU &mother, const unsigned char *table_dev, const NavMeta &meta, const Tracks &t,
                                double step_max, int64_t n, double *step, int32_t *hit, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    // phase 2: pooled over the warp where the candidate grid says a ray meets many daughters, per lane where it meets few
    const int64_t form = g_nav_form.load(std::memory_order_relaxed);
    const bool coop = form == 2 || (form == 0 && meta.dense);
    return coop ? launch_step_form<true>(mother, table_dev, meta, t, step_max, n, step, hit, s)
                : launch_step_form<false>(mother, table_dev, meta, t, step_max, n, step, hit, s);
}

cudaError_t launch_volume_safety(const SolidU &mother, const unsigned char *table_dev, const NavMeta &meta, const Tracks &t,
                                 int64_t n, double *safety, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    static NavDevState states[64];
    unsigned grid = 0;
    cudaError_t err = nav_grid_size(nav_safety_kernel, states, meta.bytes, n, &grid);
    if (err != cudaSuccess) return err;
    return launch_kernel(nav_safety_kernel, grid, kNavBlock, meta.bytes, s, mother, meta, table_dev, t, n, safety);
}

} // namespace vg
