// vg_nav.cu -- ComputeStep and the volume safety (sec. 8(c) c.2, R12, R13;
// the distance to the geometric border against the physics step, "coordinate
// transformations and distance calculations").
//
// Design: persistent CTAs (a multiple of the SM count), each stages the daughter table blob (vg_params.h) into
// shared memory ONCE with a TMA bulk copy (cp.async.bulk.shared::cluster.global + mbarrier complete_tx) and then
// strides over track tiles, one thread per track.  Per track:
//   phase 1 (FP32 pipe, warp-uniform loop): ray against the bounding sphere of EVERY daughter in the mother
//           frame -> a 64-bit candidate mask per lane.  The sphere radii carry the FP32 error bound, so the test
//           can only keep too many daughters, never drop one the ray can touch: a culled daughter's DistanceToIn
//           is +inf by construction and the result is bit-identical to evaluating all daughters.
//   phase 2 (FP64 pipe, per-lane loop): each lane walks ITS OWN candidates (typically 0-2 of 64), one loop per solid
//           kind so that the lanes of a warp execute the same DistanceToIn code on different daughters: transform
//           p, d with the daughter's 3x4 matrix, DistanceToIn, lexicographic min of (distance, index).
// The tie-break of R13 (lowest index, mother first) is kept by comparing (t, k) pairs explicitly, because
// candidates are not visited in index order.
#include "vg_kernels.cuh"
#include "vg_solid.cuh"
#include "vg_tma.cuh"

namespace vg {

constexpr int kNavBlock = 128;

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

// phase 2 for the candidates of one kind: every lane walks its own bit mask
template <class S>
VG_DEV void eval_candidates(unsigned long long mk, int base, const unsigned char *dtab, double x, double y, double z,
                            double dx, double dy, double dz, double &best, int &who)
{
    while (mk) {
        int k = base + __ffsll((long long)mk) - 1;
        mk &= mk - 1;
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

// kStep = true: ComputeStep; false: volume safety (directions unused)
template <bool kStep>
__global__ void __launch_bounds__(kNavBlock) nav_kernel(const __grid_constant__ SolidU mother,
                                                        const __grid_constant__ NavMeta meta,
                                                        const unsigned char *__restrict__ table, Tracks t,
                                                        double step_max, int64_t n, double *__restrict__ out,
                                                        int32_t *__restrict__ hit)
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
        double dx = 0, dy = 0, dz = 0;
        if (kStep) {
            dx = ldg1(t.dx + i);
            dy = ldg1(t.dy + i);
            dz = ldg1(t.dz + i);
        }
        if (!waited) { // the track loads above are already in flight while the table lands
            mbar_wait(&bar, 0);
            waited = true;
        }
        if (kStep) {
            double best = solid_dist_out(mother, x, y, z, dx, dy, dz);
            int who = -1;
            const float xf = float(x), yf = float(y), zf = float(z), dxf = float(dx), dyf = float(dy), dzf = float(dz);
#pragma unroll 1
            for (int c = 0; c < meta.nchunks; ++c) {
                const int base = 64 * c;
                const int lim = min(64, ((nd - base) + kCullUnroll - 1) / kCullUnroll * kCullUnroll);
                unsigned long long m = 0;
#pragma unroll 1
                for (int j0 = 0; j0 < lim; j0 += kCullUnroll) {
#pragma unroll
                    for (int u = 0; u < kCullUnroll; ++u) {
                        float4 s = cull[base + j0 + u]; // warp-uniform address: shared-memory broadcast
                        float vx = s.x - xf, vy = s.y - yf, vz = s.z - zf;
                        float vv = fmaf(vx, vx, fmaf(vy, vy, vz * vz));
                        float tca = fmaf(vx, dxf, fmaf(vy, dyf, vz * dzf));
                        float d2 = fmaf(-tca, tca, vv);
                        bool keep = d2 <= s.w && (tca >= 0.f || vv <= s.w);
                        m |= (unsigned long long)keep << (j0 + u);
                    }
                }
                if (meta.kmask[kBox][c]) eval_candidates<Box>(m & meta.kmask[kBox][c], base, dtab, x, y, z, dx, dy, dz, best, who);
                if (meta.kmask[kTube][c]) eval_candidates<Tube>(m & meta.kmask[kTube][c], base, dtab, x, y, z, dx, dy, dz, best, who);
                if (meta.kmask[kOrb][c]) eval_candidates<Orb>(m & meta.kmask[kOrb][c], base, dtab, x, y, z, dx, dy, dz, best, who);
                if (meta.kmask[kCone][c]) eval_candidates<Cone>(m & meta.kmask[kCone][c], base, dtab, x, y, z, dx, dy, dz, best, who);
                if (meta.kmask[kTrd][c]) eval_candidates<Trd>(m & meta.kmask[kTrd][c], base, dtab, x, y, z, dx, dy, dz, best, who);
            }
            bool phys = best > step_max; // the physics step is shorter than the geometric one
            stg1(out + i, phys ? step_max : best);
            stg1i(hit + i, phys ? -2 : who);
        } else {
            double best = -solid_sdf(mother, x, y, z);
#pragma unroll 1
            for (int k = 0; k < nd; ++k) {
                const Daughter &D = daughter_at(dtab, k);
                double lx = fma(D.m[0], x, fma(D.m[1], y, fma(D.m[2], z, D.m[3])));
                double ly = fma(D.m[4], x, fma(D.m[5], y, fma(D.m[6], z, D.m[7])));
                double lz = fma(D.m[8], x, fma(D.m[9], y, fma(D.m[10], z, D.m[11])));
                best = dmin(best, solid_sdf(D.s, lx, ly, lz));
            }
            stg1(out + i, best);
        }
    }
}

template <bool kStep>
static cudaError_t launch_nav(const SolidU &mother, const unsigned char *table_dev, const NavMeta &meta, const Tracks &t,
                              double step_max, int64_t n, double *out, int32_t *hit, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    size_t smem = meta.bytes;
    // caches of the device queries, per host thread AND per device (the shared-memory opt-in is a per-device attribute of
    // the kernel): after the first launch on a device the path makes no CUDA call but cudaGetDevice and the launch
    constexpr int kMaxDev = 64;
    struct DevCache {
        int sm_count = 0, per_sm = 0;
        size_t smem_granted = 48 * 1024, smem_occ = size_t(-1);
    };
    static thread_local DevCache cache[kMaxDev];
    cudaError_t err;
    int dev = 0;
    if ((err = cudaGetDevice(&dev)) != cudaSuccess) return err;
    if (dev < 0 || dev >= kMaxDev) return cudaErrorInvalidDevice;
    int &sm_count = cache[dev].sm_count, &per_sm = cache[dev].per_sm;
    size_t &smem_granted = cache[dev].smem_granted, &smem_occ = cache[dev].smem_occ;
    if (sm_count == 0) {
        if ((err = cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return err;
    }
    if (smem > smem_granted) {
        if ((err = cudaFuncSetAttribute(nav_kernel<kStep>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem))) !=
            cudaSuccess)
            return err;
        smem_granted = smem;
    }
    if (smem != smem_occ) {
        if ((err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, nav_kernel<kStep>, kNavBlock, smem)) !=
            cudaSuccess)
            return err;
        if (per_sm < 1) per_sm = 1;
        smem_occ = smem;
    }
    int64_t want = (n + kNavBlock - 1) / kNavBlock;
    int64_t cap = int64_t(sm_count) * per_sm; // persistent: one resident wave, a multiple of the SM count
    unsigned grid = unsigned(want < cap ? want : cap);
    return launch_kernel(nav_kernel<kStep>, grid, kNavBlock, smem, s, mother, meta, table_dev, t, step_max, n, out, hit);
}

cudaError_t launch_compute_step(const SolidU &mother, const unsigned char *table_dev, const NavMeta &meta, const Tracks &t,
                                double step_max, int64_t n, double *step, int32_t *hit, cudaStream_t s)
{
    return launch_nav<true>(mother, table_dev, meta, t, step_max, n, step, hit, s);
}

cudaError_t launch_volume_safety(const SolidU &mother, const unsigned char *table_dev, const NavMeta &meta, const Tracks &t,
                                 int64_t n, double *safety, cudaStream_t s)
{
    return launch_nav<false>(mother, table_dev, meta, t, 0.0, n, safety, nullptr, s);
}

} // namespace vg
