// vg_nav.cu -- ComputeStep and the volume safety (sec. 8(c) c.2, R12, R13;
// the distance to the geometric border against the physics step, "coordinate
// transformations and distance calculations").
//
// Design: persistent CTAs (a multiple of the SM count), each stages the daughter table
// (nd x sizeof(Daughter), 16-byte multiple) into shared memory ONCE with a TMA bulk copy
// (cp.async.bulk.shared::cluster.global + mbarrier complete_tx) and then strides over track tiles.  One
// thread owns one track and walks the daughters in index order: every lane of a warp reads the same table
// entry (shared-memory broadcast, no bank conflict), the switch on the daughter's kind is warp-uniform, and
// the sequential strict '<' reproduces the tie-break of R13 (lowest index, mother first) with no reduction.
#include "vg_kernels.cuh"

namespace vg {

constexpr int kNavBlock = 128;

VG_DEV uint32_t smem_u32(const void *p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }

// one elected thread: arm the barrier with the byte count and issue the bulk copy global -> shared
VG_DEV void tma_load_table(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    uint32_t b = smem_u32(bar), d = smem_u32(dst_smem);
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(b), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(d),
                 "l"(src_gmem), "r"(bytes), "r"(b)
                 : "memory");
}

VG_DEV void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

VG_DEV void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t b = smem_u32(bar), done = 0;
    while (!done) { // try_wait suspends the thread in hardware for a bounded time; loop until the phase flips
        asm volatile("{\n"
                     ".reg .pred p;\n"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
                     "selp.u32 %0, 1, 0, p;\n"
                     "}\n"
                     : "=r"(done)
                     : "r"(b), "r"(parity)
                     : "memory");
    }
}

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

// kStep = true: ComputeStep; false: volume safety (directions unused)
template <bool kStep>
__global__ void __launch_bounds__(kNavBlock) nav_kernel(const __grid_constant__ SolidU mother,
                                                        const Daughter *__restrict__ table, int nd, Tracks t,
                                                        double step_max, int64_t n, double *__restrict__ out,
                                                        int32_t *__restrict__ hit)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar;
    const Daughter *tab = reinterpret_cast<const Daughter *>(smem_raw);

    if (threadIdx.x == 0) mbar_init(&bar, 1);
    __syncthreads();
    if (threadIdx.x == 0 && nd > 0) tma_load_table(smem_raw, table, uint32_t(nd) * uint32_t(sizeof(Daughter)), &bar);
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
#pragma unroll 1
            for (int k = 0; k < nd; ++k) {
                const Daughter &D = tab[k];
                double lx = fma(D.m[0], x, fma(D.m[1], y, fma(D.m[2], z, D.m[3])));
                double ly = fma(D.m[4], x, fma(D.m[5], y, fma(D.m[6], z, D.m[7])));
                double lz = fma(D.m[8], x, fma(D.m[9], y, fma(D.m[10], z, D.m[11])));
                double ldx = fma(D.m[0], dx, fma(D.m[1], dy, D.m[2] * dz));
                double ldy = fma(D.m[4], dx, fma(D.m[5], dy, D.m[6] * dz));
                double ldz = fma(D.m[8], dx, fma(D.m[9], dy, D.m[10] * dz));
                double tk = solid_dist_in(D.s, lx, ly, lz, ldx, ldy, ldz);
                bool take = tk >= 0.0 && tk < best; // R13: strict '<', a daughter the track is inside of (-1) is skipped
                best = take ? tk : best;
                who = take ? k : who;
            }
            bool phys = best > step_max; // the physics step is shorter than the geometric one
            stg1(out + i, phys ? step_max : best);
            stg1i(hit + i, phys ? -2 : who);
        } else {
            double best = -solid_sdf(mother, x, y, z);
#pragma unroll 1
            for (int k = 0; k < nd; ++k) {
                const Daughter &D = tab[k];
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
static cudaError_t launch_nav(const SolidU &mother, const Daughter *table_dev, int nd, const Tracks &t, double step_max,
                              int64_t n, double *out, int32_t *hit, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    size_t smem = size_t(nd > 0 ? nd : 1) * sizeof(Daughter);
    static thread_local int sm_count = 0;
    cudaError_t err;
    if (sm_count == 0) {
        int dev = 0;
        if ((err = cudaGetDevice(&dev)) != cudaSuccess) return err;
        if ((err = cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return err;
    }
    static thread_local size_t smem_granted = 48 * 1024; // default dynamic shared memory limit
    if (smem > smem_granted) {
        if ((err = cudaFuncSetAttribute(nav_kernel<kStep>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem))) !=
            cudaSuccess)
            return err;
        smem_granted = smem;
    }
    int per_sm = 0;
    if ((err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, nav_kernel<kStep>, kNavBlock, smem)) != cudaSuccess)
        return err;
    if (per_sm < 1) per_sm = 1;
    int64_t want = (n + kNavBlock - 1) / kNavBlock;
    int64_t cap = int64_t(sm_count) * per_sm; // persistent: one resident wave, a multiple of the SM count
    unsigned grid = unsigned(want < cap ? want : cap);
    nav_kernel<kStep><<<grid, kNavBlock, smem, s>>>(mother, table_dev, nd, t, step_max, n, out, hit);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return cudaGetLastError();
}

cudaError_t launch_compute_step(const SolidU &mother, const Daughter *table_dev, int nd, const Tracks &t,
                                double step_max, int64_t n, double *step, int32_t *hit, cudaStream_t s)
{
    return launch_nav<true>(mother, table_dev, nd, t, step_max, n, step, hit, s);
}

cudaError_t launch_volume_safety(const SolidU &mother, const Daughter *table_dev, int nd, const Tracks &t, int64_t n,
                                 double *safety, cudaStream_t s)
{
    return launch_nav<false>(mother, table_dev, nd, t, 0.0, n, safety, nullptr, s);
}

} // namespace vg
