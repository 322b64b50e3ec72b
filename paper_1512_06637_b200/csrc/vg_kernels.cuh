// vg_kernels.cuh -- the one streaming kernel every (solid, query) pair instantiates.
//
// Layout: six FP64 SoA arrays in, one array out, each track touched once.
// One thread evaluates TPT = 2 consecutive tracks: every input array is read with one 128-bit
// ld.global.nc.L1::no_allocate per thread (a warp reads 512 contiguous bytes per array), the result leaves as
// one 128-bit (64-bit for Inside) streaming store.  The solid's constants arrive by value in kernel-parameter
// space (`__grid_constant__`), so they are warp-uniform constant-bank operands.  A 64-bit-per-track
// instantiation (TPT = 1) serves arrays that are only 8-byte aligned and the odd tail.
#pragma once
#include "vg_shapes.cuh"

#include <atomic>

namespace vg {

struct Tracks {
    const double *x, *y, *z, *dx, *dy, *dz;
};

#ifndef VG_BLOCK
#define VG_BLOCK 256
#endif
#ifndef VG_MINB
#define VG_MINB 1
#endif
constexpr int kBlock = VG_BLOCK;

extern std::atomic<int64_t> g_launches; // kernel launches made by the library (vg_launch_count)

template <class S, int Q>
VG_DEV void eval_store(const typename S::P &p, double x, double y, double z, double dx, double dy, double dz,
                       double step_max, double &od, int &oi)
{
    if (Q == qInside) {
        oi = S::inside(p, x, y, z);
    } else if (Q == qSafeIn) {
        od = S::safety(p, x, y, z);
    } else if (Q == qSafeOut) {
        od = -S::safety(p, x, y, z);
    } else {
        double t = (Q == qDistIn) ? S::dist_in(p, x, y, z, dx, dy, dz) : S::dist_out(p, x, y, z, dx, dy, dz);
        od = t <= step_max ? t : inf(); // reading R5; -1 passes because step_max >= 0
    }
}

template <class S, int Q, int TPT>
__global__ void __launch_bounds__(kBlock, VG_MINB) query_kernel(const __grid_constant__ typename S::P p, Tracks t,
                                                       double step_max, int64_t n, void *out)
{
    constexpr bool kDir = (Q == qDistIn || Q == qDistOut);
    int64_t i = (int64_t(blockIdx.x) * kBlock + threadIdx.x) * TPT;
    if (i >= n) return;
    if (TPT == 2 && i + 1 < n) {
        double2 x = ldg2(t.x + i), y = ldg2(t.y + i), z = ldg2(t.z + i);
        double2 dx = make_double2(0, 0), dy = dx, dz = dx;
        if (kDir) {
            dx = ldg2(t.dx + i);
            dy = ldg2(t.dy + i);
            dz = ldg2(t.dz + i);
        }
        double d0 = 0, d1 = 0;
        int i0 = 0, i1 = 0;
        eval_store<S, Q>(p, x.x, y.x, z.x, dx.x, dy.x, dz.x, step_max, d0, i0);
        eval_store<S, Q>(p, x.y, y.y, z.y, dx.y, dy.y, dz.y, step_max, d1, i1);
        if (Q == qInside)
            stg2i(static_cast<int32_t *>(out) + i, i0, i1);
        else
            stg2(static_cast<double *>(out) + i, d0, d1);
    } else {
        double x = ldg1(t.x + i), y = ldg1(t.y + i), z = ldg1(t.z + i);
        double dx = 0, dy = 0, dz = 0;
        if (kDir) {
            dx = ldg1(t.dx + i);
            dy = ldg1(t.dy + i);
            dz = ldg1(t.dz + i);
        }
        double d0 = 0;
        int i0 = 0;
        eval_store<S, Q>(p, x, y, z, dx, dy, dz, step_max, d0, i0);
        if (Q == qInside)
            stg1i(static_cast<int32_t *>(out) + i, i0);
        else
            stg1(static_cast<double *>(out) + i, d0);
    }
}

template <class S, int Q>
cudaError_t launch_query(const typename S::P &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                         cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
#ifdef VG_FORCE_TPT1
    vec = false;
#endif
    if (vec) {
        int64_t threads = (n + 1) / 2;
        unsigned grid = unsigned((threads + kBlock - 1) / kBlock);
        query_kernel<S, Q, 2><<<grid, kBlock, 0, stream>>>(p, t, step_max, n, out);
    } else {
        unsigned grid = unsigned((n + kBlock - 1) / kBlock);
        query_kernel<S, Q, 1><<<grid, kBlock, 0, stream>>>(p, t, step_max, n, out);
    }
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return cudaGetLastError();
}

template <class S>
cudaError_t launch_any(int q, const typename S::P &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                       cudaStream_t stream)
{
    switch (q) {
    case qInside: return launch_query<S, qInside>(p, t, step_max, n, out, vec, stream);
    case qDistIn: return launch_query<S, qDistIn>(p, t, step_max, n, out, vec, stream);
    case qDistOut: return launch_query<S, qDistOut>(p, t, step_max, n, out, vec, stream);
    case qSafeIn: return launch_query<S, qSafeIn>(p, t, step_max, n, out, vec, stream);
    case qSafeOut: return launch_query<S, qSafeOut>(p, t, step_max, n, out, vec, stream);
    }
    return cudaErrorInvalidValue;
}

// one translation unit per solid defines these (vg_k_<solid>.cu), so the solids compile in parallel
cudaError_t launch_box(int q, const BoxP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                       cudaStream_t s);
cudaError_t launch_orb(int q, const OrbP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                       cudaStream_t s);
cudaError_t launch_tube(int q, const TubeP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                        cudaStream_t s);
cudaError_t launch_cone(int q, const ConeP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                        cudaStream_t s);
cudaError_t launch_trd(int q, const TrdP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                       cudaStream_t s);
cudaError_t launch_polycone(int q, const PolyconeP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                            cudaStream_t s);

// navigation (vg_nav.cu)
cudaError_t launch_compute_step(const SolidU &mother, const unsigned char *table_dev, const NavMeta &meta, const Tracks &t,
                                double step_max, int64_t n, double *step, int32_t *hit, cudaStream_t s);
cudaError_t launch_volume_safety(const SolidU &mother, const unsigned char *table_dev, const NavMeta &meta, const Tracks &t, int64_t n,
                                 double *safety, cudaStream_t s);

// probes (vg_probe.cu)
cudaError_t probe_fp64_fma_rate(int launches, double *fma_per_s, cudaStream_t s);
cudaError_t probe_empty_launch(int launches, cudaStream_t s);

} // namespace vg
