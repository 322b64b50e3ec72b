// vg_host.cu -- host-buffer entry points: tracks arrive from a host scheduler every step (PAPER.md:61 the
// scheduler hands baskets to the geometry; PAPER.md:122 the GPU only pays off once the transfer is amortised;
// SURVEY.md sec. 8(f) f4).  The arrays are cut into chunks; chunk c uses slot c % kSlots = {a CUDA stream, a
// device staging area}: H2D copies of the six (or three) coordinate arrays, the SAME kernel the device entry
// points launch, D2H copy of the result.  Operations of one slot are ordered by its stream, different slots
// overlap, so that the two copy engines and the SMs work at the same time when the host memory is pinned.
// Staging memory is allocated once per device on first use (never per call).
#include "../../include/vg.h"
#include "vg_kernels.cuh"

#include <cstdio>
#include <mutex>

namespace vg {

constexpr int kSlots = 4;
constexpr int64_t kMaxChunk = int64_t(1) << 20; // tracks per chunk: 8 MiB per coordinate array
constexpr int64_t kMinChunk = int64_t(1) << 16;
constexpr int64_t kBigChunk = int64_t(1) << 19; // the automatic choice stays at or below this
constexpr int kMaxDev = 16;
constexpr int64_t kZeroCopyMax = int64_t(1) << 14; // tracks: up to here a call on pinned memory runs without copies

struct HostPipe {
    bool ready = false;
    cudaStream_t st[kSlots];
    double *in[kSlots];   // 6 * kMaxChunk doubles
    double *outd[kSlots]; // 4 * kMaxChunk doubles (one result; four for the fused five-query call)
    int32_t *outi[kSlots]; // kMaxChunk int32
    std::mutex mu;
};

static HostPipe g_pipe[kMaxDev];

static cudaError_t pipe_slot(HostPipe **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDev) return cudaErrorInvalidDevice;
    *out = &g_pipe[dev];
    return cudaSuccess;
}

// called with p.mu held
static cudaError_t pipe_init(HostPipe &p)
{
    cudaError_t e;
    if (!p.ready) {
        for (int s = 0; s < kSlots; ++s) {
            if ((e = cudaStreamCreateWithFlags(&p.st[s], cudaStreamNonBlocking)) != cudaSuccess) return e;
            if ((e = cudaMalloc(&p.in[s], 6 * kMaxChunk * sizeof(double))) != cudaSuccess) return e;
            if ((e = cudaMalloc(&p.outd[s], 4 * kMaxChunk * sizeof(double))) != cudaSuccess) return e;
            if ((e = cudaMalloc(&p.outi[s], kMaxChunk * sizeof(int32_t))) != cudaSuccess) return e;
        }
        p.ready = true;
    }
    return cudaSuccess;
}

static int64_t pick_chunk(int64_t n)
{
    const int64_t forced = g_host_chunk.load(std::memory_order_relaxed); // vg_set_option(VG_OPT_HOST_CHUNK)
    if (forced > 0) return forced < kMaxChunk ? (forced + 1) / 2 * 2 : kMaxChunk;
    // One chunk per slot, between 64 Ki and 512 Ki tracks: every cudaMemcpyAsync costs ~5 us of engine set-up, so copies
    // under ~2 MB per array leave the link idle (measured, DESIGN.md Appendix A.2: 1 Mi tracks 1.70 ms with 128 Ki
    // chunks, 1.41 ms with 256-512 Ki), while fewer than three chunks cannot overlap H2D with D2H.
    int64_t c = (n + kSlots - 1) / kSlots;
    c = (c + 4095) / 4096 * 4096;
    if (c < kMinChunk) c = kMinChunk;
    if (c > kBigChunk) c = kBigChunk;
    return c;
}

} // namespace vg

using namespace vg;

extern "C" int vg_set_error(int code, const char *msg); // vg_api.cu

static int cuda_fail(cudaError_t e, const char *fn)
{
    char buf[256];
    snprintf(buf, sizeof buf, "%s: %s", fn, cudaGetErrorString(e));
    return vg_set_error(VG_ERR_CUDA, buf);
}

// distance in doubles between consecutive arrays if it is the same for all of them and at least n (no overlap), else 0
static int64_t equal_pitch(const double *const *h, int count, int64_t n)
{
    if (count < 2) return 0;
    const int64_t pitch = h[1] - h[0];
    if (pitch < n) return 0;
    for (int a = 2; a < count; ++a)
        if (h[a] - h[a - 1] != pitch) return 0;
    return pitch;
}

constexpr int qAll = 5; // run_host: the five answers at once, `all` = {cls, dist_in, dist_out, safety_in, safety_out} (HOST, may be NULL)

// shape != NULL: query q of the shape (or all five); volume != NULL: ComputeStep
static int run_host(const char *fn, const vg_shape *shape, const vg_volume *volume, int q, const double *const h[6],
                    double step_max, int64_t n, void *out, int32_t *hit, void *const *all = nullptr)
{
    bool dir = volume || q == qDistIn || q == qDistOut || q == qAll;
    int na = dir ? 6 : 3;
    if (n < 0) return vg_set_error(VG_ERR_ARG, "host entry: n < 0");
    for (int a = 0; a < na; ++a)
        if (!h[a]) return vg_set_error(VG_ERR_ARG, "host entry: NULL track array");
    if (q == qAll) {
        if (!all[0] && !all[1] && !all[2] && !all[3] && !all[4]) return vg_set_error(VG_ERR_ARG, "host entry: every output is NULL");
    } else if (!out || (volume && !hit))
        return vg_set_error(VG_ERR_ARG, "host entry: NULL output array");
    if (n == 0) return VG_OK;
    HostPipe *p = nullptr;
    cudaError_t e = pipe_slot(&p);
    if (e != cudaSuccess) return cuda_fail(e, fn);
    std::lock_guard<std::mutex> lock(p->mu);
    if ((e = pipe_init(*p)) != cudaSuccess) return cuda_fail(e, fn);
    // Small calls on pinned memory skip the copies altogether: pinned host memory is addressable from the device (unified
    // addressing), so the kernel reads the tracks and writes the results straight over the link.  One launch and one
    // synchronisation instead of copy + launch + copy; worth it while the transfer is latency, not bandwidth.
    if (n <= kZeroCopyMax) {
        bool pinned = true;
        const void *ptrs[12] = { h[0], h[1], h[2], dir ? h[3] : nullptr, dir ? h[4] : nullptr, dir ? h[5] : nullptr, out, hit,
                                 all ? all[0] : nullptr, all ? all[1] : nullptr, all ? all[2] : nullptr, all ? all[3] : nullptr };
        const void *last = all ? all[4] : nullptr;
        for (int a = 0; a < 13 && pinned; ++a) {
            const void *q = a < 12 ? ptrs[a] : last;
            if (!q) continue;
            cudaPointerAttributes at;
            if (cudaPointerGetAttributes(&at, q) != cudaSuccess) {
                cudaGetLastError();
                pinned = false;
            } else {
                pinned = at.type == cudaMemoryTypeHost && at.devicePointer == q;
            }
        }
        if (pinned) {
            cudaStream_t st = p->st[0];
            int rc0;
            if (volume) rc0 = vg_compute_step(volume, h[0], h[1], h[2], h[3], h[4], h[5], step_max, n, static_cast<double *>(out), hit, st);
            else if (q == qAll)
                rc0 = vg_query_all(shape, h[0], h[1], h[2], h[3], h[4], h[5], step_max, n, static_cast<int32_t *>(all[0]),
                                   static_cast<double *>(all[1]), static_cast<double *>(all[2]), static_cast<double *>(all[3]),
                                   static_cast<double *>(all[4]), st);
            else if (q == qInside) rc0 = vg_inside(shape, h[0], h[1], h[2], n, static_cast<int32_t *>(out), st);
            else if (q == qDistIn) rc0 = vg_distance_to_in(shape, h[0], h[1], h[2], h[3], h[4], h[5], step_max, n, static_cast<double *>(out), st);
            else if (q == qDistOut) rc0 = vg_distance_to_out(shape, h[0], h[1], h[2], h[3], h[4], h[5], step_max, n, static_cast<double *>(out), st);
            else if (q == qSafeIn) rc0 = vg_safety_to_in(shape, h[0], h[1], h[2], n, static_cast<double *>(out), st);
            else rc0 = vg_safety_to_out(shape, h[0], h[1], h[2], n, static_cast<double *>(out), st);
            if (rc0 != VG_OK) return rc0;
            e = cudaStreamSynchronize(st);
            return e == cudaSuccess ? VG_OK : cuda_fail(e, fn);
        }
    }
    int64_t chunk = pick_chunk(n);
    // Host arrays that sit at one constant distance from each other (rows of one allocation) travel as one 2-D copy per
    // chunk: every copy costs a few microseconds of set-up, which is most of the time of a small call.
    int64_t in_pitch = equal_pitch(h, na, n);
    int64_t out_pitch = 0;
    if (q == qAll && all[1] && all[2] && all[3] && all[4]) {
        const double *od4[4] = { static_cast<double *>(all[1]), static_cast<double *>(all[2]), static_cast<double *>(all[3]),
                                 static_cast<double *>(all[4]) };
        out_pitch = equal_pitch(od4, 4, n);
    }
    int rc = VG_OK;
    int c = 0;
    for (int64_t o = 0; o < n && rc == VG_OK; o += chunk, ++c) {
        int s = c % kSlots;
        int64_t m = n - o < chunk ? n - o : chunk;
        cudaStream_t st = p->st[s];
        double *d[6] = { nullptr, nullptr, nullptr, nullptr, nullptr, nullptr };
        for (int a = 0; a < na; ++a) d[a] = p->in[s] + a * kMaxChunk;
        if (in_pitch > 0) { // equally spaced host arrays (one [6][N] basket): ONE strided copy instead of six
            e = cudaMemcpy2DAsync(d[0], kMaxChunk * sizeof(double), h[0] + o, size_t(in_pitch) * sizeof(double), m * sizeof(double), na,
                                  cudaMemcpyHostToDevice, st);
            if (e == cudaErrorInvalidValue) { // equally spaced but not ONE allocation (the driver refuses the span): six copies
                cudaGetLastError();
                in_pitch = 0;
            } else if (e != cudaSuccess) {
                return cuda_fail(e, fn);
            }
        }
        if (in_pitch == 0) {
            for (int a = 0; a < na; ++a) {
                e = cudaMemcpyAsync(d[a], h[a] + o, m * sizeof(double), cudaMemcpyHostToDevice, st);
                if (e != cudaSuccess) return cuda_fail(e, fn);
            }
        }
        if (volume) {
            rc = vg_compute_step(volume, d[0], d[1], d[2], d[3], d[4], d[5], step_max, m, p->outd[s], p->outi[s], st);
            if (rc != VG_OK) break;
            e = cudaMemcpyAsync(static_cast<double *>(out) + o, p->outd[s], m * sizeof(double), cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(hit + o, p->outi[s], m * sizeof(int32_t), cudaMemcpyDeviceToHost, st);
        } else if (q == qAll) {
            double *od[4];
            for (int a = 0; a < 4; ++a) od[a] = all[a + 1] ? p->outd[s] + a * kMaxChunk : nullptr;
            rc = vg_query_all(shape, d[0], d[1], d[2], d[3], d[4], d[5], step_max, m, all[0] ? p->outi[s] : nullptr, od[0],
                              od[1], od[2], od[3], st);
            if (rc != VG_OK) break;
            if (all[0])
                e = cudaMemcpyAsync(static_cast<int32_t *>(all[0]) + o, p->outi[s], m * sizeof(int32_t), cudaMemcpyDeviceToHost, st);
            if (out_pitch > 0 && e == cudaSuccess) {
                e = cudaMemcpy2DAsync(static_cast<double *>(all[1]) + o, size_t(out_pitch) * sizeof(double), od[0], kMaxChunk * sizeof(double),
                                      m * sizeof(double), 4, cudaMemcpyDeviceToHost, st);
                if (e == cudaErrorInvalidValue) {
                    cudaGetLastError();
                    out_pitch = 0;
                    e = cudaSuccess;
                }
            }
            if (out_pitch == 0) {
                for (int a = 0; a < 4 && e == cudaSuccess; ++a)
                    if (od[a])
                        e = cudaMemcpyAsync(static_cast<double *>(all[a + 1]) + o, od[a], m * sizeof(double), cudaMemcpyDeviceToHost, st);
            }
        } else if (q == qInside) {
            rc = vg_inside(shape, d[0], d[1], d[2], m, p->outi[s], st);
            if (rc != VG_OK) break;
            e = cudaMemcpyAsync(static_cast<int32_t *>(out) + o, p->outi[s], m * sizeof(int32_t), cudaMemcpyDeviceToHost, st);
        } else {
            switch (q) {
            case qDistIn: rc = vg_distance_to_in(shape, d[0], d[1], d[2], d[3], d[4], d[5], step_max, m, p->outd[s], st); break;
            case qDistOut: rc = vg_distance_to_out(shape, d[0], d[1], d[2], d[3], d[4], d[5], step_max, m, p->outd[s], st); break;
            case qSafeIn: rc = vg_safety_to_in(shape, d[0], d[1], d[2], m, p->outd[s], st); break;
            case qSafeOut: rc = vg_safety_to_out(shape, d[0], d[1], d[2], m, p->outd[s], st); break;
            default: rc = vg_set_error(VG_ERR_ARG, "vg_query_host: unknown query");
            }
            if (rc != VG_OK) break;
            e = cudaMemcpyAsync(static_cast<double *>(out) + o, p->outd[s], m * sizeof(double), cudaMemcpyDeviceToHost, st);
        }
        if (e != cudaSuccess) return cuda_fail(e, fn);
    }
    for (int s = 0; s < kSlots && s < c; ++s) { // only the slots this call used
        e = cudaStreamSynchronize(p->st[s]);
        if (e != cudaSuccess && rc == VG_OK) rc = cuda_fail(e, fn);
    }
    return rc;
}

extern "C" int vg_query_host(const vg_shape *shape, int query, const double *x, const double *y, const double *z,
                             const double *dx, const double *dy, const double *dz, double step_max, int64_t n, void *out)
{
    if (!shape) return vg_set_error(VG_ERR_ARG, "vg_query_host: shape is NULL");
    if (query < qInside || query > qSafeOut) return vg_set_error(VG_ERR_ARG, "vg_query_host: unknown query");
    const double *h[6] = { x, y, z, dx, dy, dz };
    return run_host("vg_query_host", shape, nullptr, query, h, step_max, n, out, nullptr);
}

extern "C" int vg_compute_step_host(const vg_volume *volume, const double *x, const double *y, const double *z,
                                    const double *dx, const double *dy, const double *dz, double step_max, int64_t n,
                                    double *step, int32_t *hit)
{
    if (!volume) return vg_set_error(VG_ERR_ARG, "vg_compute_step_host: volume is NULL");
    const double *h[6] = { x, y, z, dx, dy, dz };
    return run_host("vg_compute_step_host", nullptr, volume, -1, h, step_max, n, step, hit);
}

extern "C" int vg_query_all_host(const vg_shape *shape, const double *x, const double *y, const double *z, const double *dx,
                                 const double *dy, const double *dz, double step_max, int64_t n, int32_t *cls,
                                 double *dist_in, double *dist_out, double *safety_in, double *safety_out)
{
    if (!shape) return vg_set_error(VG_ERR_ARG, "vg_query_all_host: shape is NULL");
    const double *h[6] = { x, y, z, dx, dy, dz };
    void *all[5] = { cls, dist_in, dist_out, safety_in, safety_out };
    return run_host("vg_query_all_host", shape, nullptr, qAll, h, step_max, n, nullptr, nullptr, all);
}
