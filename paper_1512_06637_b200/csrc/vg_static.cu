// vg_static.cu -- vg_query_host_static: one query over HOST track arrays that ALLOCATES NOTHING.
//
// Why: vg_query_host (vg_host.cu) stages the tracks in device memory it cudaMallocs on first use, and every other entry
// point wants device arrays the caller allocated.  Some callers cannot allocate: code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc.  Here the staging area is a file-scope __device__ array of a fixed,
// modest size: it is part of the library's device image, so every GPU that loads the library holds it (3.5 MiB) from
// the first use of the library on that GPU until the process exits, whether this entry point is called or not.
//
// Limits and rules (include/vg.h repeats them):
//  * at most VG_STATIC_MAX_TRACKS tracks per call (VG_ERR_PARAM beyond), solids as for vg_query_host;
//  * no cudaMalloc / cudaFree / cudaHostAlloc / stream or event creation: the copies and the kernel go to the CALLER's
//    stream, and the device address of the array is looked up once per device with cudaGetSymbolAddress (in host code
//    the array's name is a host-side stand-in, not a device address);
//  * every call on a device uses the SAME array: two calls that overlap on the GPU (different streams, or threads)
//    race.  Calls are serialised on the host by a lock and each call waits for its own work before it returns, so
//    calls through this entry point cannot overlap each other.  On a stream under CUDA graph capture the call only
//    records its copies and its kernel (it cannot wait): keeping replays apart is then the graph owner's job;
//  * the array keeps the previous call's contents.  Nothing in it has to start at zero: a call overwrites the first n
//    elements of every array its kernel reads and the kernel writes the first n results, which are all that is
//    copied out.
#include "../../include/vg.h"
#include "vg_kernels.cuh"

#include <cstdio>
#include <mutex>

namespace vg {

constexpr int64_t kStaticMax = VG_STATIC_MAX_TRACKS;
constexpr int kStaticArrays = 7; // x, y, z, dx, dy, dz, result (int32 results use the first half of theirs)
constexpr int kStaticMaxDev = 64;

static __device__ __align__(256) double g_static_scratch[kStaticArrays * kStaticMax];

static std::mutex g_static_mu;
static double *g_static_ptr[kStaticMaxDev]; // device address of g_static_scratch on each device, looked up on first use

// with g_static_mu held and the device current
static cudaError_t static_scratch(double **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kStaticMaxDev) return cudaErrorInvalidDevice;
    if (!g_static_ptr[dev]) {
        void *p = nullptr;
        if ((e = cudaGetSymbolAddress(&p, g_static_scratch)) != cudaSuccess) return e;
        g_static_ptr[dev] = static_cast<double *>(p);
    }
    *out = g_static_ptr[dev];
    return cudaSuccess;
}

} // namespace vg

using namespace vg;

extern "C" int vg_set_error(int code, const char *msg); // vg_api.cu

static int static_cuda_fail(cudaError_t e, const char *what)
{
    char buf[256];
    snprintf(buf, sizeof buf, "vg_query_host_static: %s: %s", what, cudaGetErrorString(e));
    return vg_set_error(VG_ERR_CUDA, buf);
}

extern "C" int vg_query_host_static(const vg_shape *shape, int query, const double *x, const double *y, const double *z,
                                    const double *dx, const double *dy, const double *dz, double step_max, int64_t n,
                                    void *out, void *stream)
{
    if (!shape) return vg_set_error(VG_ERR_ARG, "vg_query_host_static: shape is NULL");
    if (query < qInside || query > qSafeOut) return vg_set_error(VG_ERR_ARG, "vg_query_host_static: unknown query");
    if (n < 0) return vg_set_error(VG_ERR_ARG, "vg_query_host_static: n < 0");
    if (n > kStaticMax) {
        char buf[200];
        snprintf(buf, sizeof buf, "vg_query_host_static: n = %lld exceeds VG_STATIC_MAX_TRACKS = %lld (the static staging array); "
                 "split the call or use vg_query_host", (long long)n, (long long)kStaticMax);
        return vg_set_error(VG_ERR_PARAM, buf);
    }
    if (n == 0) return VG_OK; // nothing is read or written: the arrays may be NULL
    const bool dir = query == qDistIn || query == qDistOut;
    const double *h[6] = { x, y, z, dx, dy, dz };
    const int na = dir ? 6 : 3;
    for (int a = 0; a < na; ++a)
        if (!h[a]) return vg_set_error(VG_ERR_ARG, "vg_query_host_static: NULL track array");
    if (!out) return vg_set_error(VG_ERR_ARG, "vg_query_host_static: out is NULL");

    std::lock_guard<std::mutex> lock(g_static_mu);
    double *base = nullptr;
    cudaError_t e = static_scratch(&base);
    if (e != cudaSuccess) return static_cuda_fail(e, "cudaGetSymbolAddress");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    double *d[6];
    for (int a = 0; a < 6; ++a) d[a] = base + a * kStaticMax;
    double *res = base + 6 * kStaticMax;
    int rc = VG_OK;
    for (int a = 0; a < na && rc == VG_OK; ++a)
        if ((e = cudaMemcpyAsync(d[a], h[a], size_t(n) * sizeof(double), cudaMemcpyHostToDevice, st)) != cudaSuccess)
            rc = static_cuda_fail(e, "host -> device copy");
    if (rc == VG_OK) switch (query) { // the same kernels as every other entry point
        case qInside: rc = vg_inside(shape, d[0], d[1], d[2], n, reinterpret_cast<int32_t *>(res), st); break;
        case qDistIn: rc = vg_distance_to_in(shape, d[0], d[1], d[2], d[3], d[4], d[5], step_max, n, res, st); break;
        case qDistOut: rc = vg_distance_to_out(shape, d[0], d[1], d[2], d[3], d[4], d[5], step_max, n, res, st); break;
        case qSafeIn: rc = vg_safety_to_in(shape, d[0], d[1], d[2], n, res, st); break;
        default: rc = vg_safety_to_out(shape, d[0], d[1], d[2], n, res, st); break;
        }
    if (rc == VG_OK) {
        const size_t bytes = size_t(n) * (query == qInside ? sizeof(int32_t) : sizeof(double));
        if ((e = cudaMemcpyAsync(out, res, bytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
            rc = static_cuda_fail(e, "device -> host copy");
    }
    // A stream that is being CAPTURED into a CUDA graph cannot be waited for (and has run nothing yet): the copies and the
    // kernel are now nodes of the caller's graph, which owns the ordering from here on -- replays of such graphs must not
    // overlap each other or a direct call (the array is shared), and the host arrays must be pinned and alive at replay.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) == cudaSuccess && cap == cudaStreamCaptureStatusActive) return rc;
    // otherwise always wait: the array must be free again when the lock is released, also after an error half-way
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess && rc == VG_OK) rc = static_cuda_fail(e, "cudaStreamSynchronize");
    return rc;
}
