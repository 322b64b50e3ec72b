// vg_api.cu -- the C ABI of include/vg.h: handle registry, parameter validation, derived constants
// (SURVEY.md sec. 8(a) A0, sec. 8(b)), argument checks and kernel dispatch.  Host code only; every step of the
// path runs in the kernels of vg_k_*.cu / vg_nav.cu.
#include "../../include/vg.h"
#include "vg_kernels.cuh"
#include "vg_nav_cull.h"

#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

using namespace vg;

struct vg_world;
struct vg_volume {
    SolidU mother;
    NavMeta meta;
    unsigned char *table_dev; // the blob described in vg_params.h
    size_t table_bytes;       // all of it (meta.bytes: the part the kernels stage in shared memory)
    unsigned char *table_host; // its host copy (vg_debug_nav_cull evaluates the cull predicate on the CPU)
    int device;
    vg_world *general;        // mother or a daughter is a polycone / boolean: the volume is held as a one-level world instead
};

static thread_local char g_err[512] = "";

static int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

static int fail_cuda(cudaError_t e, const char *what)
{
    return fail(VG_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

#include "vg_derive.h" // struct vg_shape, fill_shape (uses fail)
#include "vg_pcon_grid.h"

extern "C" const char *vg_last_error(void) { return g_err; }

// for the other host translation units of the library (vg_host.cu)
extern "C" int vg_set_error(int code, const char *msg) { return fail(code, "%s", msg); }

namespace vg {
std::atomic<int64_t> g_launches{ 0 };
std::atomic<int64_t> g_pipe_min_n{ int64_t(1) << 17 };
std::atomic<int64_t> g_pdl{ 1 };
std::atomic<int64_t> g_form{ VG_FORM_AUTO };
std::atomic<int64_t> g_host_chunk{ 0 };
std::atomic<int64_t> g_nav_form{ 0 };
std::atomic<int64_t> g_coop_max_n{ VG_COOP_MAX_N_DEFAULT };
}
extern "C" int64_t vg_launch_count(void) { return vg::g_launches.load(); }

extern "C" int vg_set_option(int option, int64_t value)
{
    switch (option) {
    case VG_OPT_PIPE_MIN_N:
        if (value < 0) return fail(VG_ERR_ARG, "vg_set_option: VG_OPT_PIPE_MIN_N must be >= 0");
        vg::g_pipe_min_n.store(value);
        return VG_OK;
    case VG_OPT_PDL:
        vg::g_pdl.store(value != 0);
        return VG_OK;
    case VG_OPT_HOST_CHUNK:
        if (value < 0) return fail(VG_ERR_ARG, "vg_set_option: VG_OPT_HOST_CHUNK must be >= 0");
        vg::g_host_chunk.store(value);
        return VG_OK;
    case VG_OPT_FORM:
        if (value < VG_FORM_AUTO || value > VG_FORM_STREAMING) return fail(VG_ERR_ARG, "vg_set_option: VG_OPT_FORM must be 0..3");
        vg::g_form.store(value);
        return VG_OK;
    case VG_OPT_NAV_FORM:
        if (value < 0 || value > 2) return fail(VG_ERR_ARG, "vg_set_option: VG_OPT_NAV_FORM must be 0 (auto), 1 (per lane) or 2 (cooperative)");
        vg::g_nav_form.store(value);
        return VG_OK;
    case VG_OPT_COOP_MAX_N:
        if (value < 0) return fail(VG_ERR_ARG, "vg_set_option: VG_OPT_COOP_MAX_N must be >= 0");
        vg::g_coop_max_n.store(value);
        return VG_OK;
    }
    return fail(VG_ERR_ARG, "vg_set_option: unknown option %d", option);
}

extern "C" int64_t vg_get_option(int option)
{
    switch (option) {
    case VG_OPT_PIPE_MIN_N: return vg::g_pipe_min_n.load();
    case VG_OPT_PDL: return vg::g_pdl.load();
    case VG_OPT_FORM: return vg::g_form.load();
    case VG_OPT_HOST_CHUNK: return vg::g_host_chunk.load();
    case VG_OPT_COOP_MAX_N: return vg::g_coop_max_n.load();
    case VG_OPT_NAV_FORM: return vg::g_nav_form.load();
    }
    return fail(VG_ERR_ARG, "vg_get_option: unknown option %d", option);
}

// Builds the candidate grid and puts it on the current device.  Best effort: without a device (or memory) the shape
// is still valid and its safeties run the ordered-walk kernel.
static void upload_pcon_grid(vg_shape *s)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return;
    }
    std::vector<unsigned long long> masks, fmasks;
    std::vector<unsigned char> rows, rows2;
    PconGridGeom geom, geom2;
    pcon_grid_build(s->u.pcon, false, &geom, &masks, &rows);
    if (!s->u.pcon.w.full) pcon_grid_build(s->u.pcon, true, &geom2, &fmasks, &rows2); // same geometry, twice the columns
    const size_t mbytes = masks.size() * sizeof(unsigned long long), fbytes = fmasks.size() * sizeof(unsigned long long);
    // the per-section records of the lanes-per-track kernels (vg_pcon_coop.cuh), in the same allocation
    const PolyconeP &pc = s->u.pcon;
    std::vector<PconCoopSec> coop(pc.nsec);
    for (int k = 0; k < pc.nsec; ++k) {
        const PconSec &c = pc.sec[k];
        PconCoopSec &w = coop[k];
        std::memset(&w, 0, sizeof w);
        w.z0 = c.z0, w.z1 = c.z1, w.Ao = c.out.A, w.Bo = c.out.B, w.Ai = c.in.A, w.Bi = c.in.B, w.seco = c.out.sec, w.seci = c.in.sec;
        w.ro0 = c.out.r0, w.ero = c.out.er, w.ilo = c.out.inv_l2, w.ri0 = c.in.r0, w.eri = c.in.er, w.ili = c.in.inv_l2;
        w.flags = (pc.inner_mask >> k) & 1u;
        if (k + 1 < pc.nsec && ((pc.step_mask >> k) & 1u)) {
            const PconStep &t = pc.step[k];
            w.sz = t.z, w.solo = t.olo, w.sohi = t.ohi, w.silo = t.ilo, w.sihi = t.ihi;
            w.flags |= 2 | (t.oup ? 4 : 0) | (t.iup ? 8 : 0);
        }
    }
    std::vector<PconWalkSec> wtab(pc.nsec); // the ordered walks' records (what pcon_stage builds in shared memory)
    for (int k = 0; k < pc.nsec; ++k) {
        const PconSec &c = pc.sec[k];
        PconWalkSec &w = wtab[k];
        w.z0 = c.z0, w.z1 = c.z1, w.Ao = c.out.A, w.Bo = c.out.B, w.Ai = c.in.A, w.Bi = c.in.B;
        w.ro0 = c.out.r0, w.ero = c.out.er, w.ilo = c.out.inv_l2, w.ri0 = c.in.r0, w.eri = c.in.er, w.ili = c.in.inv_l2;
        w.seco = c.out.sec, w.seci = c.in.sec;
    }
    const size_t wbytes = wtab.size() * sizeof(PconWalkSec);
    std::vector<double> segs(64 * kPconSegStride); // the candidate grids' segment records
    for (int b = 0; b < 64; ++b) pcon_seg_record(pc, b, &segs[size_t(b) * kPconSegStride]);
    const size_t sbytes = segs.size() * sizeof(double);
    const size_t cbytes = coop.size() * sizeof(PconCoopSec), roff = (rows.size() + 15) / 16 * 16;
    unsigned char *blob = nullptr;
    bool ok = cudaMalloc(reinterpret_cast<void **>(&blob), mbytes + fbytes + roff + cbytes + wbytes + sbytes) == cudaSuccess &&
              cudaMemcpy(blob, masks.data(), mbytes, cudaMemcpyHostToDevice) == cudaSuccess &&
              (fbytes == 0 || cudaMemcpy(blob + mbytes, fmasks.data(), fbytes, cudaMemcpyHostToDevice) == cudaSuccess) &&
              cudaMemcpy(blob + mbytes + fbytes, rows.data(), rows.size(), cudaMemcpyHostToDevice) == cudaSuccess &&
              cudaMemcpy(blob + mbytes + fbytes + roff, coop.data(), cbytes, cudaMemcpyHostToDevice) == cudaSuccess &&
              cudaMemcpy(blob + mbytes + fbytes + roff + cbytes, wtab.data(), wbytes, cudaMemcpyHostToDevice) == cudaSuccess &&
              cudaMemcpy(blob + mbytes + fbytes + roff + cbytes + wbytes, segs.data(), sbytes, cudaMemcpyHostToDevice) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        if (blob) cudaFree(blob);
        return;
    }
    s->grid.masks = reinterpret_cast<const unsigned long long *>(blob);
    s->grid.face_masks = fbytes ? reinterpret_cast<const unsigned long long *>(blob + mbytes) : nullptr;
    s->grid.rows = blob + mbytes + fbytes;
    s->grid.coop = reinterpret_cast<const PconCoopSec *>(blob + mbytes + fbytes + roff);
    s->grid.wtab = reinterpret_cast<const PconWalkSec *>(blob + mbytes + fbytes + roff + cbytes);
    s->grid.segs = reinterpret_cast<const double *>(blob + mbytes + fbytes + roff + cbytes + wbytes);
    s->grid.g = geom;
    s->grid_device = dev;
}

extern "C" int vg_shape_create(vg_kind kind, const double *params, int nparams, vg_shape **out)
{
    if (!out) return fail(VG_ERR_ARG, "vg_shape_create: out is NULL");
    *out = nullptr;
    if (!params || nparams <= 0) return fail(VG_ERR_ARG, "vg_shape_create: params is NULL or empty");
    if (!all_finite(params, nparams)) return fail(VG_ERR_PARAM, "vg_shape_create: non-finite parameter");
    vg_shape *s = new (std::nothrow) vg_shape;
    if (!s) return fail(VG_ERR_NOMEM, "vg_shape_create: out of host memory");
    std::memset(s, 0, sizeof *s);
    int rc = fill_shape(s, kind, params, nparams);
    if (rc != VG_OK) {
        delete s;
        return rc;
    }
    if (kind == VG_POLYCONE) upload_pcon_grid(s);
    *out = s;
    return VG_OK;
}

extern "C" void vg_shape_destroy(vg_shape *s)
{
    if (!s) return;
    if (s->grid.masks) cudaFree(const_cast<unsigned long long *>(s->grid.masks)); // rows live in the same allocation
    if (s->ext_blob) cudaFree(s->ext_blob);
    delete[] s->ext_host;
    delete s;
}

extern "C" int vg_shape_kind(const vg_shape *s)
{
    if (!s) return fail(VG_ERR_ARG, "vg_shape_kind: NULL");
    return (s->kind == kCsg || s->kind == kBoolX) ? int(VG_BOOLEAN) : s->kind; // every form of boolean is a boolean to the caller
}

// ------------------------------------------------------------------------------------------------- queries

static bool aligned(const void *p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

static int check_arrays(const char *fn, const void *const *ptrs, int count, size_t out_align, const void *out,
                        int64_t n, bool *vec)
{
    if (n < 0) return fail(VG_ERR_ARG, "%s: n < 0", fn);
    *vec = false;
    if (n == 0) return VG_OK; // nothing is read or written: pointers are not inspected
    bool v = true;
    for (int i = 0; i < count; ++i) {
        if (!ptrs[i]) return fail(VG_ERR_ARG, "%s: NULL track array", fn);
        if (!aligned(ptrs[i], 8)) return fail(VG_ERR_ARG, "%s: track array not 8-byte aligned", fn);
        v = v && aligned(ptrs[i], 16);
    }
    if (!out) return fail(VG_ERR_ARG, "%s: NULL output array", fn);
    if (!aligned(out, out_align)) return fail(VG_ERR_ARG, "%s: output array misaligned", fn);
    v = v && aligned(out, 2 * out_align);
    *vec = v;
    return VG_OK;
}

// a volume / world lives on the device it was created on: a query made while another device is current would hand
// that device foreign pointers
static int check_device(int created_on, const char *fn)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return fail(VG_ERR_CUDA, "%s: no current CUDA device", fn);
    if (dev != created_on) return fail(VG_ERR_ARG, "%s: the handle was created on device %d, the current device is %d", fn, created_on, dev);
    return VG_OK;
}

static int run_query(const char *fn, int q, const vg_shape *s, const double *x, const double *y, const double *z,
                     const double *dx, const double *dy, const double *dz, double step_max, int64_t n, void *out,
                     void *stream)
{
    if (!s) return fail(VG_ERR_ARG, "%s: shape is NULL", fn);
    bool dir = (q == qDistIn || q == qDistOut);
    const void *ptrs[6] = { x, y, z, dx, dy, dz };
    bool vec = false;
    int rc = check_arrays(fn, ptrs, dir ? 6 : 3, q == qInside ? 4 : 8, out, n, &vec);
    if (rc != VG_OK) return rc;
    if (dir && !(step_max >= 0)) return fail(VG_ERR_ARG, "%s: step_max must be >= 0 (may be +inf)", fn);
    if (n == 0) return VG_OK;
    Tracks t{ x, y, z, dx, dy, dz };
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e = cudaErrorInvalidValue;
    switch (s->kind) {
    case VG_BOX: e = launch_box(q, s->u.box, t, step_max, n, out, vec, st); break;
    case VG_ORB: e = launch_orb(q, s->u.orb, t, step_max, n, out, vec, st); break;
    case VG_TUBE: e = launch_tube(q, s->u.tube, t, step_max, n, out, vec, st); break;
    case VG_CONE: e = launch_cone(q, s->u.cone, t, step_max, n, out, vec, st); break;
    case VG_TRD: e = launch_trd(q, s->u.trd, t, step_max, n, out, vec, st); break;
    case VG_POLYCONE: {
        PconGrid g = s->grid;
        int dev = -1;
        if (g.masks && (cudaGetDevice(&dev) != cudaSuccess || dev != s->grid_device)) g.masks = nullptr, g.face_masks = nullptr, g.coop = nullptr, g.wtab = nullptr, g.segs = nullptr;
        e = launch_polycone(q, s->u.pcon, g, t, step_max, n, out, vec, st);
        break;
    }
    case VG_BOOLEAN: e = launch_boolean(q, s->u.boolean, t, step_max, n, out, st, vec); break;
    case kCsg: e = launch_csg(q, s->u.csg, t, step_max, n, out, st); break;
    case kBoolX: {
        int rcd = check_device(s->ext_device, fn);
        if (rcd != VG_OK) return rcd;
        e = launch_boolx(q, s->u.boolean, t, step_max, n, out, st);
        break;
    }
    }
    if (e != cudaSuccess) return fail_cuda(e, fn);
    return VG_OK;
}

extern "C" int vg_inside(const vg_shape *s, const double *x, const double *y, const double *z, int64_t n, int32_t *cls,
                         void *stream)
{
    return run_query("vg_inside", qInside, s, x, y, z, nullptr, nullptr, nullptr, 0.0, n, cls, stream);
}

extern "C" int vg_distance_to_in(const vg_shape *s, const double *x, const double *y, const double *z, const double *dx,
                                 const double *dy, const double *dz, double step_max, int64_t n, double *dist,
                                 void *stream)
{
    return run_query("vg_distance_to_in", qDistIn, s, x, y, z, dx, dy, dz, step_max, n, dist, stream);
}

extern "C" int vg_distance_to_out(const vg_shape *s, const double *x, const double *y, const double *z,
                                  const double *dx, const double *dy, const double *dz, double step_max, int64_t n,
                                  double *dist, void *stream)
{
    return run_query("vg_distance_to_out", qDistOut, s, x, y, z, dx, dy, dz, step_max, n, dist, stream);
}

extern "C" int vg_safety_to_in(const vg_shape *s, const double *x, const double *y, const double *z, int64_t n,
                               double *safety, void *stream)
{
    return run_query("vg_safety_to_in", qSafeIn, s, x, y, z, nullptr, nullptr, nullptr, 0.0, n, safety, stream);
}

extern "C" int vg_safety_to_out(const vg_shape *s, const double *x, const double *y, const double *z, int64_t n,
                                double *safety, void *stream)
{
    return run_query("vg_safety_to_out", qSafeOut, s, x, y, z, nullptr, nullptr, nullptr, 0.0, n, safety, stream);
}

extern "C" int vg_query_all(const vg_shape *s, const double *x, const double *y, const double *z, const double *dx,
                            const double *dy, const double *dz, double step_max, int64_t n, int32_t *cls,
                            double *dist_in, double *dist_out, double *safety_in, double *safety_out, void *stream)
{
    const char *fn = "vg_query_all";
    if (!s) return fail(VG_ERR_ARG, "%s: shape is NULL", fn);
    const bool all = cls && dist_in && dist_out && safety_in && safety_out;
    if (all && s->kind == VG_POLYCONE && n > 0 && step_max >= 0) { // the polycone's fused kernel, when its conditions hold
        const void *ptrs6[6] = { x, y, z, dx, dy, dz };
        bool vec = false, v2 = false;
        int rcp = check_arrays(fn, ptrs6, 6, 4, cls, n, &vec);
        double *outs4[4] = { dist_in, dist_out, safety_in, safety_out };
        for (int i = 0; i < 4 && rcp == VG_OK; ++i) {
            rcp = check_arrays(fn, ptrs6, 6, 8, outs4[i], n, &v2);
            vec = vec && v2;
        }
        if (rcp != VG_OK) return rcp;
        PconGrid g = s->grid;
        int dev = -1;
        if (g.masks && (cudaGetDevice(&dev) != cudaSuccess || dev != s->grid_device)) g.masks = nullptr, g.face_masks = nullptr, g.coop = nullptr, g.wtab = nullptr, g.segs = nullptr;
        Tracks t{ x, y, z, dx, dy, dz };
        AllOut o{ cls, dist_in, dist_out, safety_in, safety_out };
        cudaError_t e = launch_polycone_all(s->u.pcon, g, t, step_max, n, o, vec, static_cast<cudaStream_t>(stream));
        if (e == cudaSuccess) return VG_OK;
        if (e != cudaErrorNotSupported) return fail_cuda(e, fn);
    }
    if (!all || s->kind >= VG_POLYCONE) { // a subset, or no fused kernel for this solid: one launch per requested answer
        if (!cls && !dist_in && !dist_out && !safety_in && !safety_out) return fail(VG_ERR_ARG, "%s: every output is NULL", fn);
        int rc = VG_OK;
        if (cls && rc == VG_OK) rc = vg_inside(s, x, y, z, n, cls, stream);
        if (dist_in && rc == VG_OK) rc = vg_distance_to_in(s, x, y, z, dx, dy, dz, step_max, n, dist_in, stream);
        if (dist_out && rc == VG_OK) rc = vg_distance_to_out(s, x, y, z, dx, dy, dz, step_max, n, dist_out, stream);
        if (safety_in && rc == VG_OK) rc = vg_safety_to_in(s, x, y, z, n, safety_in, stream);
        if (safety_out && rc == VG_OK) rc = vg_safety_to_out(s, x, y, z, n, safety_out, stream);
        return rc;
    }
    const void *ptrs[6] = { x, y, z, dx, dy, dz };
    bool vec = false, v2 = false;
    int rc = check_arrays(fn, ptrs, 6, 4, cls, n, &vec);
    if (rc != VG_OK) return rc;
    double *outs[4] = { dist_in, dist_out, safety_in, safety_out };
    for (int i = 0; i < 4; ++i) {
        if ((rc = check_arrays(fn, ptrs, 6, 8, outs[i], n, &v2)) != VG_OK) return rc;
        vec = vec && v2;
    }
    if (!(step_max >= 0)) return fail(VG_ERR_ARG, "%s: step_max must be >= 0 (may be +inf)", fn);
    if (n == 0) return VG_OK;
    Tracks t{ x, y, z, dx, dy, dz };
    AllOut o{ cls, dist_in, dist_out, safety_in, safety_out };
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e = cudaErrorInvalidValue;
    switch (s->kind) {
    case VG_BOX: e = launch_box_all(s->u.box, t, step_max, n, o, vec, st); break;
    case VG_ORB: e = launch_orb_all(s->u.orb, t, step_max, n, o, vec, st); break;
    case VG_TUBE: e = launch_tube_all(s->u.tube, t, step_max, n, o, vec, st); break;
    case VG_CONE: e = launch_cone_all(s->u.cone, t, step_max, n, o, vec, st); break;
    case VG_TRD: e = launch_trd_all(s->u.trd, t, step_max, n, o, vec, st); break;
    default: break;
    }
    if (e != cudaSuccess) return fail_cuda(e, fn);
    return VG_OK;
}

// ---------------------------------------------------------------------------------------------- navigation

static const WorldTab &world_tab(const vg_world *w); // defined with struct vg_world below

// radius of a sphere about the local origin that contains the solid (phi cuts ignored)
static double bounding_radius(const SolidU &s)
{
    switch (s.kind) {
    case kBox: return std::sqrt(s.u.box.hx * s.u.box.hx + s.u.box.hy * s.u.box.hy + s.u.box.hz * s.u.box.hz);
    case kOrb: return s.u.orb.r;
    case kTube: return std::sqrt(s.u.tube.rmax2 + s.u.tube.dz * s.u.tube.dz);
    case kCone: {
        double r = std::fmax(s.u.cone.rmax1, s.u.cone.rmax2);
        return std::sqrt(r * r + s.u.cone.dz * s.u.cone.dz);
    }
    default: {
        double a = std::fmax(s.u.trd.dx1, s.u.trd.dx2), b = std::fmax(s.u.trd.dy1, s.u.trd.dy2);
        return std::sqrt(a * a + b * b + s.u.trd.dz * s.u.trd.dz);
    }
    }
}

// the same for any vg_shape, polycones and booleans included (world nodes, reading R30)
static double shape_radius(const vg_shape *s)
{
    if (s->kind == VG_POLYCONE) {
        const PolyconeP &c = s->u.pcon;
        double zm = std::fmax(std::fabs(c.zlo), std::fabs(c.zhi));
        return std::sqrt(c.rb2 + zm * zm);
    }
    if (s->kind == kBoolX) { // a polycone operand: its radius from the host copy kept with the shape
        const BoolP &c = s->u.boolean;
        const SolidU *rec[2] = { &c.a, &c.b };
        double r[2];
        for (int o = 0, k = 0; o < 2; ++o) {
            if (rec[o]->kind == kPolycone) {
                const PolyconeP &pc = s->ext_host[k++];
                const double zm = std::fmax(std::fabs(pc.zlo), std::fabs(pc.zhi));
                r[o] = std::sqrt(pc.rb2 + zm * zm);
            } else {
                r[o] = bounding_radius(*rec[o]);
            }
        }
        if (c.op != kUnion) return r[0]; // an intersection and a subtraction lie inside A
        const double *m = c.X;           // centre of B in the frame of C: -R^T b
        const double cx = -(m[0] * m[3] + m[4] * m[7] + m[8] * m[11]), cy = -(m[1] * m[3] + m[5] * m[7] + m[9] * m[11]),
                     cz = -(m[2] * m[3] + m[6] * m[7] + m[10] * m[11]);
        return std::fmax(r[0], std::sqrt(cx * cx + cy * cy + cz * cz) + r[1]);
    }
    if (s->kind == kCsg) { // any tree lies inside the union of its primitives
        const CsgP &c = s->u.csg;
        double r = 0;
        for (int i = 0; i < c.nleaf; ++i) {
            const double *m = c.X[i];
            double cx = -(m[0] * m[3] + m[4] * m[7] + m[8] * m[11]), cy = -(m[1] * m[3] + m[5] * m[7] + m[9] * m[11]),
                   cz = -(m[2] * m[3] + m[6] * m[7] + m[10] * m[11]);
            r = std::fmax(r, std::sqrt(cx * cx + cy * cy + cz * cz) + bounding_radius(c.leaf[i]));
        }
        return r;
    }
    if (s->kind == VG_BOOLEAN) {
        const BoolP &c = s->u.boolean;
        double ra = bounding_radius(c.a);
        if (c.op != kUnion) return ra; // an intersection and a subtraction lie inside A
        const double *m = c.X;         // centre of B in the frame of C: -R^T b
        double cx = -(m[0] * m[3] + m[4] * m[7] + m[8] * m[11]), cy = -(m[1] * m[3] + m[5] * m[7] + m[9] * m[11]),
               cz = -(m[2] * m[3] + m[6] * m[7] + m[10] * m[11]);
        return std::fmax(ra, std::sqrt(cx * cx + cy * cy + cz * cz) + bounding_radius(c.b));
    }
    SolidU u;
    std::memset(&u, 0, sizeof u);
    u.kind = s->kind;
    switch (s->kind) {
    case VG_BOX: u.u.box = s->u.box; break;
    case VG_ORB: u.u.orb = s->u.orb; break;
    case VG_TUBE: u.u.tube = s->u.tube; break;
    case VG_CONE: u.u.cone = s->u.cone; break;
    default: u.u.trd = s->u.trd; break;
    }
    return bounding_radius(u);
}

static int to_solid(const vg_shape *s, SolidU *o, const char *what)
{
    std::memset(o, 0, sizeof *o);
    o->kind = s->kind;
    switch (s->kind) {
    case VG_BOX: o->u.box = s->u.box; return VG_OK;
    case VG_ORB: o->u.orb = s->u.orb; return VG_OK;
    case VG_TUBE: o->u.tube = s->u.tube; return VG_OK;
    case VG_CONE: o->u.cone = s->u.cone; return VG_OK;
    case VG_TRD: o->u.trd = s->u.trd; return VG_OK;
    default: return fail(VG_ERR_ARG, "a polycone or boolean %s is not supported in this build", what);
    }
}

constexpr double kNavDenseCell = 24.0; // measured: pooling pays only where nearly every daughter is a candidate of every ray

// Fills the candidate grid of vg_nav_cull.h for nd bounding spheres (`sph`: cx, cy, cz, r per sphere, in the frame the rays
// are in; r already carries the inflation of the FP32 test): geometry into `gr` (gdim cells per axis over the bounding box
// of the spheres), the cells' masks (ringed layout, `nchunks` 64-bit words per cell, zero-initialised by the caller),
// `prim` (the only sphere of a cell, or -1) and whether the cells list many spheres each.  `r_frame` = radius of the
// sphere about the frame's origin that holds every start point the error bounds are stated for.
static void nav_grid_fill(const std::vector<double> &sph, int nd, int nchunks, int gdim, double r_frame, NavGrid &gr,
                          unsigned long long *cells, int *prim, bool *dense_out)
{
    gr.g[0] = gr.g[1] = gr.g[2] = gdim;
    const unsigned ncell = unsigned((gdim + 2) * (gdim + 2) * (gdim + 2));
    double lo[3] = { 0, 0, 0 }, hi[3] = { 0, 0, 0 };
    for (int i = 0; i < nd; ++i)
        for (int a = 0; a < 3; ++a) {
            double l = sph[4 * i + a] - sph[4 * i + 3], h = sph[4 * i + a] + sph[4 * i + 3];
            lo[a] = i == 0 ? l : std::fmin(lo[a], l);
            hi[a] = i == 0 ? h : std::fmax(hi[a], h);
        }
    double diag = 0;
    for (int a = 0; a < 3; ++a) {
        double ext = hi[a] - lo[a];
        if (!(ext > 0)) ext = 1.0;
        lo[a] -= 1e-6 * ext, ext *= 1.0 + 2e-6;
        gr.o[a] = lo[a], gr.len[a] = ext, gr.cs[a] = ext / gdim, gr.ics[a] = gdim / ext;
        diag += ext * ext;
    }
    diag = std::sqrt(diag);
    const double pad = 1e-6 * (diag + r_frame); // see vg_nav_cull.h: covers the rounding of the walk
    gr.tpad = pad;
    gr.rm2 = r_frame * r_frame * (1.0 + 1e-9);
    for (int i = 0; i < nd; ++i) {
        const double *c = &sph[4 * i];
        const double rr = c[3] * (1.0 + 1e-6) + pad;
        for (int iz = 0; iz < gdim; ++iz)
            for (int iy = 0; iy < gdim; ++iy)
                for (int ix = 0; ix < gdim; ++ix) {
                    const int ic[3] = { ix, iy, iz };
                    double d2 = 0;
                    for (int a = 0; a < 3; ++a) { // distance from the sphere centre to the closed cell
                        double l = gr.o[a] + ic[a] * gr.cs[a], h = l + gr.cs[a];
                        double d = c[a] < l ? l - c[a] : (c[a] > h ? c[a] - h : 0.0);
                        d2 += d * d;
                    }
                    if (d2 <= rr * rr)
                        cells[size_t(((iz + 1) * (gdim + 2) + iy + 1) * (gdim + 2) + ix + 1) * nchunks + i / 64] |= 1ull << (i % 64);
                }
    }
    unsigned singles = 0, filled = 0;
    size_t listed = 0;
    for (unsigned ic = 0; ic < ncell; ++ic) {
        int pc = 0, only = -1;
        for (int c = 0; c < nchunks; ++c) {
            const unsigned long long w = cells[size_t(ic) * nchunks + c];
            pc += __builtin_popcountll(w);
            if (w) only = 64 * c + __builtin_ctzll(w);
        }
        prim[ic] = pc == 1 ? only : -1;
        singles += pc == 1, filled += pc > 0;
        listed += size_t(pc);
    }
    // the fused test pays where nearly every cell the rays cross lists one sphere (configs[4]: all of them); in a mixed
    // grid the lanes of a warp would split over both paths in every step of the walk, so it is switched off there
    if (singles * 10 < filled * 9)
        for (unsigned ic = 0; ic < ncell; ++ic) prim[ic] = -1;
    // mean number of spheres listed per non-empty cell: above kNavDenseCell a ray meets many candidates and the warp
    // pools phase 2 (vg_nav.cu)
    *dense_out = filled && double(listed) / double(filled) > kNavDenseCell;
}

// The safety grid over the box nav_grid_fill laid out (vg_nav_cull.h, nav_safety_cell): gs^3 cells, nchunks mask words
// each.  `bounded[i]`: daughter i is never empty, so |p - c| + r bounds its SafetyToIn from above.
static int nav_safe_dim(int nd)
{
    if (nd < kNavSafeGridMin) return 0;
    // about 512 cells per daughter, at most 32^3: measured at 4 Mi tracks of configs[4] (64 daughters; volume safety /
    // world safety of the 193-node tree), 12^3 cells 242 / 348 us, 16^3 208 / 316, 24^3 193 / 302, 32^3 181 / 293
#ifndef VG_NAV_SAFE_DENSITY
#define VG_NAV_SAFE_DENSITY 512
#endif
    int gs = 4;
    while (gs < kNavSafeGridMax && gs * gs * gs < VG_NAV_SAFE_DENSITY * nd) gs += 4;
    return gs;
}

// half-extents of the axis-aligned bounding box of a solid about its local origin
static void bounding_half(const SolidU &s, double h[3])
{
    switch (s.kind) {
    case kBox: h[0] = s.u.box.hx, h[1] = s.u.box.hy, h[2] = s.u.box.hz; break;
    case kOrb: h[0] = h[1] = h[2] = s.u.orb.r; break;
    case kTube: h[0] = h[1] = std::sqrt(s.u.tube.rmax2), h[2] = s.u.tube.dz; break;
    case kCone: h[0] = h[1] = std::fmax(s.u.cone.rmax1, s.u.cone.rmax2), h[2] = s.u.cone.dz; break;
    default: h[0] = std::fmax(s.u.trd.dx1, s.u.trd.dx2), h[1] = std::fmax(s.u.trd.dy1, s.u.trd.dy2), h[2] = s.u.trd.dz; break;
    }
}

// `fh`: half-extents of the mother's bounding box about its origin (the grid's box, a little larger)
static void nav_safe_grid_fill(const std::vector<double> &sph, const std::vector<char> &bounded, int nd, int nchunks,
                               const double fh[3], NavGrid &gr, unsigned long long *scells)
{
    const int gs = gr.gs;
    double cs[3];
    for (int a = 0; a < 3; ++a) {
        const double h = fh[a] > 0 ? fh[a] * (1.0 + 1e-6) : 1.0;
        gr.so[a] = -h, gr.slen[a] = 2.0 * h, cs[a] = gr.slen[a] / gs, gr.sics[a] = gs / gr.slen[a];
    }
    gr.spad = gr.tpad;
    std::vector<double> dn(nd), df(nd);
    for (int iz = 0; iz < gs; ++iz)
        for (int iy = 0; iy < gs; ++iy)
            for (int ix = 0; ix < gs; ++ix) {
                const int ic[3] = { ix, iy, iz };
                double U = INFINITY;
                long long first = -1; // the daughter that attains U
                for (int i = 0; i < nd; ++i) {
                    const double *c = &sph[4 * i];
                    double n2 = 0, f2 = 0;
                    for (int a = 0; a < 3; ++a) { // nearest and farthest point of the padded closed cell from the centre
                        const double l = gr.so[a] + ic[a] * cs[a] - gr.spad, h = gr.so[a] + (ic[a] + 1) * cs[a] + gr.spad;
                        const double d = c[a] < l ? l - c[a] : (c[a] > h ? c[a] - h : 0.0);
                        const double f = std::fmax(std::fabs(c[a] - l), std::fabs(c[a] - h));
                        n2 += d * d, f2 += f * f;
                    }
                    dn[i] = std::sqrt(n2), df[i] = std::sqrt(f2);
                    if (bounded[i] && df[i] + c[3] < U) U = df[i] + c[3], first = i;
                }
                U = U * (1.0 + 1e-9) + gr.spad;
                unsigned long long *m = scells + size_t((iz * gs + iy) * gs + ix) * size_t(nchunks + 1);
                for (int i = 0; i < nd; ++i)
                    if (dn[i] - sph[4 * i + 3] <= U) m[i / 64] |= 1ull << (i % 64);
                m[nchunks] = first >= 0 ? (unsigned long long)first : ~0ull;
            }
}

// Host side of vg_volume_create for a volume of primitives: validation, the mother and daughter records, the FP32
// bounding spheres and the candidate grid, as one blob in host memory (layout: vg_params.h).  No CUDA call.
// `with_safe` = false leaves the safety grid out (vg_debug_nav_cull for the stages that do not read it).
static int nav_build_host(const vg_shape *mother, int nd, const vg_shape *const *daughters, const double *xforms,
                          vg_volume *v, unsigned char **host_out, bool with_safe = true)
{
    int rc = to_solid(mother, &v->mother, "mother");
    NavMeta &mt = v->meta;
    mt.nd = nd;
    mt.nchunks = (nd + 63) / 64;
    int ndp = (nd + kCullUnroll - 1) / kCullUnroll * kCullUnroll;
    mt.off_d = unsigned(16 * ndp);
    // the candidate grid (vg_nav_cull.h): about one cell per daughter, at most kNavGridMax cells per axis
    int gdim = 1;
    while (gdim < kNavGridMax && gdim * gdim * gdim < nd) ++gdim;
    NavGrid &gr = mt.grid;
    gr.off_g = (mt.off_d + unsigned(nd) * unsigned(kDaughterStride) + 15u) / 16u * 16u;
    const unsigned ncell = unsigned((gdim + 2) * (gdim + 2) * (gdim + 2)); // with a ring of empty cells (vg_nav_cull.h)
    const unsigned nchunks_alloc = mt.nchunks == 3 ? 4u : unsigned(mt.nchunks); // kernels exist for 1, 2 and 4 chunks
    gr.off_p = (gr.off_g + 8u * ncell * (nchunks_alloc ? nchunks_alloc : 1u) + 15u) / 16u * 16u;
    mt.bytes = (gr.off_p + 4u * ncell + 15u) / 16u * 16u;
    if (nchunks_alloc) mt.nchunks = int(nchunks_alloc);
    // the safety grid's masks follow the part of the blob the kernels stage in shared memory (vg_params.h)
    gr.gs = with_safe ? nav_safe_dim(nd) : 0;
    gr.off_s = mt.bytes;
    v->table_bytes = size_t(mt.bytes) + 8u * size_t(gr.gs) * gr.gs * gr.gs * size_t(mt.nchunks + 1); // (+ 1: vg_nav_cull.h)
    std::vector<double> sph; // bounding spheres of the daughters in the mother frame: cx, cy, cz, r (FP64)
    unsigned char *host = nullptr;
    if (rc == VG_OK) {
        host = new (std::nothrow) unsigned char[v->table_bytes];
        if (!host) rc = fail(VG_ERR_NOMEM, "vg_volume_create: out of host memory");
        else std::memset(host, 0, v->table_bytes);
    }
    double r_mother = rc == VG_OK ? bounding_radius(v->mother) : 0.0;
    for (int i = 0; rc == VG_OK && i < ndp; ++i) { // padding entries of the cull table: never hit
        float pad[4] = { 0.f, 0.f, 0.f, -1.f };
        std::memcpy(host + 16 * i, pad, 16);
    }
    for (int i = 0; rc == VG_OK && i < nd; ++i) {
        if (!daughters[i]) {
            rc = fail(VG_ERR_ARG, "vg_volume_create: daughter %d is NULL", i);
            break;
        }
        const double *m = xforms + 12 * i;
        if (!all_finite(m, 12)) {
            rc = fail(VG_ERR_PARAM, "vg_volume_create: non-finite transform of daughter %d", i);
            break;
        }
        for (int r = 0; r < 3 && rc == VG_OK; ++r)
            for (int c = 0; c < 3; ++c) {
                double dot = m[4 * r] * m[4 * c] + m[4 * r + 1] * m[4 * c + 1] + m[4 * r + 2] * m[4 * c + 2];
                if (std::fabs(dot - (r == c ? 1.0 : 0.0)) > 1e-9) {
                    rc = fail(VG_ERR_PARAM, "vg_volume_create: rotation of daughter %d is not orthonormal", i);
                    break;
                }
            }
        if (rc != VG_OK) break;
        Daughter d;
        std::memset(&d, 0, sizeof d);
        std::memcpy(d.m, m, 12 * sizeof(double));
        rc = to_solid(daughters[i], &d.s, "daughter");
        if (rc != VG_OK) break;
        std::memcpy(host + mt.off_d + size_t(i) * kDaughterStride, &d, sizeof d);
        mt.kmask[d.s.kind][i / 64] |= 1ull << (i % 64);
        // bounding sphere in the mother frame: centre c = -R^T b, radius r of the solid about its local origin.
        // The cull runs in FP32; with S >= |c - p| + r for every p in the mother the FP32 evaluation of
        // |c - p|^2 - ((c - p).d)^2 is off by < 30 u S^2 (u = 2^-24), so the squared radius is inflated by
        // 64 u S^2 on top of a relative 1e-6 and rounded UP to float: a daughter the ray can touch is never culled.
        double cx = -(m[0] * m[3] + m[4] * m[7] + m[8] * m[11]);
        double cy = -(m[1] * m[3] + m[5] * m[7] + m[9] * m[11]);
        double cz = -(m[2] * m[3] + m[6] * m[7] + m[10] * m[11]);
        double r = bounding_radius(d.s);
        double S = r_mother + std::sqrt(cx * cx + cy * cy + cz * cz) + r;
        double r2 = r * r * (1.0 + 1e-6) + 64.0 * std::ldexp(1.0, -24) * S * S;
        float e[4] = { float(cx), float(cy), float(cz), std::nextafterf(float(r2), INFINITY) };
        std::memcpy(host + 16 * i, e, 16);
        mt.all[i / 64] |= 1ull << (i % 64);
        sph.insert(sph.end(), { cx, cy, cz, std::sqrt(double(e[3])) });
    }
    if (rc == VG_OK) { // the candidate grid over the bounding box of the spheres (vg_nav_cull.h)
        bool dense = false;
        nav_grid_fill(sph, nd, mt.nchunks, gdim, r_mother, gr, reinterpret_cast<unsigned long long *>(host + gr.off_g),
                      reinterpret_cast<int *>(host + gr.off_p), &dense);
        mt.dense = dense;
        if (gr.gs > 0) // primitives are never empty: every daughter bounds the minimum from above
        {
            double fh[3];
            bounding_half(v->mother, fh);
            nav_safe_grid_fill(sph, std::vector<char>(size_t(nd), 1), nd, mt.nchunks, fh, gr,
                               reinterpret_cast<unsigned long long *>(host + gr.off_s));
        }
    }
    if (rc != VG_OK) {
        delete[] host;
        host = nullptr;
    }
    *host_out = host;
    return rc;
}

extern "C" int vg_volume_create(const vg_shape *mother, int nd, const vg_shape *const *daughters, const double *xforms,
                                vg_volume **out)
{
    if (!out) return fail(VG_ERR_ARG, "vg_volume_create: out is NULL");
    *out = nullptr;
    if (!mother) return fail(VG_ERR_ARG, "vg_volume_create: mother is NULL");
    if (nd < 0 || nd > VG_MAX_DAUGHTERS)
        return fail(VG_ERR_PARAM, "vg_volume_create: ndaughters must be in [0, %d]", VG_MAX_DAUGHTERS);
    if (nd > 0 && (!daughters || !xforms)) return fail(VG_ERR_ARG, "vg_volume_create: NULL daughters or xforms");
    vg_volume *v = new (std::nothrow) vg_volume;
    if (!v) return fail(VG_ERR_NOMEM, "vg_volume_create: out of host memory");
    std::memset(v, 0, sizeof *v);
    bool general = mother->kind >= VG_POLYCONE;
    for (int i = 0; i < nd && !general; ++i) general = daughters[i] && daughters[i]->kind >= VG_POLYCONE;
    if (general) { // polycones / booleans do not fit the fixed-size daughter records: a one-level world serves the volume
        std::vector<const vg_shape *> shapes(1, mother);
        std::vector<int32_t> parent(1, -1);
        std::vector<double> xf = { 1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0 };
        for (int i = 0; i < nd; ++i) {
            shapes.push_back(daughters[i]);
            parent.push_back(0);
            xf.insert(xf.end(), xforms + 12 * i, xforms + 12 * i + 12);
        }
        int rcw = vg_world_create(nd + 1, shapes.data(), parent.data(), xf.data(), &v->general);
        if (rcw != VG_OK) {
            delete v;
            return rcw;
        }
        v->meta.nd = nd;
        *out = v;
        return VG_OK;
    }
    unsigned char *host = nullptr;
    int rc = nav_build_host(mother, nd, daughters, xforms, v, &host);
    NavMeta &mt = v->meta;
    if (rc == VG_OK) {
        cudaError_t e = cudaMalloc(reinterpret_cast<void **>(&v->table_dev), v->table_bytes);
        if (e != cudaSuccess) rc = fail_cuda(e, "vg_volume_create: cudaMalloc");
        if (rc == VG_OK) {
            e = cudaMemcpy(v->table_dev, host, v->table_bytes, cudaMemcpyHostToDevice);
            if (e != cudaSuccess) rc = fail_cuda(e, "vg_volume_create: cudaMemcpy");
        }
    }
    if (rc == VG_OK && cudaGetDevice(&v->device) != cudaSuccess) v->device = -1;
    if (rc != VG_OK) {
        delete[] host;
        if (v->table_dev) cudaFree(v->table_dev);
        delete v;
        return rc;
    }
    v->table_host = host;
    *out = v;
    return VG_OK;
}

extern "C" void vg_volume_destroy(vg_volume *v)
{
    if (!v) return;
    if (v->general) vg_world_destroy(v->general);
    if (v->table_dev) cudaFree(v->table_dev);
    delete[] v->table_host;
    delete v;
}

extern "C" int vg_compute_step(const vg_volume *v, const double *x, const double *y, const double *z, const double *dx,
                               const double *dy, const double *dz, double step_max, int64_t n, double *step,
                               int32_t *hit, void *stream)
{
    const char *fn = "vg_compute_step";
    if (!v) return fail(VG_ERR_ARG, "%s: volume is NULL", fn);
    if (n > 0 && !v->general) {
        int rcd = check_device(v->device, fn);
        if (rcd != VG_OK) return rcd;
    }
    const void *ptrs[6] = { x, y, z, dx, dy, dz };
    bool vec = false;
    int rc = check_arrays(fn, ptrs, 6, 8, step, n, &vec);
    if (rc != VG_OK) return rc;
    if (n == 0) return VG_OK;
    if (!hit || !aligned(hit, 4)) return fail(VG_ERR_ARG, "%s: hit array NULL or misaligned", fn);
    if (!(step_max >= 0)) return fail(VG_ERR_ARG, "%s: step_max must be >= 0 (may be +inf)", fn);
    Tracks t{ x, y, z, dx, dy, dz };
    cudaError_t e = v->general ? launch_world_step(world_tab(v->general), nullptr, t, step_max, n, step, hit, static_cast<cudaStream_t>(stream))
                               : launch_compute_step(v->mother, v->table_dev, v->meta, t, step_max, n, step, hit,
                                                     static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, fn);
    return VG_OK;
}

extern "C" int vg_volume_safety(const vg_volume *v, const double *x, const double *y, const double *z, int64_t n,
                                double *safety, void *stream)
{
    const char *fn = "vg_volume_safety";
    if (!v) return fail(VG_ERR_ARG, "%s: volume is NULL", fn);
    if (n > 0 && !v->general) {
        int rcd = check_device(v->device, fn);
        if (rcd != VG_OK) return rcd;
    }
    const void *ptrs[3] = { x, y, z };
    bool vec = false;
    int rc = check_arrays(fn, ptrs, 3, 8, safety, n, &vec);
    if (rc != VG_OK) return rc;
    if (n == 0) return VG_OK;
    Tracks t{ x, y, z, nullptr, nullptr, nullptr };
    cudaError_t e = v->general ? launch_world_safety(world_tab(v->general), nullptr, t, n, safety, static_cast<cudaStream_t>(stream))
                               : launch_volume_safety(v->mother, v->table_dev, v->meta, t, n, safety, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, fn);
    return VG_OK;
}

// ------------------------------------------------------------------------------------- hierarchy of volumes

struct vg_world {
    int nn;
    WorldTab tab;          // device pointers into ONE allocation: node records, FP32 cull spheres, child lists, then the
    unsigned char *blob;   // polycone and boolean constants of the nodes that are not primitives (reading R30)
    int device;
};

static const WorldTab &world_tab(const vg_world *w) { return w->tab; }

static bool rigid(const double *m)
{
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) {
            double dot = m[4 * r] * m[4 * c] + m[4 * r + 1] * m[4 * c + 1] + m[4 * r + 2] * m[4 * c + 2];
            if (std::fabs(dot - (r == c ? 1.0 : 0.0)) > 1e-9) return false;
        }
    return true;
}

// C = A o B for row-major 3x4 [R | b]: first B, then A
static void compose(const double *A, const double *B, double *C)
{
    for (int r = 0; r < 3; ++r) {
        for (int c = 0; c < 3; ++c) C[4 * r + c] = A[4 * r] * B[c] + A[4 * r + 1] * B[4 + c] + A[4 * r + 2] * B[8 + c];
        C[4 * r + 3] = A[4 * r] * B[3] + A[4 * r + 1] * B[7] + A[4 * r + 2] * B[11] + A[4 * r + 3];
    }
}

// --------------------------------------------------------------------------------------------- boolean solids

// an operand as a list of primitives with their transforms (frame of the operand -> frame of the primitive) and a postfix
// program over them (vg_params.h CsgP)
struct CsgOperand {
    int nleaf = 0, nprog = 0;
    SolidU leaf[kCsgMaxLeaf];
    double X[kCsgMaxLeaf][12];
    unsigned char prog[kCsgMaxProg];
};

static const double kIdentity12[12] = { 1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0 };

static int csg_operand(const vg_shape *s, CsgOperand *o)
{
    if (s->kind == kCsg) {
        const CsgP &c = s->u.csg;
        o->nleaf = c.nleaf, o->nprog = c.nprog;
        std::memcpy(o->leaf, c.leaf, sizeof o->leaf);
        std::memcpy(o->X, c.X, sizeof o->X);
        std::memcpy(o->prog, c.prog, sizeof o->prog);
        return VG_OK;
    }
    if (s->kind == VG_BOOLEAN) {
        const BoolP &c = s->u.boolean;
        o->nleaf = 2, o->nprog = 3;
        o->leaf[0] = c.a, o->leaf[1] = c.b;
        std::memcpy(o->X[0], kIdentity12, sizeof kIdentity12);
        std::memcpy(o->X[1], c.X, sizeof c.X);
        o->prog[0] = 0, o->prog[1] = 1, o->prog[2] = (unsigned char)(0x80 | c.op);
        return VG_OK;
    }
    o->nleaf = 1, o->nprog = 1;
    std::memcpy(o->X[0], kIdentity12, sizeof kIdentity12);
    o->prog[0] = 0;
    return to_solid(s, &o->leaf[0], "operand");
}

extern "C" int vg_boolean_create(int op, const vg_shape *a, const vg_shape *b, const double *xform_b, vg_shape **out)
{
    const char *fn = "vg_boolean_create";
    if (!out) return fail(VG_ERR_ARG, "%s: out is NULL", fn);
    *out = nullptr;
    if (op < VG_UNION || op > VG_SUBTRACTION) return fail(VG_ERR_PARAM, "%s: op must be VG_UNION, VG_INTERSECTION or VG_SUBTRACTION", fn);
    if (!a || !b || !xform_b) return fail(VG_ERR_ARG, "%s: NULL operand or transform", fn);
    if (!all_finite(xform_b, 12)) return fail(VG_ERR_PARAM, "%s: non-finite transform", fn);
    if (!rigid(xform_b)) return fail(VG_ERR_PARAM, "%s: the rotation of B is not orthonormal", fn);
    vg_shape *s = new (std::nothrow) vg_shape;
    if (!s) return fail(VG_ERR_NOMEM, "%s: out of host memory", fn);
    std::memset(s, 0, sizeof *s);
    int rc = VG_OK;
    if ((a->kind == VG_POLYCONE && b->kind <= VG_POLYCONE) || (b->kind == VG_POLYCONE && a->kind <= VG_POLYCONE)) {
        // a polycone operand (vg_boolx.cu): its constants go to device memory, the operand record points at them
        s->kind = kBoolX;
        BoolP &c = s->u.boolean;
        c.op = op;
        std::memcpy(c.X, xform_b, sizeof c.X);
        const vg_shape *opnd[2] = { a, b };
        SolidU *rec[2] = { &c.a, &c.b };
        const int npc = (a->kind == VG_POLYCONE) + (b->kind == VG_POLYCONE);
        PolyconeP *blob = nullptr;
        cudaError_t e = cudaGetDevice(&s->ext_device);
        if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void **>(&blob), size_t(npc) * sizeof(PolyconeP));
        if (e != cudaSuccess) rc = fail_cuda(e, "vg_boolean_create: a polycone operand needs device memory");
        s->ext_blob = blob;
        s->ext_host = new (std::nothrow) PolyconeP[2];
        if (!s->ext_host && rc == VG_OK) rc = fail(VG_ERR_NOMEM, "vg_boolean_create: out of host memory");
        for (int i = 0, k = 0; i < 2 && rc == VG_OK; ++i) {
            if (opnd[i]->kind == VG_POLYCONE) {
                e = cudaMemcpy(blob + k, &opnd[i]->u.pcon, sizeof(PolyconeP), cudaMemcpyHostToDevice);
                if (e != cudaSuccess) rc = fail_cuda(e, "vg_boolean_create: cudaMemcpy");
                s->ext_host[k] = opnd[i]->u.pcon;
                rec[i]->kind = kPolycone;
                rec[i]->u.pcon = blob + k++;
            } else {
                rc = to_solid(opnd[i], rec[i], "operand");
            }
        }
        if (rc != VG_OK && blob) cudaFree(blob);
        if (rc != VG_OK) delete[] s->ext_host;
    } else if (a->kind == kBoolX || b->kind == kBoolX || a->kind == VG_POLYCONE || b->kind == VG_POLYCONE) {
        rc = fail(VG_ERR_ARG, "%s: a polycone may be an operand of a boolean of two solids, not a leaf of a nested tree", fn);
    } else if (a->kind < VG_POLYCONE && b->kind < VG_POLYCONE) { // two primitives: the specialised kernels of vg_bool.cu
        s->kind = VG_BOOLEAN;
        BoolP &c = s->u.boolean;
        c.op = op;
        std::memcpy(c.X, xform_b, sizeof c.X);
        rc = to_solid(a, &c.a, "operand");
        if (rc == VG_OK) rc = to_solid(b, &c.b, "operand");
    } else { // an operand is a boolean (reading R31): flatten the tree
        CsgOperand oa, ob;
        rc = csg_operand(a, &oa);
        if (rc == VG_OK) rc = csg_operand(b, &ob);
        if (rc == VG_OK && oa.nleaf + ob.nleaf > kCsgMaxLeaf)
            rc = fail(VG_ERR_PARAM, "%s: more than %d primitives in the tree", fn, kCsgMaxLeaf);
        if (rc == VG_OK) {
            s->kind = kCsg;
            CsgP &c = s->u.csg;
            c.nleaf = oa.nleaf + ob.nleaf;
            for (int i = 0; i < oa.nleaf; ++i) {
                c.leaf[i] = oa.leaf[i];
                std::memcpy(c.X[i], oa.X[i], sizeof c.X[i]);
            }
            for (int i = 0; i < ob.nleaf; ++i) { // frame of the tree -> frame of B -> frame of the primitive
                c.leaf[oa.nleaf + i] = ob.leaf[i];
                compose(ob.X[i], xform_b, c.X[oa.nleaf + i]);
            }
            int k = 0;
            for (int i = 0; i < oa.nprog; ++i) c.prog[k++] = oa.prog[i];
            for (int i = 0; i < ob.nprog; ++i) c.prog[k++] = ob.prog[i] < 0x80 ? (unsigned char)(ob.prog[i] + oa.nleaf) : ob.prog[i];
            c.prog[k++] = (unsigned char)(0x80 | op);
            c.nprog = k;
        }
    }
    if (rc != VG_OK) {
        delete s;
        return rc;
    }
    *out = s;
    return VG_OK;
}

extern "C" int vg_world_create(int nn, const vg_shape *const *shapes, const int32_t *parent, const double *xforms,
                               vg_world **out)
{
    const char *fn = "vg_world_create";
    if (!out) return fail(VG_ERR_ARG, "%s: out is NULL", fn);
    *out = nullptr;
    if (nn < 1 || nn > VG_MAX_NODES) return fail(VG_ERR_PARAM, "%s: nnodes must be in [1, %d]", fn, VG_MAX_NODES);
    if (!shapes || !parent || !xforms) return fail(VG_ERR_ARG, "%s: NULL shapes, parent or xforms", fn);
    if (parent[0] != -1) return fail(VG_ERR_PARAM, "%s: node 0 is the root, parent[0] must be -1", fn);
    std::vector<WorldNode> nodes(nn);
    std::vector<int32_t> kids(nn > 1 ? nn - 1 : 1, 0);
    std::vector<int> count(nn, 0), fill(nn, 0);
    std::vector<PolyconeP> pcons;
    std::vector<BoolP> bools;
    std::vector<int> boolx; // entries of `bools` whose polycone operands still hold an index into `pcons`
    std::vector<CsgP> csgs;
    std::vector<double> radius(nn, 0.0);
    for (int i = 1; i < nn; ++i) {
        if (parent[i] < 0 || parent[i] >= i) return fail(VG_ERR_PARAM, "%s: need 0 <= parent[%d] < %d", fn, i, i);
        if (++count[parent[i]] > VG_MAX_DAUGHTERS)
            return fail(VG_ERR_PARAM, "%s: node %d has more than %d children", fn, parent[i], VG_MAX_DAUGHTERS);
    }
    for (int i = 0, off = 0; i < nn; ++i) {
        WorldNode &N = nodes[i];
        std::memset(&N, 0, sizeof N);
        if (!shapes[i]) return fail(VG_ERR_ARG, "%s: shape %d is NULL", fn, i);
        const double *m = xforms + 12 * i;
        if (!all_finite(m, 12)) return fail(VG_ERR_PARAM, "%s: non-finite transform of node %d", fn, i);
        if (!rigid(m)) return fail(VG_ERR_PARAM, "%s: rotation of node %d is not orthonormal", fn, i);
        if (shapes[i]->kind == kBoolX) { // a boolean with polycone operands: its polycones join the world's side array
            N.s.kind = kBoolX;
            N.ext = int(bools.size());
            BoolP b = shapes[i]->u.boolean;
            SolidU *rec[2] = { &b.a, &b.b };
            for (int o = 0, k = 0; o < 2; ++o)
                if (rec[o]->kind == kPolycone) {
                    // the index for now; becomes the device address once the world's blob exists (below)
                    rec[o]->u.pcon = reinterpret_cast<const PolyconeP *>(uintptr_t(pcons.size()));
                    pcons.push_back(shapes[i]->ext_host[k++]);
                }
            bools.push_back(b);
            boolx.push_back(int(bools.size()) - 1);
        } else if (shapes[i]->kind == VG_POLYCONE) { // R30: constants in a side array, the record keeps kind + index
            N.s.kind = kPolycone;
            N.ext = int(pcons.size());
            pcons.push_back(shapes[i]->u.pcon);
        } else if (shapes[i]->kind == VG_BOOLEAN) {
            N.s.kind = kBoolean;
            N.ext = int(bools.size());
            bools.push_back(shapes[i]->u.boolean);
        } else if (shapes[i]->kind == kCsg) {
            N.s.kind = kCsg;
            N.ext = int(csgs.size());
            csgs.push_back(shapes[i]->u.csg);
        } else {
            int rc = to_solid(shapes[i], &N.s, "node");
            if (rc != VG_OK) return rc;
        }
        radius[i] = shape_radius(shapes[i]);
        std::memcpy(N.X, m, sizeof N.X);
        if (i == 0) std::memcpy(N.G, m, sizeof N.G);
        else compose(m, nodes[parent[i]].G, N.G);
        N.parent = parent[i];
        N.child0 = off;
        N.nchild = count[i];
        off += count[i];
        if (i > 0) kids[nodes[parent[i]].child0 + fill[parent[i]]++] = i; // ascending i: lists come out sorted
    }
    for (int i = 0; i < nn; ++i) {
        // bounding sphere in the parent's frame: centre c = -R^T b.  The tests evaluate |p - c|^2 (- (v.d)^2) in FP64 with
        // |p - c| <= S = (parent's radius) + |c| + r: rounding error < 16 u S^2 (u = 2^-53); inflate well beyond it.
        WorldNode &N = nodes[i];
        const double *m = N.X;
        double cx = -(m[0] * m[3] + m[4] * m[7] + m[8] * m[11]);
        double cy = -(m[1] * m[3] + m[5] * m[7] + m[9] * m[11]);
        double cz = -(m[2] * m[3] + m[6] * m[7] + m[10] * m[11]);
        double r = radius[i];
        double rp = i > 0 ? radius[parent[i]] : r;
        double S = rp + std::sqrt(cx * cx + cy * cy + cz * cz) + r;
        N.bs[0] = cx, N.bs[1] = cy, N.bs[2] = cz;
        N.bs[3] = r * r * (1.0 + 1e-9) + 1e-12 * S * S;
        N.br = std::sqrt(N.bs[3]);
    }
    // the same spheres for the FP32 culls of Locate and Step, in child-list order; error bound as in vg_volume_create:
    // the FP32 evaluation is off by < 30 u S^2 (u = 2^-24), so r^2 is inflated by 64 u S^2 on top of a relative 1e-6
    std::vector<float> cull(4 * kids.size(), 0.f);
    for (int p = 0; p < nn; ++p)
        for (int j = 0; j < nodes[p].nchild; ++j) {
            const WorldNode &N = nodes[kids[nodes[p].child0 + j]];
            const double r = radius[kids[nodes[p].child0 + j]];
            const double S = radius[p] + std::sqrt(N.bs[0] * N.bs[0] + N.bs[1] * N.bs[1] + N.bs[2] * N.bs[2]) + r;
            const double r2 = r * r * (1.0 + 1e-6) + 64.0 * std::ldexp(1.0, -24) * S * S;
            float *e = &cull[4 * size_t(nodes[p].child0 + j)];
            e[0] = float(N.bs[0]), e[1] = float(N.bs[1]), e[2] = float(N.bs[2]), e[3] = std::nextafterf(float(r2), INFINITY);
        }
    // candidate grids (vg_nav_cull.h) for the nodes with many children: Step walks the grid along the ray, Locate looks up
    // the point's cell, instead of testing the bounding sphere of every child
    std::vector<WorldGrid> grids;
    std::vector<unsigned long long> gcells;
    std::vector<int> gprim;
    for (int p = 0; p < nn; ++p) {
        WorldNode &P = nodes[p];
        P.grid = -1;
        if (P.nchild < kWorldGridMin || P.nchild > 64) continue;
        std::vector<double> sph;
        for (int j = 0; j < P.nchild; ++j) {
            const WorldNode &C = nodes[kids[P.child0 + j]];
            sph.insert(sph.end(), { C.bs[0], C.bs[1], C.bs[2], std::sqrt(double(cull[4 * size_t(P.child0 + j) + 3])) });
        }
        int gdim = 1;
        while (gdim < kNavGridMax && gdim * gdim * gdim < P.nchild) ++gdim;
        const size_t ncell = size_t(gdim + 2) * (gdim + 2) * (gdim + 2);
        WorldGrid wg;
        std::memset(&wg, 0, sizeof wg);
        wg.cells0 = unsigned(gcells.size()), wg.prim0 = unsigned(gprim.size());
        wg.all = P.nchild == 64 ? ~0ull : ((1ull << P.nchild) - 1ull);
        gcells.resize(gcells.size() + ncell, 0ull);
        gprim.resize(gprim.size() + ncell, -1);
        bool dense = false;
        nav_grid_fill(sph, P.nchild, 1, gdim, radius[p], wg.g, gcells.data() + wg.cells0, gprim.data() + wg.prim0, &dense);
        // the safety grid (nav_safety_cell): a boolean can be empty, so only the other kinds bound the minimum from above
        wg.g.gs = nav_safe_dim(P.nchild);
        wg.g.off_s = unsigned(gcells.size());
        if (wg.g.gs > 0) {
            std::vector<char> bounded;
            for (int j = 0; j < P.nchild; ++j) bounded.push_back(shapes[kids[P.child0 + j]]->kind < VG_BOOLEAN); // (a tree or a polycone-operand boolean: kind > VG_BOOLEAN)
            gcells.resize(gcells.size() + 2 * size_t(wg.g.gs) * wg.g.gs * wg.g.gs, 0ull); // a mask and the first child per cell
            double fh[3] = { radius[p], radius[p], radius[p] }; // a polycone or boolean node: the cube about its sphere
            if (P.s.kind < kPolycone) bounding_half(P.s, fh);
            nav_safe_grid_fill(sph, bounded, P.nchild, 1, fh, wg.g, gcells.data() + wg.g.off_s);
        }
        P.grid = int(grids.size());
        grids.push_back(wg);
    }
    vg_world *w = new (std::nothrow) vg_world;
    if (!w) return fail(VG_ERR_NOMEM, "%s: out of host memory", fn);
    std::memset(w, 0, sizeof *w);
    w->nn = nn;
    auto up16 = [](size_t v) { return (v + 15) / 16 * 16; };
    const size_t wgbytes = up16(grids.size() * sizeof(WorldGrid)), gcbytes = up16(gcells.size() * sizeof(unsigned long long)),
                 gpbytes = up16(gprim.size() * sizeof(int));
    const size_t nbytes = size_t(nn) * sizeof(WorldNode), cbytes = cull.size() * sizeof(float), kbytes = up16(kids.size() * sizeof(int32_t));
    const size_t pbytes = up16(pcons.size() * sizeof(PolyconeP)), bbytes = up16(bools.size() * sizeof(BoolP)), gbytes = csgs.size() * sizeof(CsgP);
    static_assert(sizeof(WorldNode) % 16 == 0, "the float4 array follows the node records");
    unsigned char *blob = nullptr;
    cudaError_t e = cudaGetDevice(&w->device);
    const size_t goff = up16(nbytes + cbytes + kbytes + pbytes + bbytes + gbytes); // the grids follow everything else
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void **>(&blob), goff + wgbytes + gcbytes + gpbytes + 16);
    if (e == cudaSuccess) e = cudaMemcpy(blob, nodes.data(), nbytes, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(blob + nbytes, cull.data(), cbytes, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(blob + nbytes + cbytes, kids.data(), kids.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && !pcons.empty())
        e = cudaMemcpy(blob + nbytes + cbytes + kbytes, pcons.data(), pcons.size() * sizeof(PolyconeP), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) { // polycone operands of boolean nodes: index -> address in this world's polycone array
        const PolyconeP *pc0 = reinterpret_cast<const PolyconeP *>(blob + nbytes + cbytes + kbytes);
        for (int k : boolx) {
            SolidU *rec[2] = { &bools[k].a, &bools[k].b };
            for (int o = 0; o < 2; ++o)
                if (rec[o]->kind == kPolycone) rec[o]->u.pcon = pc0 + reinterpret_cast<uintptr_t>(rec[o]->u.pcon);
        }
    }
    if (e == cudaSuccess && !bools.empty())
        e = cudaMemcpy(blob + nbytes + cbytes + kbytes + pbytes, bools.data(), bools.size() * sizeof(BoolP), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && !csgs.empty())
        e = cudaMemcpy(blob + nbytes + cbytes + kbytes + pbytes + bbytes, csgs.data(), gbytes, cudaMemcpyHostToDevice);
    if (e == cudaSuccess && !grids.empty()) {
        e = cudaMemcpy(blob + goff, grids.data(), grids.size() * sizeof(WorldGrid), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(blob + goff + wgbytes, gcells.data(), gcells.size() * sizeof(unsigned long long), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(blob + goff + wgbytes + gcbytes, gprim.data(), gprim.size() * sizeof(int), cudaMemcpyHostToDevice);
    }
    if (e != cudaSuccess) {
        if (blob) cudaFree(blob);
        delete w;
        return fail_cuda(e, fn);
    }
    w->blob = blob;
    w->tab.grids = reinterpret_cast<WorldGrid *>(blob + goff);
    w->tab.gcells = reinterpret_cast<unsigned long long *>(blob + goff + wgbytes);
    w->tab.gprim = reinterpret_cast<int *>(blob + goff + wgbytes + gcbytes);
    w->tab.nodes = reinterpret_cast<WorldNode *>(blob);
    w->tab.cull = reinterpret_cast<float4 *>(blob + nbytes);
    w->tab.kids = reinterpret_cast<int32_t *>(blob + nbytes + cbytes);
    w->tab.pcons = reinterpret_cast<PolyconeP *>(blob + nbytes + cbytes + kbytes);
    w->tab.bools = reinterpret_cast<BoolP *>(blob + nbytes + cbytes + kbytes + pbytes);
    w->tab.csgs = reinterpret_cast<CsgP *>(blob + nbytes + cbytes + kbytes + pbytes + bbytes);
    w->tab.nnodes = nn;
    w->tab.has_ext = !(pcons.empty() && bools.empty() && csgs.empty());
    *out = w;
    return VG_OK;
}

extern "C" void vg_world_destroy(vg_world *w)
{
    if (!w) return;
    if (w->blob) cudaFree(w->blob);
    delete w;
}

extern "C" int vg_world_locate(const vg_world *w, const double *x, const double *y, const double *z, int64_t n,
                               int32_t *node, void *stream)
{
    const char *fn = "vg_world_locate";
    if (!w) return fail(VG_ERR_ARG, "%s: world is NULL", fn);
    if (n > 0) {
        int rcd = check_device(w->device, fn);
        if (rcd != VG_OK) return rcd;
    }
    const void *ptrs[3] = { x, y, z };
    bool vec = false;
    int rc = check_arrays(fn, ptrs, 3, 4, node, n, &vec);
    if (rc != VG_OK || n == 0) return rc;
    Tracks t{ x, y, z, nullptr, nullptr, nullptr };
    cudaError_t e = launch_world_locate(w->tab, t, n, node, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, fn);
    return VG_OK;
}

extern "C" int vg_world_step(const vg_world *w, const int32_t *node, const double *x, const double *y, const double *z,
                             const double *dx, const double *dy, const double *dz, double step_max, int64_t n,
                             double *step, int32_t *next, void *stream)
{
    const char *fn = "vg_world_step";
    if (!w) return fail(VG_ERR_ARG, "%s: world is NULL", fn);
    if (n > 0) {
        int rcd = check_device(w->device, fn);
        if (rcd != VG_OK) return rcd;
    }
    const void *ptrs[6] = { x, y, z, dx, dy, dz };
    bool vec = false;
    int rc = check_arrays(fn, ptrs, 6, 8, step, n, &vec);
    if (rc != VG_OK || n == 0) return rc;
    if (!node || !aligned(node, 4) || !next || !aligned(next, 4)) return fail(VG_ERR_ARG, "%s: node / next array NULL or misaligned", fn);
    if (!(step_max >= 0)) return fail(VG_ERR_ARG, "%s: step_max must be >= 0 (may be +inf)", fn);
    Tracks t{ x, y, z, dx, dy, dz };
    cudaError_t e = launch_world_step(w->tab, node, t, step_max, n, step, next,
                                      static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, fn);
    return VG_OK;
}

extern "C" int vg_world_safety(const vg_world *w, const int32_t *node, const double *x, const double *y, const double *z,
                               int64_t n, double *safety, void *stream)
{
    const char *fn = "vg_world_safety";
    if (!w) return fail(VG_ERR_ARG, "%s: world is NULL", fn);
    if (n > 0) {
        int rcd = check_device(w->device, fn);
        if (rcd != VG_OK) return rcd;
    }
    const void *ptrs[3] = { x, y, z };
    bool vec = false;
    int rc = check_arrays(fn, ptrs, 3, 8, safety, n, &vec);
    if (rc != VG_OK || n == 0) return rc;
    if (!node || !aligned(node, 4)) return fail(VG_ERR_ARG, "%s: node array NULL or misaligned", fn);
    Tracks t{ x, y, z, nullptr, nullptr, nullptr };
    cudaError_t e = launch_world_safety(w->tab, node, t, n, safety, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, fn);
    return VG_OK;
}

extern "C" int vg_debug_nav_cull(const vg_shape *mother, int nd, const vg_shape *const *daughters, const double *xforms,
                                 const double *x, const double *y, const double *z, const double *dx, const double *dy,
                                 const double *dz, const double *t_lim, int64_t n, uint64_t *masks, int stage,
                                 double *grid)
{
    const char *fn = "vg_debug_nav_cull";
    if (!mother || nd < 1 || nd > VG_MAX_DAUGHTERS || !daughters || !xforms || !x || !y || !z || !dx || !dy || !dz || !masks || n < 0)
        return fail(VG_ERR_ARG, "%s: bad argument", fn);
    if (mother->kind >= VG_POLYCONE) return fail(VG_ERR_ARG, "%s: the mother must be a primitive", fn);
    for (int i = 0; i < nd; ++i)
        if (!daughters[i] || daughters[i]->kind >= VG_POLYCONE) return fail(VG_ERR_ARG, "%s: daughter %d is not a primitive", fn, i);
    vg_volume v;
    std::memset(&v, 0, sizeof v);
    unsigned char *host = nullptr;
    int rc = nav_build_host(mother, nd, daughters, xforms, &v, &host, stage == 4);
    if (rc != VG_OK) return rc;
    const NavMeta &mt = v.meta;
    const float4 *cull = reinterpret_cast<const float4 *>(host);
    const unsigned long long *cells = reinterpret_cast<const unsigned long long *>(host + mt.grid.off_g);
    const int *prim = reinterpret_cast<const int *>(host + mt.grid.off_p);
    if (grid)
        for (int a = 0; a < 3; ++a) grid[a] = mt.grid.o[a], grid[3 + a] = mt.grid.cs[a], grid[6 + a] = double(mt.grid.g[a]);
    if (grid && stage == 4) { // the safety grid's own box
        for (int a = 0; a < 3; ++a) grid[a] = mt.grid.so[a], grid[3 + a] = mt.grid.gs ? mt.grid.slen[a] / mt.grid.gs : 0.0, grid[6 + a] = double(mt.grid.gs);
        grid[9] = double(mt.grid.gs);
    }
    for (int64_t i = 0; i < n; ++i) {
        unsigned long long m[4] = { 0, 0, 0, 0 }, hit[4] = { 0, 0, 0, 0 };
        const double tl = t_lim ? t_lim[i] : INFINITY;
        if (stage == 0) { // both stages, as the kernel runs them
            if (mt.nchunks == 1) nav_cull<1>(mt.grid, cull, cells, prim, mt.all, x[i], y[i], z[i], dx[i], dy[i], dz[i], tl, reinterpret_cast<unsigned long long(&)[1]>(m));
            else if (mt.nchunks == 2) nav_cull<2>(mt.grid, cull, cells, prim, mt.all, x[i], y[i], z[i], dx[i], dy[i], dz[i], tl, reinterpret_cast<unsigned long long(&)[2]>(m));
            else nav_cull<4>(mt.grid, cull, cells, prim, mt.all, x[i], y[i], z[i], dx[i], dy[i], dz[i], tl, m);
        } else if (stage == 1) { // the grid walk alone
            if (mt.nchunks == 1) nav_grid_walk<1, false>(mt.grid, cells, prim, cull, x[i], y[i], z[i], dx[i], dy[i], dz[i], tl, reinterpret_cast<unsigned long long(&)[1]>(m), reinterpret_cast<unsigned long long(&)[1]>(hit));
            else if (mt.nchunks == 2) nav_grid_walk<2, false>(mt.grid, cells, prim, cull, x[i], y[i], z[i], dx[i], dy[i], dz[i], tl, reinterpret_cast<unsigned long long(&)[2]>(m), reinterpret_cast<unsigned long long(&)[2]>(hit));
            else nav_grid_walk<4, false>(mt.grid, cells, prim, cull, x[i], y[i], z[i], dx[i], dy[i], dz[i], tl, m, hit);
        } else if (stage == 3) { // the candidates of the POINT (world Locate, the volume safety of a point inside a daughter): its grid cell
            const unsigned long long *cell = nav_point_cell_masks(mt.grid, cells, mt.nchunks, x[i], y[i], z[i]);
            for (int c = 0; c < mt.nchunks; ++c) m[c] = cell ? cell[c] : 0ull;
        } else if (stage == 4) { // the candidates of the point's SAFETY: its cell of the safety grid, else every daughter
            const unsigned long long *cell = nav_safety_cell(
                mt.grid, reinterpret_cast<const unsigned long long *>(host + mt.grid.off_s), mt.nchunks, x[i], y[i], z[i]);
            for (int c = 0; c < mt.nchunks; ++c) m[c] = cell ? cell[c] : mt.all[c];
        } else { // the FP32 sphere test alone, applied to every daughter
            for (int c = 0; c < 4; ++c) m[c] = c < mt.nchunks ? mt.all[c] : 0ull;
            if (mt.nchunks == 1) nav_sphere_refine<1>(cull, x[i], y[i], z[i], dx[i], dy[i], dz[i], reinterpret_cast<unsigned long long(&)[1]>(m));
            else if (mt.nchunks == 2) nav_sphere_refine<2>(cull, x[i], y[i], z[i], dx[i], dy[i], dz[i], reinterpret_cast<unsigned long long(&)[2]>(m));
            else nav_sphere_refine<4>(cull, x[i], y[i], z[i], dx[i], dy[i], dz[i], m);
        }
        for (int c = 0; c < 4; ++c) masks[4 * i + c] = m[c];
    }
    delete[] host;
    return VG_OK;
}

extern "C" int vg_debug_boolean_program(const vg_shape *s, int *kinds, double *xforms, unsigned char *prog, int *nprog)
{
    if (!s || (s->kind != VG_BOOLEAN && s->kind != kCsg)) return fail(VG_ERR_ARG, "vg_debug_boolean_program: not a boolean");
    CsgOperand o;
    int rc = csg_operand(s, &o);
    if (rc != VG_OK) return rc;
    for (int i = 0; i < o.nleaf; ++i) {
        if (kinds) kinds[i] = o.leaf[i].kind;
        if (xforms) std::memcpy(xforms + 12 * i, o.X[i], 12 * sizeof(double));
    }
    if (prog) std::memcpy(prog, o.prog, size_t(o.nprog));
    if (nprog) *nprog = o.nprog;
    return o.nleaf;
}

extern "C" int vg_debug_polycone_grid(const vg_shape *s, uint64_t *masks, uint64_t *face_masks, unsigned char *row_section,
                                      double *geom, int *dims)
{
    if (!s || s->kind != VG_POLYCONE) return fail(VG_ERR_ARG, "vg_debug_polycone_grid: not a polycone");
    std::vector<unsigned long long> m;
    std::vector<unsigned char> rows;
    PconGridGeom g;
    pcon_grid_build(s->u.pcon, false, &g, &m, &rows);
    if (masks) std::memcpy(masks, m.data(), m.size() * sizeof(unsigned long long));
    if (row_section) std::memcpy(row_section, rows.data(), rows.size());
    if (geom) geom[0] = g.inv_cr, geom[1] = g.inv_cz, geom[2] = g.zg0;
    if (dims) dims[0] = kPconGridZ, dims[1] = kPconGridR;
    if (face_masks) {
        pcon_grid_build(s->u.pcon, true, &g, &m, &rows);
        std::memcpy(face_masks, m.data(), m.size() * sizeof(unsigned long long));
    }
    return VG_OK;
}

// -------------------------------------------------------------------------------------------------- probes

extern "C" int vg_probe_fp64_fma_rate(int launches, double *fma_per_s, void *stream)
{
    if (!fma_per_s || launches <= 0) return fail(VG_ERR_ARG, "vg_probe_fp64_fma_rate: bad arguments");
    *fma_per_s = 0.0;
    cudaError_t e = probe_fp64_fma_rate(launches, fma_per_s, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, "vg_probe_fp64_fma_rate");
    return VG_OK;
}

extern "C" int vg_probe_stream(int query, const double *x, const double *y, const double *z, const double *dx, const double *dy,
                               const double *dz, int64_t n, void *out, void *stream)
{
    if (query < qInside || query > qSafeOut) return fail(VG_ERR_ARG, "vg_probe_stream: unknown query");
    const bool dir = (query == qDistIn || query == qDistOut);
    const void *ptrs[6] = { x, y, z, dx, dy, dz };
    bool vec = false;
    int rc = check_arrays("vg_probe_stream", ptrs, dir ? 6 : 3, query == qInside ? 4 : 8, out, n, &vec);
    if (rc != VG_OK || n == 0) return rc;
    Tracks t{ x, y, z, dx, dy, dz };
    cudaError_t e = probe_stream(query, t, n, out, vec, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, "vg_probe_stream");
    return VG_OK;
}

extern "C" int vg_probe_empty_launch(int launches, void *stream)
{
    if (launches < 0) return fail(VG_ERR_ARG, "vg_probe_empty_launch: launches < 0");
    cudaError_t e = probe_empty_launch(launches, static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) return fail_cuda(e, "vg_probe_empty_launch");
    return VG_OK;
}
