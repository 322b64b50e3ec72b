"""paper_1512_06637_b200 -- Python binding of libvg.so (include/vg.h), argument marshalling only.

Every step of the path (Inside, DistanceToIn/Out, SafetyToIn/Out, ComputeStep)
runs in the sm_100a kernels behind the C ABI.  PyTorch is used for device memory and streams only: the
functions below take CUDA float64 tensors (struct-of-arrays, one tensor per coordinate), pass their
`data_ptr()` and the current CUDA stream to the library and return torch tensors.  There is NO CPU or eager
fallback: if libvg.so cannot be built/loaded the import fails, and a call without a CUDA device raises.

The function names are those of the C ABI (`vg_shape_create`, `vg_inside`, `vg_distance_to_in`, ...);
`Shape` / `Volume` are thin handle owners with the same calls as methods.
"""
import ctypes as C
import math

import torch

from . import build as _build

BOX, ORB, TUBE, CONE, TRD, POLYCONE = range(6)
BOOLEAN = 6
UNION, INTERSECTION, SUBTRACTION = 0, 1, 2
OUTSIDE, SURFACE, INSIDE = 0, 1, 2
HIT_MOTHER, HIT_STEPMAX = -1, -2
KTOLERANCE = 1e-9
OK, ERR_ARG, ERR_PARAM, ERR_ALIGN, ERR_CUDA, ERR_NOMEM = 0, -1, -2, -3, -4, -5

_VP = C.c_void_p
_PD = C.POINTER(C.c_double)


class VgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libvg error %d: %s" % (code, msg))
        self.code = code


def _load():
    path = _build.build()  # no-op when libvg.so is newer than its sources; raises if nvcc fails
    lib = C.CDLL(path)
    lib.vg_last_error.restype = C.c_char_p
    lib.vg_shape_create.argtypes = [C.c_int, _PD, C.c_int, C.POINTER(_VP)]
    lib.vg_shape_destroy.argtypes = [_VP]
    lib.vg_shape_destroy.restype = None
    lib.vg_shape_kind.argtypes = [_VP]
    lib.vg_inside.argtypes = [_VP, _VP, _VP, _VP, C.c_int64, _VP, _VP]
    for name in ("vg_distance_to_in", "vg_distance_to_out"):
        getattr(lib, name).argtypes = [_VP] + [_VP] * 6 + [C.c_double, C.c_int64, _VP, _VP]
    for name in ("vg_safety_to_in", "vg_safety_to_out"):
        getattr(lib, name).argtypes = [_VP, _VP, _VP, _VP, C.c_int64, _VP, _VP]
    lib.vg_query_all.argtypes = [_VP] + [_VP] * 6 + [C.c_double, C.c_int64] + [_VP] * 5 + [_VP]
    lib.vg_volume_create.argtypes = [_VP, C.c_int, C.POINTER(_VP), _PD, C.POINTER(_VP)]
    lib.vg_volume_destroy.argtypes = [_VP]
    lib.vg_volume_destroy.restype = None
    lib.vg_compute_step.argtypes = [_VP] + [_VP] * 6 + [C.c_double, C.c_int64, _VP, _VP, _VP]
    lib.vg_volume_safety.argtypes = [_VP, _VP, _VP, _VP, C.c_int64, _VP, _VP]
    lib.vg_boolean_create.argtypes = [C.c_int, _VP, _VP, _PD, C.POINTER(_VP)]
    lib.vg_world_create.argtypes = [C.c_int, C.POINTER(_VP), C.POINTER(C.c_int32), _PD, C.POINTER(_VP)]
    lib.vg_world_destroy.argtypes = [_VP]
    lib.vg_world_destroy.restype = None
    lib.vg_world_locate.argtypes = [_VP, _VP, _VP, _VP, C.c_int64, _VP, _VP]
    lib.vg_world_step.argtypes = [_VP, _VP] + [_VP] * 6 + [C.c_double, C.c_int64, _VP, _VP, _VP]
    lib.vg_world_safety.argtypes = [_VP, _VP, _VP, _VP, _VP, C.c_int64, _VP, _VP]
    lib.vg_query_host.argtypes = [_VP, C.c_int] + [_VP] * 6 + [C.c_double, C.c_int64, _VP]
    lib.vg_query_host_static.argtypes = [_VP, C.c_int] + [_VP] * 6 + [C.c_double, C.c_int64, _VP, _VP]
    lib.vg_query_all_host.argtypes = [_VP] + [_VP] * 6 + [C.c_double, C.c_int64] + [_VP] * 5
    lib.vg_compute_step_host.argtypes = [_VP] + [_VP] * 6 + [C.c_double, C.c_int64, _VP, _VP]
    lib.vg_probe_fp64_fma_rate.argtypes = [C.c_int, _PD, _VP]
    lib.vg_probe_empty_launch.argtypes = [C.c_int, _VP]
    lib.vg_probe_stream.argtypes = [C.c_int] + [_VP] * 6 + [C.c_int64, _VP, _VP]
    lib.vg_debug_nav_cull.argtypes = [_VP, C.c_int, C.POINTER(_VP), _PD] + [_VP] * 7 + [C.c_int64, _VP, C.c_int, _VP]
    lib.vg_launch_count.restype = C.c_int64
    lib.vg_set_option.argtypes = [C.c_int, C.c_int64]
    lib.vg_get_option.argtypes = [C.c_int]
    lib.vg_get_option.restype = C.c_int64
    return lib


_lib = _load()
LIB_PATH = _build.LIB


OPT_PIPE_MIN_N = 0
OPT_PDL = 1
OPT_FORM = 2
OPT_HOST_CHUNK = 3
OPT_COOP_MAX_N = 4
OPT_NAV_FORM = 5
FORM_AUTO, FORM_DIRECT, FORM_PIPELINED, FORM_STREAMING = 0, 1, 2, 3
INT64_MAX = 2 ** 63 - 1


def vg_set_option(option, value):
    """Launch policy (vg.h): OPT_PIPE_MIN_N = batch size from which the TMA-pipelined kernel is used."""
    _check(_lib.vg_set_option(int(option), int(value)))


def vg_get_option(option):
    return int(_lib.vg_get_option(int(option)))


def _check(rc):
    if rc != OK:
        raise VgError(rc, _lib.vg_last_error().decode("utf-8", "replace"))


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _tracks(arrs):
    """Validate SoA track tensors: CUDA, float64, 1-D, contiguous, same length and device."""
    n = arrs[0].numel()
    dev = arrs[0].device
    for a in arrs:
        if not isinstance(a, torch.Tensor) or not a.is_cuda:
            raise TypeError("track arrays must be CUDA tensors (there is no CPU path)")
        if a.dtype != torch.float64 or a.dim() != 1 or not a.is_contiguous():
            raise TypeError("track arrays must be 1-D contiguous float64")
        if a.numel() != n or a.device != dev:
            raise ValueError("track arrays must have the same length and device")
    return n, dev


def _out(out, n, dev, dtype):
    if out is None:
        return torch.empty(n, dtype=dtype, device=dev)
    if out.dtype != dtype or out.numel() != n or out.device != dev or not out.is_contiguous():
        raise TypeError("out: wrong dtype, length, device or layout")
    return out


def _p(t):
    return C.c_void_p(t.data_ptr())


# ---------------------------------------------------------------------------------------------- C-ABI names

def vg_shape_create(kind, params):
    par = (C.c_double * len(params))(*[float(v) for v in params])
    h = _VP()
    _check(_lib.vg_shape_create(int(kind), par, len(params), C.byref(h)))
    return h


def vg_shape_destroy(h):
    _lib.vg_shape_destroy(h)


def vg_boolean_create(op, a, b, xform_b):
    flat = [float(v) for v in xform_b]
    if len(flat) != 12:
        raise ValueError("xform_b must hold 12 doubles")
    h = _VP()
    _check(_lib.vg_boolean_create(int(op), _handle(a), _handle(b), (C.c_double * 12)(*flat), C.byref(h)))
    return h


def _handle(s):
    return s._h if isinstance(s, (Shape, Volume, World)) else s


def vg_inside(shape, x, y, z, out=None, stream=None):
    n, dev = _tracks((x, y, z))
    out = _out(out, n, dev, torch.int32)
    with torch.cuda.device(dev):
        _check(_lib.vg_inside(_handle(shape), _p(x), _p(y), _p(z), n, _p(out), _stream(stream)))
    return out


def _dist(fn, shape, x, y, z, dx, dy, dz, step_max, out, stream):
    n, dev = _tracks((x, y, z, dx, dy, dz))
    out = _out(out, n, dev, torch.float64)
    with torch.cuda.device(dev):
        _check(fn(_handle(shape), _p(x), _p(y), _p(z), _p(dx), _p(dy), _p(dz), float(step_max), n, _p(out),
                  _stream(stream)))
    return out


def vg_distance_to_in(shape, x, y, z, dx, dy, dz, step_max=math.inf, out=None, stream=None):
    return _dist(_lib.vg_distance_to_in, shape, x, y, z, dx, dy, dz, step_max, out, stream)


def vg_distance_to_out(shape, x, y, z, dx, dy, dz, step_max=math.inf, out=None, stream=None):
    return _dist(_lib.vg_distance_to_out, shape, x, y, z, dx, dy, dz, step_max, out, stream)


def _safe(fn, shape, x, y, z, out, stream):
    n, dev = _tracks((x, y, z))
    out = _out(out, n, dev, torch.float64)
    with torch.cuda.device(dev):
        _check(fn(_handle(shape), _p(x), _p(y), _p(z), n, _p(out), _stream(stream)))
    return out


def vg_safety_to_in(shape, x, y, z, out=None, stream=None):
    return _safe(_lib.vg_safety_to_in, shape, x, y, z, out, stream)


def vg_safety_to_out(shape, x, y, z, out=None, stream=None):
    return _safe(_lib.vg_safety_to_out, shape, x, y, z, out, stream)


def vg_query_all(shape, x, y, z, dx, dy, dz, step_max=math.inf, out=None, stream=None):
    """All five answers in one call (one fused kernel for every solid but the polycone).  `out`: optional tuple
    (cls int32, dist_in, dist_out, safety_in, safety_out) of preallocated tensors.  Returns that tuple."""
    n, dev = _tracks((x, y, z, dx, dy, dz))
    out = tuple(out) if out is not None else (None,) * 5
    cls = _out(out[0], n, dev, torch.int32)
    res = [_out(o, n, dev, torch.float64) for o in out[1:]]
    with torch.cuda.device(dev):
        _check(_lib.vg_query_all(_handle(shape), _p(x), _p(y), _p(z), _p(dx), _p(dy), _p(dz), float(step_max), n, _p(cls),
                                 *[_p(r) for r in res], _stream(stream)))
    return (cls, *res)


def vg_volume_create(mother, daughters, xforms):
    nd = len(daughters)
    arr = (_VP * max(1, nd))(*[_handle(d) for d in daughters])
    flat = [float(v) for row in xforms for v in (row if hasattr(row, "__len__") else [row])]
    if len(flat) != 12 * nd:
        raise ValueError("xforms must hold 12 doubles per daughter")
    xf = (C.c_double * max(1, len(flat)))(*flat)
    h = _VP()
    _check(_lib.vg_volume_create(_handle(mother), nd, arr, xf, C.byref(h)))
    return h


def vg_debug_nav_cull(mother, daughters, xforms, x, y, z, dx, dy, dz, t_lim=None, stage=0):
    """Host-only (numpy float64 arrays in, no device): the candidate masks of ComputeStep's conservative cull as
    uint64 (n, 4), and the candidate grid's geometry (origin[3], cell size[3], cells per axis[3]; stage 4 appends the
    safety grid's cells per axis)."""
    import numpy as np
    nd = len(daughters)
    arr = (_VP * max(1, nd))(*[_handle(d) for d in daughters])
    flat = [float(v) for row in xforms for v in row]
    xf = (C.c_double * max(1, len(flat)))(*flat)
    a = [np.ascontiguousarray(v, dtype=np.float64) for v in (x, y, z, dx, dy, dz)]
    n = a[0].size
    tl = None if t_lim is None else np.ascontiguousarray(t_lim, dtype=np.float64)
    masks = np.zeros((n, 4), dtype=np.uint64)
    grid = np.zeros(10 if int(stage) == 4 else 9, dtype=np.float64)
    _check(_lib.vg_debug_nav_cull(_handle(mother), nd, arr, xf, *[v.ctypes.data for v in a],
                                  None if tl is None else tl.ctypes.data, n, masks.ctypes.data, int(stage), grid.ctypes.data))
    return masks, grid


def vg_volume_destroy(h):
    _lib.vg_volume_destroy(h)


def vg_compute_step(volume, x, y, z, dx, dy, dz, step_max=math.inf, step=None, hit=None, stream=None):
    n, dev = _tracks((x, y, z, dx, dy, dz))
    step = _out(step, n, dev, torch.float64)
    hit = _out(hit, n, dev, torch.int32)
    with torch.cuda.device(dev):
        _check(_lib.vg_compute_step(_handle(volume), _p(x), _p(y), _p(z), _p(dx), _p(dy), _p(dz), float(step_max), n,
                                    _p(step), _p(hit), _stream(stream)))
    return step, hit


def vg_volume_safety(volume, x, y, z, out=None, stream=None):
    n, dev = _tracks((x, y, z))
    out = _out(out, n, dev, torch.float64)
    with torch.cuda.device(dev):
        _check(_lib.vg_volume_safety(_handle(volume), _p(x), _p(y), _p(z), n, _p(out), _stream(stream)))
    return out


# ---- hierarchy of volumes (readings R22-R25) ----

def vg_world_create(shapes, parents, xforms):
    nn = len(shapes)
    arr = (_VP * nn)(*[_handle(s) for s in shapes])
    par = (C.c_int32 * nn)(*[int(v) for v in parents])
    flat = [float(v) for row in xforms for v in row]
    if len(flat) != 12 * nn:
        raise ValueError("xforms must hold 12 doubles per node")
    xf = (C.c_double * len(flat))(*flat)
    h = _VP()
    _check(_lib.vg_world_create(nn, arr, par, xf, C.byref(h)))
    return h


def vg_world_destroy(h):
    _lib.vg_world_destroy(h)


def _nodes(node, n, dev):
    if not isinstance(node, torch.Tensor) or node.dtype != torch.int32 or node.numel() != n or node.device != dev or \
            not node.is_contiguous():
        raise TypeError("node: int32 CUDA tensor of the tracks' length expected")
    return node


def vg_world_locate(world, x, y, z, out=None, stream=None):
    n, dev = _tracks((x, y, z))
    out = _out(out, n, dev, torch.int32)
    with torch.cuda.device(dev):
        _check(_lib.vg_world_locate(_handle(world), _p(x), _p(y), _p(z), n, _p(out), _stream(stream)))
    return out


def vg_world_step(world, node, x, y, z, dx, dy, dz, step_max=math.inf, step=None, next=None, stream=None):
    n, dev = _tracks((x, y, z, dx, dy, dz))
    node = _nodes(node, n, dev)
    step = _out(step, n, dev, torch.float64)
    nxt = _out(next, n, dev, torch.int32)
    with torch.cuda.device(dev):
        _check(_lib.vg_world_step(_handle(world), _p(node), _p(x), _p(y), _p(z), _p(dx), _p(dy), _p(dz), float(step_max), n,
                                  _p(step), _p(nxt), _stream(stream)))
    return step, nxt


def vg_world_safety(world, node, x, y, z, out=None, stream=None):
    n, dev = _tracks((x, y, z))
    node = _nodes(node, n, dev)
    out = _out(out, n, dev, torch.float64)
    with torch.cuda.device(dev):
        _check(_lib.vg_world_safety(_handle(world), _p(node), _p(x), _p(y), _p(z), n, _p(out), _stream(stream)))
    return out


# ---- host-buffer entry points (tracks arriving from a host scheduler) ----

QUERY_ID = {"inside": 0, "distance_to_in": 1, "distance_to_out": 2, "safety_to_in": 3, "safety_to_out": 4}


def _host_tracks(arrs):
    n = arrs[0].numel()
    for a in arrs:
        if not isinstance(a, torch.Tensor) or a.is_cuda:
            raise TypeError("host entry points take CPU tensors (pinned memory makes the copies asynchronous)")
        if a.dtype != torch.float64 or a.dim() != 1 or not a.is_contiguous() or a.numel() != n:
            raise TypeError("track arrays must be 1-D contiguous float64 of one length")
    return n


def vg_query_host(shape, query, x, y, z, dx=None, dy=None, dz=None, step_max=math.inf, out=None):
    """One query over HOST track arrays: chunked H2D copy -> kernel -> D2H copy inside the library, pipelined
    over several streams.  Returns when `out` (a CPU tensor; int32 for "inside", else float64) is complete."""
    q = QUERY_ID[query] if isinstance(query, str) else int(query)
    needs_dir = q in (1, 2)
    arrs = (x, y, z, dx, dy, dz) if needs_dir else (x, y, z)
    n = _host_tracks(arrs)
    dtype = torch.int32 if q == 0 else torch.float64
    if out is None:
        out = torch.empty(n, dtype=dtype, pin_memory=True)
    elif out.is_cuda or out.dtype != dtype or out.numel() != n or not out.is_contiguous():
        raise TypeError("out: wrong dtype, length, device or layout")
    null = C.c_void_p(0)
    ptrs = [_p(a) for a in arrs] + ([] if needs_dir else [null] * 3)
    _check(_lib.vg_query_host(_handle(shape), q, *ptrs, float(step_max), n, _p(out)))
    return out


STATIC_MAX_TRACKS = 65536  # include/vg.h VG_STATIC_MAX_TRACKS


def vg_query_host_static(shape, query, x, y, z, dx=None, dy=None, dz=None, step_max=math.inf, out=None, stream=None):
    """vg_query_host without any allocation inside the library (include/vg.h): at most STATIC_MAX_TRACKS tracks, staged in
    a static device array that all calls share.  `out` is a CPU tensor the caller owns (created here if None)."""
    q = QUERY_ID[query] if isinstance(query, str) else int(query)
    needs_dir = q in (1, 2)
    arrs = (x, y, z, dx, dy, dz) if needs_dir else (x, y, z)
    n = _host_tracks(arrs)
    dtype = torch.int32 if q == 0 else torch.float64
    if out is None:
        out = torch.empty(n, dtype=dtype)
    elif out.is_cuda or out.dtype != dtype or out.numel() != n or not out.is_contiguous():
        raise TypeError("out: wrong dtype, length, device or layout")
    null = C.c_void_p(0)
    ptrs = [_p(a) for a in arrs] + ([] if needs_dir else [null] * 3)
    _check(_lib.vg_query_host_static(_handle(shape), q, *ptrs, float(step_max), n, _p(out), _stream(stream)))
    return out


def vg_query_all_host(shape, x, y, z, dx, dy, dz, step_max=math.inf, out=None):
    """All five answers over HOST track arrays (one pass of the tracks over the host link).  `out`: optional tuple of
    CPU tensors (cls int32, dist_in, dist_out, safety_in, safety_out).  Returns that tuple when complete."""
    n = _host_tracks((x, y, z, dx, dy, dz))
    if out is None:
        out = [torch.empty(n, dtype=torch.int32, pin_memory=True)] + \
              [torch.empty(n, dtype=torch.float64, pin_memory=True) for _ in range(4)]
    out = tuple(out)
    for o, dt in zip(out, (torch.int32,) + (torch.float64,) * 4):
        if o.is_cuda or o.dtype != dt or o.numel() != n or not o.is_contiguous():
            raise TypeError("out: wrong dtype, length, device or layout")
    _check(_lib.vg_query_all_host(_handle(shape), _p(x), _p(y), _p(z), _p(dx), _p(dy), _p(dz), float(step_max), n,
                                  *[_p(o) for o in out]))
    return out


def vg_compute_step_host(volume, x, y, z, dx, dy, dz, step_max=math.inf, step=None, hit=None):
    n = _host_tracks((x, y, z, dx, dy, dz))
    if step is None:
        step = torch.empty(n, dtype=torch.float64, pin_memory=True)
    if hit is None:
        hit = torch.empty(n, dtype=torch.int32, pin_memory=True)
    for o, dt in ((step, torch.float64), (hit, torch.int32)):
        if o.is_cuda or o.dtype != dt or o.numel() != n or not o.is_contiguous():
            raise TypeError("step/hit: wrong dtype, length, device or layout")
    _check(_lib.vg_compute_step_host(_handle(volume), _p(x), _p(y), _p(z), _p(dx), _p(dy), _p(dz), float(step_max), n,
                                     _p(step), _p(hit)))
    return step, hit


# ------------------------------------------------------------------------------- measurement helpers

def vg_probe_fp64_fma_rate(launches=20, stream=None):
    """Achieved FP64 FMA lanes per second of a register-resident DFMA chain (roofline denominator)."""
    r = C.c_double(0.0)
    _check(_lib.vg_probe_fp64_fma_rate(int(launches), C.byref(r), _stream(stream)))
    return r.value


def vg_probe_empty_launch(launches, stream=None):
    _check(_lib.vg_probe_empty_launch(int(launches), _stream(stream)))


def vg_probe_stream(query, x, y, z, dx=None, dy=None, dz=None, out=None, stream=None):
    """One launch of the arithmetic-free query kernel (same loads, store, grid and form as query `query` on these arrays)."""
    q = QUERY_ID[query] if isinstance(query, str) else int(query)
    n = x.numel()
    need6 = q in (1, 2)
    arrs = [x, y, z] + ([dx, dy, dz] if need6 else [None, None, None])
    _check(_lib.vg_probe_stream(q, *[(_p(a) if a is not None else None) for a in arrs], n, _p(out), _stream(stream)))
    return out


def vg_launch_count():
    """Kernel launches made by libvg in this process so far (bench.py's `gpu_launches`)."""
    return int(_lib.vg_launch_count())


# ------------------------------------------------------------------------------------- handle owners

class Shape:
    """One solid; `params` as in include/vg.h."""

    def __init__(self, kind, params):
        self.kind, self.params = int(kind), [float(v) for v in params]
        self._h = vg_shape_create(kind, params)

    def __del__(self, _destroy=_lib.vg_shape_destroy):
        h, self._h = getattr(self, "_h", None), None
        if h:
            _destroy(h)

    def inside(self, x, y, z, **kw):
        return vg_inside(self, x, y, z, **kw)

    def distance_to_in(self, x, y, z, dx, dy, dz, step_max=math.inf, **kw):
        return vg_distance_to_in(self, x, y, z, dx, dy, dz, step_max, **kw)

    def distance_to_out(self, x, y, z, dx, dy, dz, step_max=math.inf, **kw):
        return vg_distance_to_out(self, x, y, z, dx, dy, dz, step_max, **kw)

    def safety_to_in(self, x, y, z, **kw):
        return vg_safety_to_in(self, x, y, z, **kw)

    def safety_to_out(self, x, y, z, **kw):
        return vg_safety_to_out(self, x, y, z, **kw)

    def query(self, name, x, y, z, dx=None, dy=None, dz=None, step_max=math.inf, **kw):
        if name in ("distance_to_in", "distance_to_out"):
            return getattr(self, name)(x, y, z, dx, dy, dz, step_max, **kw)
        return getattr(self, name)(x, y, z, **kw)

    def query_all(self, x, y, z, dx, dy, dz, step_max=math.inf, **kw):
        return vg_query_all(self, x, y, z, dx, dy, dz, step_max, **kw)

    def query_all_host(self, x, y, z, dx, dy, dz, step_max=math.inf, **kw):
        return vg_query_all_host(self, x, y, z, dx, dy, dz, step_max, **kw)

    def query_host(self, name, x, y, z, dx=None, dy=None, dz=None, step_max=math.inf, out=None):
        return vg_query_host(self, name, x, y, z, dx, dy, dz, step_max, out)

    def query_host_static(self, name, x, y, z, dx=None, dy=None, dz=None, step_max=math.inf, out=None, stream=None):
        return vg_query_host_static(self, name, x, y, z, dx, dy, dz, step_max, out, stream)


class Boolean(Shape):
    """C = A op B of two primitives (readings R27-R29): `xform_b` is the row-major 3x4 [R | b] from the frame of C (= of A)
    to the frame of B.  Every query of Shape applies."""

    def __init__(self, op, a, b, xform_b):
        self.kind, self.op = BOOLEAN, int(op)
        self._h = vg_boolean_create(op, a, b, xform_b)


class Volume:
    """Mother solid + placed daughters; `xforms` (nd, 12) row-major [R | b], mother -> local (reading R12)."""

    def __init__(self, mother, daughters, xforms):
        self.nd = len(daughters)
        self._h = vg_volume_create(mother, daughters, [list(map(float, r)) for r in xforms])

    def __del__(self, _destroy=_lib.vg_volume_destroy):
        h, self._h = getattr(self, "_h", None), None
        if h:
            _destroy(h)

    def compute_step(self, x, y, z, dx, dy, dz, step_max=math.inf, **kw):
        return vg_compute_step(self, x, y, z, dx, dy, dz, step_max, **kw)

    def compute_step_host(self, x, y, z, dx, dy, dz, step_max=math.inf, **kw):
        return vg_compute_step_host(self, x, y, z, dx, dy, dz, step_max, **kw)

    def safety(self, x, y, z, **kw):
        return vg_volume_safety(self, x, y, z, **kw)


class World:
    """Tree of placed solids: node 0 is the root, `parents[i] < i`, `xforms` (nn, 12) row-major [R | b] from the
    parent's local frame (the world frame for the root) to the node's (readings R22-R25)."""

    def __init__(self, shapes, parents, xforms):
        self.nn = len(shapes)
        self._h = vg_world_create(shapes, parents, [list(map(float, r)) for r in xforms])

    def __del__(self, _destroy=_lib.vg_world_destroy):
        h, self._h = getattr(self, "_h", None), None
        if h:
            _destroy(h)

    def locate(self, x, y, z, **kw):
        return vg_world_locate(self, x, y, z, **kw)

    def step(self, node, x, y, z, dx, dy, dz, step_max=math.inf, **kw):
        return vg_world_step(self, node, x, y, z, dx, dy, dz, step_max, **kw)

    def safety(self, node, x, y, z, **kw):
        return vg_world_safety(self, node, x, y, z, **kw)
