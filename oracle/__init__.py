"""ORACLE -- test infrastructure, not the product.

ctypes binding of oracle/vg_oracle.c (plain scalar CPU implementation of the geometry
definitions of SURVEY.md sec. 8(c), the questions of PAPER.md:110-114).  Host numpy arrays in,
host numpy arrays out.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package; it imports nothing of the CUDA path.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

BOX, ORB, TUBE, CONE, TRD, POLYCONE = range(6)
OUTSIDE, SURFACE, INSIDE = 0, 1, 2
KTOL = 1e-9

_P = C.POINTER(C.c_double)
_PI = C.POINTER(C.c_int32)


def _load(path):
    lib = C.CDLL(path)
    lib.orc_shape_create.restype = C.c_void_p
    lib.orc_shape_create.argtypes = [C.c_int, _P, C.c_int]
    lib.orc_shape_destroy.argtypes = [C.c_void_p]
    lib.orc_volume_create.restype = C.c_void_p
    lib.orc_volume_create.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_void_p), _P]
    lib.orc_volume_destroy.argtypes = [C.c_void_p]
    lib.orc_num_threads.restype = C.c_int
    lib.orc_set_num_threads.argtypes = [C.c_int]
    for name in ("orc_sdf", "orc_safety_to_in", "orc_safety_to_out"):
        getattr(lib, name).argtypes = [C.c_void_p, _P, _P, _P, C.c_int64, _P]
    lib.orc_inside.argtypes = [C.c_void_p, _P, _P, _P, C.c_int64, _PI]
    for name in ("orc_distance_to_in", "orc_distance_to_out"):
        getattr(lib, name).argtypes = [C.c_void_p, _P, _P, _P, _P, _P, _P, C.c_double, C.c_int64, _P]
    lib.orc_cross.argtypes = [C.c_void_p, _P, _P, _P, _P, _P, _P, C.c_int64, _P]
    lib.orc_compute_step.argtypes = [C.c_void_p, _P, _P, _P, _P, _P, _P, C.c_double, C.c_int64, _P, _PI]
    lib.orc_volume_safety.argtypes = [C.c_void_p, _P, _P, _P, C.c_int64, _P]
    lib.orc_boolean_create.restype = C.c_void_p
    lib.orc_boolean_create.argtypes = [C.c_int, C.c_void_p, C.c_void_p, _P]
    lib.orc_boolean_create_nested.restype = C.c_void_p
    lib.orc_boolean_create_nested.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, _P]
    lib.orc_boolean_destroy.argtypes = [C.c_void_p]
    lib.orc_boolean_inside.argtypes = [C.c_void_p, _P, _P, _P, C.c_int64, _PI]
    lib.orc_boolean_sdf.argtypes = [C.c_void_p, _P, _P, _P, C.c_int64, _P]
    lib.orc_boolean_distance.argtypes = [C.c_void_p, C.c_int, _P, _P, _P, _P, _P, _P, C.c_double, C.c_int64, _P]
    lib.orc_all_crossings.restype = C.c_int
    lib.orc_all_crossings.argtypes = [C.c_void_p] + [C.c_double] * 6 + [_P, C.c_int]
    lib.orc_line_crossings.restype = C.c_int
    lib.orc_line_crossings.argtypes = [C.c_void_p] + [C.c_double] * 6 + [_P, C.c_int]
    lib.orc_boolean_events.restype = C.c_int
    lib.orc_boolean_events.argtypes = [C.c_void_p] + [C.c_double] * 6 + [_P, C.c_int]
    lib.orc_world_create.restype = C.c_void_p
    lib.orc_world_create.argtypes = [C.c_int, C.POINTER(C.c_void_p), _PI, _P]
    lib.orc_world_create_mixed.restype = C.c_void_p
    lib.orc_world_create_mixed.argtypes = [C.c_int, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), _PI, _P]
    lib.orc_world_destroy.argtypes = [C.c_void_p]
    lib.orc_world_locate.argtypes = [C.c_void_p, _P, _P, _P, C.c_int64, _PI]
    lib.orc_world_step.argtypes = [C.c_void_p, _PI, _P, _P, _P, _P, _P, _P, C.c_double, C.c_int64, _P, _PI]
    lib.orc_world_safety.argtypes = [C.c_void_p, _PI, _P, _P, _P, C.c_int64, _P]
    return lib


_LIBS = {}


def _lib(long_double=False):
    if long_double not in _LIBS:
        paths = _build.build()
        if not long_double and os.environ.get("ORACLE_SANITIZE") == "1":  # ASan + UBSan build (tests/test_oracle_sanitizers.py)
            paths = (_build.build_sanitized(), paths[1])
        _LIBS[long_double] = _load(paths[1] if long_double else paths[0])
    return _LIBS[long_double]


def _arr(a):
    return np.ascontiguousarray(np.atleast_1d(a), dtype=np.float64)


def _ptr(a):
    return a.ctypes.data_as(_P)


def num_threads():
    return _lib().orc_num_threads()


def set_num_threads(n):
    for lib in _LIBS.values():
        lib.orc_set_num_threads(int(n))
    _lib().orc_set_num_threads(int(n))


class Shape:
    """One solid.  `params` as in include/vg.h / SURVEY.md sec. 8(b)."""

    def __init__(self, kind, params, long_double=False):
        self._l = _lib(long_double)
        self.kind = int(kind)
        self.params = _arr(params)
        self._h = self._l.orc_shape_create(self.kind, _ptr(self.params), len(self.params))
        if not self._h:
            raise ValueError("oracle: invalid shape parameters kind=%d %r" % (kind, list(self.params)))

    def __del__(self):
        if getattr(self, "_h", None):
            self._l.orc_shape_destroy(self._h)
            self._h = None

    def _pts(self, x, y, z):
        x, y, z = _arr(x), _arr(y), _arr(z)
        assert x.shape == y.shape == z.shape
        return x, y, z

    def _f3(self, fn, x, y, z):
        x, y, z = self._pts(x, y, z)
        out = np.empty_like(x)
        fn(self._h, _ptr(x), _ptr(y), _ptr(z), x.size, _ptr(out))
        return out

    def sdf(self, x, y, z):
        return self._f3(self._l.orc_sdf, x, y, z)

    def safety_to_in(self, x, y, z):
        return self._f3(self._l.orc_safety_to_in, x, y, z)

    def safety_to_out(self, x, y, z):
        return self._f3(self._l.orc_safety_to_out, x, y, z)

    def inside(self, x, y, z):
        x, y, z = self._pts(x, y, z)
        out = np.empty(x.shape, dtype=np.int32)
        self._l.orc_inside(self._h, _ptr(x), _ptr(y), _ptr(z), x.size, out.ctypes.data_as(_PI))
        return out

    def _f6(self, fn, x, y, z, dx, dy, dz, *extra):
        x, y, z = self._pts(x, y, z)
        dx, dy, dz = self._pts(dx, dy, dz)
        assert dx.shape == x.shape
        out = np.empty_like(x)
        fn(self._h, _ptr(x), _ptr(y), _ptr(z), _ptr(dx), _ptr(dy), _ptr(dz), *extra, x.size, _ptr(out))
        return out

    def distance_to_in(self, x, y, z, dx, dy, dz, step_max=np.inf):
        return self._f6(self._l.orc_distance_to_in, x, y, z, dx, dy, dz, float(step_max))

    def distance_to_out(self, x, y, z, dx, dy, dz, step_max=np.inf):
        return self._f6(self._l.orc_distance_to_out, x, y, z, dx, dy, dz, float(step_max))

    def cross(self, x, y, z, dx, dy, dz):
        return self._f6(self._l.orc_cross, x, y, z, dx, dy, dz)

    def all_crossings(self, p, d):
        """Every crossing t > 0 of the boundary by the ray p + t d, ascending (one track)."""
        out = np.empty(512, dtype=np.float64)
        n = self._l.orc_all_crossings(self._h, *[float(v) for v in p], *[float(v) for v in d], _ptr(out), out.size)
        return out[:n].copy()

    def line_crossings(self, p, d):
        """Every crossing of the boundary by the whole line p + t d, t of either sign, ascending (reading R32)."""
        out = np.empty(512, dtype=np.float64)
        n = self._l.orc_line_crossings(self._h, *[float(v) for v in p], *[float(v) for v in d], _ptr(out), out.size)
        return out[:n].copy()


class Volume:
    """Mother solid + placed daughters; `xforms` is (nd, 12) row-major [R | b], mother -> local."""

    def __init__(self, mother, daughters, xforms):
        self._l = mother._l
        self.mother = mother
        self.daughters = list(daughters)
        self.xforms = np.ascontiguousarray(np.asarray(xforms, dtype=np.float64).reshape(len(self.daughters), 12))
        arr = (C.c_void_p * max(1, len(self.daughters)))(*[d._h for d in self.daughters])
        self._h = self._l.orc_volume_create(mother._h, len(self.daughters), arr, _ptr(self.xforms))
        if not self._h:
            raise ValueError("oracle: invalid volume")

    def __del__(self):
        if getattr(self, "_h", None):
            self._l.orc_volume_destroy(self._h)
            self._h = None

    def compute_step(self, x, y, z, dx, dy, dz, step_max=np.inf):
        x, y, z, dx, dy, dz = map(_arr, (x, y, z, dx, dy, dz))
        step = np.empty_like(x)
        hit = np.empty(x.shape, dtype=np.int32)
        self._l.orc_compute_step(self._h, _ptr(x), _ptr(y), _ptr(z), _ptr(dx), _ptr(dy), _ptr(dz), float(step_max),
                                 x.size, _ptr(step), hit.ctypes.data_as(_PI))
        return step, hit

    def safety(self, x, y, z):
        x, y, z = map(_arr, (x, y, z))
        out = np.empty_like(x)
        self._l.orc_volume_safety(self._h, _ptr(x), _ptr(y), _ptr(z), x.size, _ptr(out))
        return out


UNION, INTERSECTION, SUBTRACTION = 0, 1, 2


class Boolean:
    """C = A op B (readings R27-R29, vg_oracle.c): `xform` is the row-major 3x4 [R | b] from the frame of C (= of A)
    to the frame of B; A and B are Shapes or Booleans (R31, at most 8 primitives per tree).  Same query names as Shape;
    the safeties are the composed bound of R29."""

    def leaves(self, pre=None):
        """[(primitive Shape, 3x4 matrix frame of this boolean -> frame of the primitive)] in tree order."""
        pre = np.eye(4) if pre is None else pre
        out = []
        for operand, M in ((self.a, pre), (self.b, np.vstack([self.xform.reshape(3, 4), [0, 0, 0, 1]]) @ pre)):
            out += operand.leaves(M) if isinstance(operand, Boolean) else [(operand, M[:3])]
        return out

    def __init__(self, op, a, b, xform):
        self._l = a._l
        self.op, self.a, self.b = int(op), a, b
        self.xform = np.ascontiguousarray(np.asarray(xform, dtype=np.float64).reshape(12))
        na, nb = isinstance(a, Boolean), isinstance(b, Boolean)  # R31: an operand may be a boolean itself
        self._h = self._l.orc_boolean_create_nested(self.op, None if na else a._h, a._h if na else None,
                                                    None if nb else b._h, b._h if nb else None, _ptr(self.xform))
        if not self._h:
            raise ValueError("oracle: invalid boolean")

    def __del__(self):
        if getattr(self, "_h", None):
            self._l.orc_boolean_destroy(self._h)
            self._h = None

    def inside(self, x, y, z):
        x, y, z = map(_arr, (x, y, z))
        out = np.empty(x.shape, dtype=np.int32)
        self._l.orc_boolean_inside(self._h, _ptr(x), _ptr(y), _ptr(z), x.size, out.ctypes.data_as(_PI))
        return out

    def sdf(self, x, y, z):
        x, y, z = map(_arr, (x, y, z))
        out = np.empty_like(x)
        self._l.orc_boolean_sdf(self._h, _ptr(x), _ptr(y), _ptr(z), x.size, _ptr(out))
        return out

    def safety_to_in(self, x, y, z):
        return self.sdf(x, y, z)

    def safety_to_out(self, x, y, z):
        return -self.sdf(x, y, z)

    def _dist(self, which, x, y, z, dx, dy, dz, step_max):
        x, y, z, dx, dy, dz = map(_arr, (x, y, z, dx, dy, dz))
        out = np.empty_like(x)
        self._l.orc_boolean_distance(self._h, which, _ptr(x), _ptr(y), _ptr(z), _ptr(dx), _ptr(dy), _ptr(dz),
                                     float(step_max), x.size, _ptr(out))
        return out

    def distance_to_in(self, x, y, z, dx, dy, dz, step_max=np.inf):
        return self._dist(0, x, y, z, dx, dy, dz, step_max)

    def distance_to_out(self, x, y, z, dx, dy, dz, step_max=np.inf):
        return self._dist(1, x, y, z, dx, dy, dz, step_max)

    def events(self, p, d):
        """Every t (either sign) at which the membership of the boolean flips along the whole line p + t d (R28)."""
        out = np.empty(8 * 272, dtype=np.float64)
        n = self._l.orc_boolean_events(self._h, *[float(v) for v in p], *[float(v) for v in d], _ptr(out), out.size)
        return out[:n].copy()


class World:
    """Tree of placed solids (readings R22-R25, R30, vg_oracle.c; a node is a Shape or a Boolean): node 0 is the root, `parents[i] < i`,
    `xforms` is (nn, 12) row-major [R | b] from the parent's local frame (the world frame for the root)."""

    def __init__(self, shapes, parents, xforms):
        self.shapes = list(shapes)
        self._l = self.shapes[0]._l
        nn = len(self.shapes)
        self.parents = np.ascontiguousarray(np.asarray(parents, dtype=np.int32).reshape(nn))
        self.xforms = np.ascontiguousarray(np.asarray(xforms, dtype=np.float64).reshape(nn, 12))
        arr = (C.c_void_p * nn)(*[None if isinstance(s, Boolean) else s._h for s in self.shapes])
        barr = (C.c_void_p * nn)(*[s._h if isinstance(s, Boolean) else None for s in self.shapes])
        self._h = self._l.orc_world_create_mixed(nn, arr, barr, self.parents.ctypes.data_as(_PI), _ptr(self.xforms))
        if not self._h:
            raise ValueError("oracle: invalid world")

    def __del__(self):
        if getattr(self, "_h", None):
            self._l.orc_world_destroy(self._h)
            self._h = None

    def locate(self, x, y, z):
        x, y, z = map(_arr, (x, y, z))
        node = np.empty(x.shape, dtype=np.int32)
        self._l.orc_world_locate(self._h, _ptr(x), _ptr(y), _ptr(z), x.size, node.ctypes.data_as(_PI))
        return node

    def step(self, node, x, y, z, dx, dy, dz, step_max=np.inf):
        x, y, z, dx, dy, dz = map(_arr, (x, y, z, dx, dy, dz))
        node = np.ascontiguousarray(node, dtype=np.int32)
        step = np.empty_like(x)
        nxt = np.empty(x.shape, dtype=np.int32)
        self._l.orc_world_step(self._h, node.ctypes.data_as(_PI), _ptr(x), _ptr(y), _ptr(z), _ptr(dx), _ptr(dy),
                               _ptr(dz), float(step_max), x.size, _ptr(step), nxt.ctypes.data_as(_PI))
        return step, nxt

    def safety(self, node, x, y, z):
        x, y, z = map(_arr, (x, y, z))
        node = np.ascontiguousarray(node, dtype=np.int32)
        out = np.empty_like(x)
        self._l.orc_world_safety(self._h, node.ctypes.data_as(_PI), _ptr(x), _ptr(y), _ptr(z), x.size, _ptr(out))
        return out
