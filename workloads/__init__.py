"""Seeded synthetic workloads: the five configurations of BASELINE.json (`configs[0..4]`).

This module serves BOTH the oracle tests and the CUDA path (tests, bench.py, smoke) and holds
none of the method's arithmetic: it only draws numbers (numpy Philox) and lays out parameters.
The one geometric decision the recipe needs -- rejecting points that lie in the 1e-6 surface
band (BASELINE.json configs[0]) -- is taken by a callback the caller
supplies (`band(x, y, z) -> bool mask of points to redraw`), so that the oracle legs reject with
the oracle's sdf and the product legs with the library's own safety query.

Recipe (SURVEY.md sec. 8(d) "Generator"; the paper's workload is "randomly placed particles with
random speed"): points c + (2u-1) h per axis in the sampling box, directions
dz = 2u1-1, phi = 2 pi u2, d = (sqrt(1-dz^2) cos phi, sqrt(1-dz^2) sin phi, dz), renormalised once.
"""
import math

import numpy as np

# shape kinds: the enumeration of include/vg.h (and, independently, of the oracle)
BOX, ORB, TUBE, CONE, TRD, POLYCONE = range(6)
KIND_NAME = {BOX: "box", ORB: "orb", TUBE: "tube", CONE: "cone", TRD: "trd", POLYCONE: "polycone"}

BASE_SEED = 1512066370          # + k for config k, + 100 * shape_index for a second shape of the config
SURFACE_BAND = 1e-6             # generators keep |sdf| >= 1e-6 (BASELINE.json configs[0], R17)
STEP_MAX = 1e30                 # BASELINE.json configs[0], [4]
TWO_PI = 2.0 * math.pi

QUERIES5 = ("inside", "distance_to_in", "distance_to_out", "safety_to_in", "safety_to_out")


def config_seed(k, shape_index=0):
    return BASE_SEED + k + 100 * shape_index


def _rng(seed):
    return np.random.Generator(np.random.Philox(int(seed)))


def draw_tracks(seed, n, center, half, band=None, max_rounds=64):
    """n tracks as six float64 arrays (x, y, z, dx, dy, dz).

    `band(x, y, z)` returns True for points to be redrawn (inside the surface band, or outside the
    region the config allows); redraws come from the continuing stream until none remain.
    """
    rng = _rng(seed)
    n = int(n)
    c = np.asarray(center, dtype=np.float64)
    h = np.asarray(half, dtype=np.float64)
    u = rng.random((n, 3))
    p = c + (2.0 * u - 1.0) * h
    v = rng.random((n, 2))
    dz = 2.0 * v[:, 0] - 1.0
    phi = TWO_PI * v[:, 1]
    s = np.sqrt(np.maximum(0.0, 1.0 - dz * dz))
    dx = s * np.cos(phi)
    dy = s * np.sin(phi)
    norm = np.sqrt(dx * dx + dy * dy + dz * dz)
    dx, dy, dz = dx / norm, dy / norm, dz / norm
    x, y, z = (np.ascontiguousarray(p[:, i]) for i in range(3))
    if band is not None and n > 0:
        bad = np.flatnonzero(np.asarray(band(x, y, z), dtype=bool))
        rounds = 0
        while bad.size:
            rounds += 1
            if rounds > max_rounds:
                raise RuntimeError("draw_tracks: rejection did not terminate")
            q = c + (2.0 * rng.random((bad.size, 3)) - 1.0) * h
            x[bad], y[bad], z[bad] = q[:, 0], q[:, 1], q[:, 2]
            still = np.asarray(band(x[bad], y[bad], z[bad]), dtype=bool)
            bad = bad[still]
    return x, y, z, np.ascontiguousarray(dx), np.ascontiguousarray(dy), np.ascontiguousarray(dz)


# --------------------------------------------------------------------------- shapes of the configs

def bounding_half(kind, params):
    """Centre and half-extent of the axis-aligned box of the FULL-phi solid (reading R16)."""
    p = list(params)
    if kind == BOX:
        return (0.0, 0.0, 0.0), (p[0], p[1], p[2])
    if kind == ORB:
        return (0.0, 0.0, 0.0), (p[0], p[0], p[0])
    if kind == TUBE:
        return (0.0, 0.0, 0.0), (p[1], p[1], p[2])
    if kind == CONE:
        r = max(p[1], p[3])
        return (0.0, 0.0, 0.0), (r, r, p[4])
    if kind == TRD:
        return (0.0, 0.0, 0.0), (max(p[0], p[1]), max(p[2], p[3]), p[4])
    if kind == POLYCONE:
        nz = int(p[2])
        zs = [p[3 + 3 * i] for i in range(nz)]
        r = max(p[5 + 3 * i] for i in range(nz))
        return (0.0, 0.0, 0.5 * (zs[0] + zs[-1])), (r, r, 0.5 * (zs[-1] - zs[0]))
    raise ValueError(kind)


def polycone_params(seed, nz=10):
    """configs[3]: z uniform-sorted in [-50,50], rmin uniform [0,5], rmax uniform [10,30], full phi."""
    rng = _rng(seed + 7)
    z = np.sort(rng.uniform(-50.0, 50.0, nz))
    rmin = rng.uniform(0.0, 5.0, nz)
    rmax = rng.uniform(10.0, 30.0, nz)
    out = [0.0, TWO_PI, float(nz)]
    for i in range(nz):
        out += [float(z[i]), float(rmin[i]), float(rmax[i])]
    return out


# a polycone with two z steps (reading R26): the radii jump outwards at z = -4 (the bore opens) and inwards at z = 6
STEPPED_POLYCONE = [0.0, TWO_PI, 7.0, -12.0, 0.0, 6.0, -4.0, 1.0, 8.0, -4.0, 3.0, 12.0, 2.0, 2.0, 10.0, 6.0, 2.0, 11.0,
                    6.0, 0.0, 5.0, 14.0, 1.5, 4.0]


class ShapeCase:
    """One (shape, sampling box, seed) of a config."""

    def __init__(self, cfg, name, kind, params, center, half, seed, sizes, queries):
        self.cfg, self.name, self.kind = cfg, name, kind
        self.params = [float(v) for v in params]
        self.center, self.half = tuple(center), tuple(half)
        self.seed, self.sizes, self.queries = seed, tuple(sizes), tuple(queries)

    def tracks(self, n=None, band=None):
        return draw_tracks(self.seed, self.sizes[-1] if n is None else n, self.center, self.half, band)


def _scaled(kind, params, scale=1.5):
    c, h = bounding_half(kind, params)
    return c, tuple(scale * v for v in h)


def shape_cases(k):
    """The ShapeCase list of BASELINE.json configs[k], k = 0..3 (config 4 is `navigator_case`)."""
    if k == 0:
        par = [5.0, 5.0, 5.0]
        return [ShapeCase(0, "box", BOX, par, (0, 0, 0), (10, 10, 10), config_seed(0), [65536], QUERIES5)]
    if k == 1:
        par = [5.0, 10.0, 15.0, 0.0, 4.0 * math.pi / 3.0]
        c, h = _scaled(TUBE, par)
        return [ShapeCase(1, "tube", TUBE, par, c, h, config_seed(1), [1048576], QUERIES5)]
    if k == 2:
        cone = [2.0, 6.0, 4.0, 12.0, 20.0, 0.0, TWO_PI]
        trd = [5.0, 10.0, 7.0, 3.0, 15.0]
        c0, h0 = _scaled(CONE, cone)
        c1, h1 = _scaled(TRD, trd)
        return [ShapeCase(2, "cone", CONE, cone, c0, h0, config_seed(2, 0), [4194304], QUERIES5),
                ShapeCase(2, "trd", TRD, trd, c1, h1, config_seed(2, 1), [4194304], QUERIES5)]
    if k == 3:
        sizes = [2 ** 10, 2 ** 14, 2 ** 18, 2 ** 22, 2 ** 24]
        pc = polycone_params(config_seed(3, 0))
        orb = [20.0]
        c0, h0 = _scaled(POLYCONE, pc)
        c1, h1 = _scaled(ORB, orb)
        q = ("distance_to_in", "safety_to_in")
        return [ShapeCase(3, "polycone", POLYCONE, pc, c0, h0, config_seed(3, 0), sizes, q),
                ShapeCase(3, "orb", ORB, orb, c1, h1, config_seed(3, 1), sizes, q)]
    raise ValueError("config %r has no shape cases" % (k,))


# ------------------------------------------------------------------------------ navigator (configs[4])

def quaternion_to_matrix(q):
    """Rotation matrix (local -> mother) of a unit quaternion (x, y, z, w)."""
    x, y, z, w = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]], dtype=np.float64)


def placement(Q, c):
    """3x4 row-major mother -> local transform [R | b] of a daughter centred at c with local -> mother
    rotation Q: R = Q^T, b = -Q^T c (reading R12)."""
    R = np.asarray(Q, dtype=np.float64).T
    b = -R @ np.asarray(c, dtype=np.float64)
    return np.concatenate([R, b[:, None]], axis=1).reshape(12)


class NavigatorCase:
    """configs[4]: mother box (100,100,100), 64 daughters on a 4x4x4 grid (readings R14, R15)."""

    def __init__(self, seed=None, n=4194304, grid=4, pitch=50.0, mother_half=100.0, dhalf=8.0):
        self.cfg = 4
        self.seed = config_seed(4) if seed is None else seed
        self.sizes = (n,)
        self.mother_kind, self.mother_params = BOX, [mother_half] * 3
        self.center, self.half = (0.0, 0.0, 0.0), (mother_half,) * 3
        rng = _rng(self.seed + 7)
        kinds, params, xf, centers = [], [], [], []
        off = 0.5 * (grid - 1) * pitch
        for iz in range(grid):
            for iy in range(grid):
                for ix in range(grid):
                    c = (ix * pitch - off, iy * pitch - off, iz * pitch - off)
                    u1, u2, u3 = rng.random(3)
                    q = (math.sqrt(1 - u1) * math.sin(TWO_PI * u2), math.sqrt(1 - u1) * math.cos(TWO_PI * u2),
                         math.sqrt(u1) * math.sin(TWO_PI * u3), math.sqrt(u1) * math.cos(TWO_PI * u3))
                    if (ix + iy + iz) % 2 == 0:
                        kinds.append(BOX)
                        params.append([dhalf, dhalf, dhalf])
                    else:
                        kinds.append(TUBE)
                        params.append([0.0, dhalf, dhalf, 0.0, TWO_PI])
                    xf.append(placement(quaternion_to_matrix(q), c))
                    centers.append(c)
        self.daughter_kinds, self.daughter_params = kinds, params
        self.xforms = np.ascontiguousarray(np.stack(xf))
        self.centers = np.asarray(centers)

    def tracks(self, n=None, band=None):
        return draw_tracks(self.seed, self.sizes[-1] if n is None else n, self.center, self.half, band)


def navigator_case(**kw):
    return NavigatorCase(**kw)


# ------------------------------------------------------------- hierarchy of volumes

class WorldCase:
    """A three-level tree of placed solids (readings R22-R25): the mother box and the 64 daughters of
    configs[4] (nodes 1..64), and two grand-daughters with seeded random rotations inside every daughter
    (nodes 65..192): an orb r = 3 and a trd inside each box, a hollow tube segment and a cone inside each tube.
    Bounding spheres are disjoint and inside the parent, so siblings never overlap whatever the rotation.

    Tracks: half of the points uniform in the mother box, half uniform in the local cube [-8, 8]^3 of a random
    daughter (so that about a third of the tracks start below the root), isotropic directions.
    """

    def __init__(self, seed=None, n=4194304):
        nav = NavigatorCase(seed=config_seed(4) if seed is None else seed, n=n)
        self.cfg, self.seed, self.sizes = 5, nav.seed + 11, (n,)
        self.center, self.half = nav.center, nav.half
        rng = _rng(self.seed)
        kinds, params, parents, xf = [nav.mother_kind], [nav.mother_params], [-1], [placement(np.eye(3), (0, 0, 0))]
        for k in range(len(nav.daughter_kinds)):
            kinds.append(nav.daughter_kinds[k])
            params.append(nav.daughter_params[k])
            parents.append(0)
            xf.append(nav.xforms[k])
        inner = {BOX: [(ORB, [3.0], (-3.5, 0.0, 0.0)), (TRD, [1.5, 2.5, 2.0, 1.0, 1.5], (4.0, 1.0, -1.0))],
                 TUBE: [(TUBE, [1.0, 3.0, 3.0, 0.0, 4.0 * math.pi / 3.0], (0.0, 3.5, 2.0)),
                        (CONE, [0.0, 1.0, 0.0, 2.5, 2.0, 0.0, TWO_PI], (0.0, -4.0, -3.0))]}
        for k in range(len(nav.daughter_kinds)):
            for kind, par, c in inner[nav.daughter_kinds[k]]:
                u1, u2, u3 = rng.random(3)
                q = (math.sqrt(1 - u1) * math.sin(TWO_PI * u2), math.sqrt(1 - u1) * math.cos(TWO_PI * u2),
                     math.sqrt(u1) * math.sin(TWO_PI * u3), math.sqrt(u1) * math.cos(TWO_PI * u3))
                kinds.append(kind)
                params.append(par)
                parents.append(1 + k)
                xf.append(placement(quaternion_to_matrix(q), c))
        self.kinds, self.params = kinds, params
        self.parents = np.asarray(parents, dtype=np.int32)
        self.xforms = np.ascontiguousarray(np.stack(xf))
        self.level1 = np.arange(1, 1 + len(nav.daughter_kinds))

    def tracks(self, n=None, band=None, max_rounds=64):
        """`band(x, y, z)` -> True for points to redraw (surface band of any node, or outside the world)."""
        n = int(self.sizes[-1] if n is None else n)
        rng = _rng(self.seed + 1)

        def points(m):
            p = (2.0 * rng.random((m, 3)) - 1.0) * np.asarray(self.half)
            low = rng.random(m) < 0.5
            which = self.level1[rng.integers(0, len(self.level1), m)]
            loc = (2.0 * rng.random((m, 3)) - 1.0) * getattr(self, "local_cube", 8.0)
            M = self.xforms[which].reshape(m, 3, 4)
            # local -> mother: p = R^T (p_loc - b)
            back = np.einsum("nji,nj->ni", M[:, :, :3], loc - M[:, :, 3])
            p[low] = back[low]
            return p

        p = points(n)
        v = rng.random((n, 2))
        dz = 2.0 * v[:, 0] - 1.0
        phi = TWO_PI * v[:, 1]
        s = np.sqrt(np.maximum(0.0, 1.0 - dz * dz))
        dx, dy = s * np.cos(phi), s * np.sin(phi)
        norm = np.sqrt(dx * dx + dy * dy + dz * dz)
        dx, dy, dz = dx / norm, dy / norm, dz / norm
        x, y, z = (np.ascontiguousarray(p[:, i]) for i in range(3))
        if band is not None and n > 0:
            bad = np.flatnonzero(np.asarray(band(x, y, z), dtype=bool))
            rounds = 0
            while bad.size:
                rounds += 1
                if rounds > max_rounds:
                    raise RuntimeError("WorldCase.tracks: rejection did not terminate")
                q = points(bad.size)
                x[bad], y[bad], z[bad] = q[:, 0], q[:, 1], q[:, 2]
                bad = bad[np.asarray(band(x[bad], y[bad], z[bad]), dtype=bool)]
        return x, y, z, np.ascontiguousarray(dx), np.ascontiguousarray(dy), np.ascontiguousarray(dz)


def world_case(**kw):
    return WorldCase(**kw)


# ------------------------------------------------------------------ boolean solids

UNION, INTERSECTION, SUBTRACTION = 0, 1, 2
OP_NAME = {UNION: "union", INTERSECTION: "intersection", SUBTRACTION: "subtraction"}


class BooleanCase:
    """C = A op B (readings R27-R29): B placed in the frame of A by a seeded rotation and an offset; tracks
    from points uniform in 1.2 x the box that bounds A and the bounding sphere of B, isotropic directions."""

    def __init__(self, name, op, kind_a, par_a, kind_b, par_b, offset, quat, seed):
        self.name, self.op = name, op
        self.kind_a, self.par_a = kind_a, [float(v) for v in par_a]
        self.kind_b, self.par_b = kind_b, [float(v) for v in par_b]
        self.xform = placement(quaternion_to_matrix(quat), offset)
        self.seed = seed
        ca, ha = bounding_half(kind_a, par_a)
        cb, hb = bounding_half(kind_b, par_b)
        rb = math.sqrt(sum(v * v for v in hb)) + math.sqrt(sum(v * v for v in cb))
        lo = [min(ca[i] - ha[i], offset[i] - rb) for i in range(3)]
        hi = [max(ca[i] + ha[i], offset[i] + rb) for i in range(3)]
        self.center = tuple(0.5 * (lo[i] + hi[i]) for i in range(3))
        self.half = tuple(0.6 * (hi[i] - lo[i]) for i in range(3))

    def tracks(self, n, band=None):
        return draw_tracks(self.seed, n, self.center, self.half, band)


def boolean_cases():
    s2 = math.sqrt(0.5)
    q = [(0.0, 0.0, 0.0, 1.0), (s2, 0.0, 0.0, s2), (0.18257418583505536, 0.3651483716701107, 0.5477225575051661, 0.7302967433402214),
         (0.5, -0.5, 0.5, 0.5)]
    seed = BASE_SEED + 600
    return [
        BooleanCase("tube_union_box", UNION, TUBE, [5.0, 10.0, 15.0, 0.0, 4.0 * math.pi / 3.0], BOX, [4.0, 4.0, 20.0], (6.0, -2.0, 1.0), q[2], seed),
        BooleanCase("box_union_orb", UNION, BOX, [5.0, 5.0, 5.0], ORB, [6.0], (3.0, 2.0, -1.0), q[0], seed + 1),
        BooleanCase("cone_intersection_orb", INTERSECTION, CONE, [2.0, 6.0, 4.0, 12.0, 20.0, 0.0, TWO_PI], ORB, [14.0], (2.0, 1.0, 6.0), q[0], seed + 2),
        BooleanCase("trd_intersection_tube", INTERSECTION, TRD, [5.0, 10.0, 7.0, 3.0, 15.0], TUBE, [2.0, 8.0, 12.0, 0.0, TWO_PI], (1.0, 0.5, -2.0), q[1], seed + 3),
        BooleanCase("box_minus_tube", SUBTRACTION, BOX, [10.0, 10.0, 10.0], TUBE, [0.0, 4.0, 12.0, 0.0, TWO_PI], (1.0, -2.0, 0.0), q[2], seed + 4),
        BooleanCase("orb_minus_box", SUBTRACTION, ORB, [12.0], BOX, [9.0, 3.0, 20.0], (0.0, 2.0, 0.0), q[3], seed + 5),
        BooleanCase("tube_minus_cone", SUBTRACTION, TUBE, [0.0, 10.0, 10.0, 0.0, TWO_PI], CONE, [0.0, 2.0, 0.0, 9.0, 8.0, 0.5, 5.0], (0.0, 0.0, 3.0), q[0], seed + 6),
    ]


class MixedWorldCase:
    """A tree whose nodes are not only primitives (reading R30): the mother box (100) holds eight daughters at
    (+-50, +-50, +-50) with seeded rotations -- two stepped polycones, two booleans box-minus-tube, two configs[3]
    polycones, two booleans tube-union-box -- and a grand-daughter inside the material of each stepped polycone (an orb)
    and of each box-minus-tube (a small box in a corner clear of the bore).  13 nodes.

    `nodes[i]` is ("shape", kind, params) or ("boolean", BooleanCase); tracks as in WorldCase (half in the mother box,
    half in the local cube [-14, 14]^3 of a random daughter)."""

    def __init__(self, seed=None, n=1048576):
        self.seed = (config_seed(4) + 23) if seed is None else seed
        self.sizes = (n,)
        self.center, self.half = (0.0, 0.0, 0.0), (100.0, 100.0, 100.0)
        rng = _rng(self.seed)
        bools = {b.name: b for b in boolean_cases()}
        kinds4 = [("shape", POLYCONE, STEPPED_POLYCONE), ("boolean", bools["box_minus_tube"]),
                  ("shape", POLYCONE, polycone_params(config_seed(3, 0))), ("boolean", bools["tube_union_box"])]
        nodes, parents, xf = [("shape", BOX, [100.0, 100.0, 100.0])], [-1], [placement(np.eye(3), (0, 0, 0))]

        def rot():
            u1, u2, u3 = rng.random(3)
            return quaternion_to_matrix((math.sqrt(1 - u1) * math.sin(TWO_PI * u2), math.sqrt(1 - u1) * math.cos(TWO_PI * u2),
                                         math.sqrt(u1) * math.sin(TWO_PI * u3), math.sqrt(u1) * math.cos(TWO_PI * u3)))
        k = 0
        for sz in (-50.0, 50.0):
            for sy in (-50.0, 50.0):
                for sx in (-50.0, 50.0):
                    nodes.append(kinds4[k % 4])
                    parents.append(0)
                    xf.append(placement(rot(), (sx, sy, sz)))
                    k += 1
        # the corner of box-minus-tube farthest from the bore: distance from the tube's axis (a line through the placement
        # centre along R^T e_z in the boolean's frame)
        M = np.asarray(bools["box_minus_tube"].xform).reshape(3, 4)
        axis, centre = M[2, :3], -M[:, :3].T @ M[:, 3]
        corners = [np.array([a, b, c]) for a in (-7.0, 7.0) for b in (-7.0, 7.0) for c in (-7.0, 7.0)]
        corner = max(corners, key=lambda p: np.linalg.norm(np.cross(p - centre, axis)))
        assert np.linalg.norm(np.cross(corner - centre, axis)) > 4.0 + 2.6 + 0.2
        for i in range(1, 9):
            kind = nodes[i]
            if kind[0] == "shape" and kind[2] is STEPPED_POLYCONE:
                nodes.append(("shape", ORB, [2.5]))
                parents.append(i)
                xf.append(placement(rot(), (7.0, 0.0, -1.0)))
            elif kind[0] == "boolean" and kind[1].name == "box_minus_tube":
                nodes.append(("shape", BOX, [1.5, 1.5, 1.5]))
                parents.append(i)
                xf.append(placement(rot(), tuple(corner)))
        self.nodes = nodes
        self.parents = np.asarray(parents, dtype=np.int32)
        self.xforms = np.ascontiguousarray(np.stack(xf))
        self.level1 = np.arange(1, 9)

    tracks = WorldCase.tracks
    local_cube = 14.0


def mixed_world_case(**kw):
    return MixedWorldCase(**kw)


# ------------------------------------------------------------------ nested booleans (reading R31)

class CsgCase:
    """A CSG tree: `tree` is ("leaf", kind, params) or ("op", op, left, right, xform) with `xform` the row-major 3x4
    [R | b] from the frame of the node (= of its left operand) to the frame of its right operand."""

    def __init__(self, name, tree, center, half, seed):
        self.name, self.tree, self.center, self.half, self.seed = name, tree, tuple(center), tuple(half), seed

    def tracks(self, n, band=None):
        return draw_tracks(self.seed, n, self.center, self.half, band)

    def build(self, mod):
        """The tree as objects of `mod` (the oracle package or the CUDA binding: both have Shape and Boolean)."""
        def mk(t):
            if t[0] == "leaf":
                return mod.Shape(t[1], t[2])
            return mod.Boolean(t[1], mk(t[2]), mk(t[3]), t[4])
        return mk(self.tree)


def csg_cases():
    s2 = math.sqrt(0.5)
    ident = placement(np.eye(3), (0, 0, 0))
    rx = quaternion_to_matrix((s2, 0.0, 0.0, s2))
    rq = quaternion_to_matrix((0.18257418583505536, 0.3651483716701107, 0.5477225575051661, 0.7302967433402214))
    leaf = lambda k, p: ("leaf", k, [float(v) for v in p])
    seed = BASE_SEED + 700
    rounded = ("op", INTERSECTION, leaf(BOX, [5, 5, 5]), leaf(ORB, [6.5]), ident)
    return [
        CsgCase("rounded_cube_with_bore", ("op", SUBTRACTION, rounded, leaf(TUBE, [0, 2, 10, 0, TWO_PI]), placement(rq, (0.5, -0.5, 0.0))),
                (0, 0, 0), (8, 8, 8), seed),
        CsgCase("three_way_union", ("op", UNION, ("op", UNION, leaf(TUBE, [5, 10, 15, 0, 4 * math.pi / 3]), leaf(BOX, [4, 4, 20]),
                                                   placement(rq, (6.0, -2.0, 1.0))),
                                    leaf(CONE, [0, 3, 0, 8, 10, 0, TWO_PI]), placement(rx, (-9.0, 4.0, 0.0))),
                (0, 0, 0), (22, 22, 26), seed + 1),
        CsgCase("box_minus_union", ("op", SUBTRACTION, leaf(BOX, [10, 10, 10]),
                                    ("op", UNION, leaf(ORB, [5]), leaf(TUBE, [0, 3, 14, 0, TWO_PI]), placement(rx, (0.0, 0.0, 2.0))),
                                    placement(rq, (1.0, -1.0, 0.5))),
                (0, 0, 0), (14, 14, 14), seed + 2),
        CsgCase("twice_drilled_block_in_a_sphere",
                ("op", INTERSECTION,
                 ("op", SUBTRACTION, ("op", SUBTRACTION, leaf(BOX, [9, 9, 9]), leaf(TUBE, [0, 3, 12, 0, TWO_PI]), ident),
                  leaf(TUBE, [0, 2.5, 12, 0, TWO_PI]), placement(rx, (0.0, 1.0, 0.0))),
                 leaf(ORB, [11]), placement(np.eye(3), (1.0, 0.0, -1.0))),
                (0, 0, 0), (13, 13, 13), seed + 3),
    ]
