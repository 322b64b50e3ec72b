"""CPU pin of ComputeStep's conservative cull (csrc/vg_nav_cull.h).

The kernel skips daughters whose DistanceToIn must be +inf: a 3-D walk of a candidate grid in FP64, then an FP32 ray /
bounding-sphere test.  A wrong bound would silently drop a hit, so the very code the kernel runs (the header is
compiled for host and device and rounds identically) is evaluated here on the CPU through the host-only export
`vg_debug_nav_cull` and checked against the oracle: NO daughter with a finite oracle DistanceToIn (not beyond the
ray-parameter limit) may be missing from the mask -- for both stages together and for each stage alone -- on rays built
to graze: through box corners (which lie ON the bounding sphere) at a tangent, through the grid's own cell edges and
corners, with one direction component ~1e-8 or exactly 0, in mothers of half-length 1e4 around daughters of radius 1e-2.
"""
import math

import numpy as np
import pytest

import oracle as O
import paper_1512_06637_b200 as vg
import workloads as W


def unit(v):
    with np.errstate(divide="ignore", invalid="ignore"):  # a zero vector stays non-finite: the callers replace or reject it
        return v / np.linalg.norm(v, axis=-1, keepdims=True)


def isotropic(rng, n):
    dz = rng.uniform(-1, 1, n)
    ph = rng.uniform(0, 2 * math.pi, n)
    s = np.sqrt(1 - dz * dz)
    return unit(np.stack([s * np.cos(ph), s * np.sin(ph), dz], axis=1))


class Scene:
    def __init__(self, mother_kind, mother_params, kinds, params, xforms):
        self.mk, self.mp, self.kinds, self.params = mother_kind, mother_params, kinds, params
        self.xf = np.ascontiguousarray(xforms, dtype=np.float64).reshape(len(kinds), 12)
        self.o_mother = O.Shape(mother_kind, mother_params)
        self.o_d = [O.Shape(k, p) for k, p in zip(kinds, params)]
        self.g_mother = vg.Shape(mother_kind, mother_params)
        self.g_d = [vg.Shape(k, p) for k, p in zip(kinds, params)]
        M = self.xf.reshape(-1, 3, 4)
        self.R, self.b = M[:, :, :3], M[:, :, 3]
        self.centers = -np.einsum("nji,nj->ni", self.R, self.b)  # c = -R^T b

    def masks(self, P, D, t_lim=None, stage=0):
        return vg.vg_debug_nav_cull(self.g_mother, self.g_d, self.xf, P[:, 0], P[:, 1], P[:, 2], D[:, 0], D[:, 1], D[:, 2],
                                    t_lim, stage)

    def oracle_tin(self, P, D):
        """(nd, n) oracle DistanceToIn of every daughter, each in its own frame (reading R12)."""
        out = np.empty((len(self.kinds), len(P)))
        for k, s in enumerate(self.o_d):
            L = P @ self.R[k].T + self.b[k]
            Ld = D @ self.R[k].T
            out[k] = s.distance_to_in(L[:, 0], L[:, 1], L[:, 2], Ld[:, 0], Ld[:, 1], Ld[:, 2])
        return out

    def check(self, P, D, what, limit_by_mother=True):
        P, D = np.ascontiguousarray(P), np.ascontiguousarray(D)
        tin = self.oracle_tin(P, D)
        tl = self.o_mother.distance_to_out(P[:, 0], P[:, 1], P[:, 2], D[:, 0], D[:, 1], D[:, 2]) if limit_by_mother else None
        must = np.isfinite(tin) & (tin >= 0)
        if tl is not None:
            must &= tin <= tl
        nd = len(self.kinds)
        kept_total = 0
        for stage in (0, 1, 2):
            m, _ = self.masks(P, D, tl if stage != 2 else None, stage)
            bits = np.zeros((nd, len(P)), dtype=bool)
            for k in range(nd):
                bits[k] = (m[:, k // 64] >> np.uint64(k % 64)) & np.uint64(1) == 1
            lost = must & ~bits
            assert not lost.any(), "%s, stage %d: %d hits culled, first (daughter, ray) %s" % (
                what, stage, lost.sum(), np.argwhere(lost)[:3].tolist())
            if stage == 0:
                kept_total = bits.sum()
        # the physics step as the limit, set exactly at the nearest hit: that daughter (tin == t_lim) must survive
        tmin = np.where(must, tin, np.inf).min(axis=0)
        sel = np.isfinite(tmin)
        if sel.any():
            for stage in (0, 1):
                m, _ = self.masks(P[sel], D[sel], tmin[sel], stage)
                win = np.where(must, tin, np.inf).argmin(axis=0)[sel]
                got = (m[np.arange(len(win)), win // 64] >> (win % 64).astype(np.uint64)) & np.uint64(1)
                assert np.all(got == 1), "%s, stage %d: the daughter hit exactly at the limit was culled (%d rays)" % (
                    what, stage, (got != 1).sum())
        return must.sum(), kept_total


# ------------------------------------------------------------------------------------------------ ray generators

def clip_into(P, half):
    return np.clip(P, -np.asarray(half) * (1 - 1e-9), np.asarray(half) * (1 - 1e-9))


def random_rays(sc, rng, n, half):
    return rng.uniform(-1, 1, (n, 3)) * np.asarray(half), isotropic(rng, n)


def surface_points(sc, rng, n):
    """Points on (or a hair off) the daughters' own surfaces, corners and edges included, in the mother frame."""
    nd = len(sc.kinds)
    H = np.zeros((nd, 3))    # box-like half-extents
    RZ = np.zeros((nd, 2))   # rmax, dz of the round solids
    for j, (kind, par) in enumerate(zip(sc.kinds, sc.params)):
        if kind == W.BOX:
            H[j] = par[:3]
        elif kind == W.TRD:
            H[j] = [max(par[0], par[1]), max(par[2], par[3]), par[4]]
        elif kind == W.ORB:
            RZ[j] = [par[0], 0.0]
        elif kind == W.TUBE:
            RZ[j] = [par[1], par[2]]
        else:
            RZ[j] = [max(par[1], par[3]), par[4]]
    kinds = np.asarray(sc.kinds)
    k = rng.integers(0, nd, n)
    u = rng.uniform(-1, 1, (n, 3))
    snap = rng.random((n, 3)) < 0.6  # faces, edges (two snapped) and corners (three)
    u = np.where(snap, np.where(u < 0, -1.0, 1.0), u)
    loc_box = u * H[k]
    loc_orb = isotropic(rng, n) * RZ[k, :1]
    ph = rng.uniform(0, 2 * math.pi, n)
    r = np.where(rng.random(n) < 0.7, 1.0, rng.random(n)) * RZ[k, 0]  # the rim circles touch the bounding sphere
    zz = np.where(rng.random(n) < 0.7, rng.choice([-1.0, 1.0], n), rng.uniform(-1, 1, n)) * RZ[k, 1]
    loc_rz = np.stack([r * np.cos(ph), r * np.sin(ph), zz], axis=1)
    kk = kinds[k][:, None]
    loc = np.where((kk == W.BOX) | (kk == W.TRD), loc_box, np.where(kk == W.ORB, loc_orb, loc_rz))
    loc = loc * (1 + rng.choice([0.0, 1e-12, -1e-12, 1e-9, -1e-9, 1e-7, -1e-7], (n, 1)))
    Q = np.einsum("nji,nj->ni", sc.R[k], loc - sc.b[k])  # R^T (loc - b)
    return k, Q


def aimed_rays(sc, rng, n, half):
    """From random start points straight at surface points of the daughters."""
    _, Q = surface_points(sc, rng, n)
    P = rng.uniform(-1, 1, (n, 3)) * np.asarray(half)
    return P, unit(Q - P + 1e-300)


def tangent_rays(sc, rng, n, half):
    """Through a surface point of a daughter at a tangent to the sphere about the daughter's centre through that
    point (for a corner: the bounding sphere itself), the start point moved +-eps along the radius."""
    k, Q = surface_points(sc, rng, n)
    rad = Q - sc.centers[k]
    rn = np.linalg.norm(rad, axis=1, keepdims=True)
    rad = rad / np.maximum(rn, 1e-300)
    T = np.cross(rad, isotropic(rng, n))
    T = unit(T + 1e-300)
    s = rng.uniform(0, 1, (n, 1)) ** 2 * 2 * max(half)
    eps = rng.choice([0.0, 1e-13, -1e-13, 1e-9, -1e-9, 1e-7, -1e-7, 1e-5, -1e-5, -1e-3], (n, 1)) * rn
    P = clip_into(Q - s * T + eps * rad, half)
    return P, unit(Q + eps * rad - P + 1e-300 * T)


def grid_rays(sc, rng, n, half, grid):
    """Start points on the candidate grid's own cell planes, edges and corners, directions along the axes, the plane and
    space diagonals, and aimed at other grid corners: the walk's ties."""
    o, cs, g = grid[:3], grid[3:6], grid[6:9].astype(int)
    P = rng.uniform(-1, 1, (n, 3)) * np.asarray(half)
    snap = rng.random((n, 3)) < 0.7
    node = o + cs * np.stack([rng.integers(0, g[a] + 1, n) for a in range(3)], axis=1)
    P = clip_into(np.where(snap, node, P), half)
    D = isotropic(rng, n)
    mode = rng.integers(0, 4, n)
    sgn = rng.choice([-1.0, 1.0], (n, 3))
    axis = np.eye(3)[rng.integers(0, 3, n)] * sgn
    diag2 = sgn * (np.ones((n, 3)) - np.eye(3)[rng.integers(0, 3, n)]) * cs
    diag3 = sgn * cs
    D = np.where((mode == 0)[:, None], axis, D)
    D = np.where((mode == 1)[:, None], unit(diag2), D)
    D = np.where((mode == 2)[:, None], unit(diag3), D)
    node2 = o + cs * np.stack([rng.integers(0, g[a] + 1, n) for a in range(3)], axis=1)
    aim = unit(node2 - P + 1e-300)
    D = np.where((mode == 3)[:, None] & (np.linalg.norm(node2 - P, axis=1, keepdims=True) > 1e-9), aim, D)
    return P, D


def tiny_component_rays(sc, rng, n, half):
    P, D = aimed_rays(sc, rng, n, half)
    a = rng.integers(0, 3, n)
    D[np.arange(n), a] = rng.choice([0.0, 1e-8, -1e-8, 1e-12, 1e-300, -0.0], n)
    bad = np.linalg.norm(D, axis=1) < 1e-3
    D[bad] = np.array([0.0, 0.6, 0.8])
    return P, unit(D)


# ------------------------------------------------------------------------------------------------------- scenes

def config4_scene():
    nav = W.navigator_case()
    return Scene(nav.mother_kind, nav.mother_params, nav.daughter_kinds, nav.daughter_params, nav.xforms), nav.half


def random_scene(seed, nd, mother_half, size, spread, kinds=(W.BOX, W.ORB, W.TUBE, W.CONE, W.TRD)):
    """nd daughters of mixed kinds, characteristic size `size`, centres uniform in +-spread, random rotations (overlaps
    do not matter for the cull)."""
    rng = np.random.default_rng(seed)
    ks, ps, xf = [], [], []
    for _ in range(nd):
        kind = kinds[rng.integers(0, len(kinds))]
        a, b, c = size * rng.uniform(0.3, 1.0, 3)
        par = {W.BOX: [a, b, c], W.ORB: [a], W.TUBE: [0.3 * a, a, b, 0.0, 2 * math.pi],
               W.CONE: [0.2 * a, a, 0.3 * b, 1.2 * b, c, 0.0, 2 * math.pi], W.TRD: [a, 0.5 * a, b, 1.3 * b, c]}[kind]
        q = rng.normal(size=4)
        q /= np.linalg.norm(q)
        ks.append(kind)
        ps.append(par)
        xf.append(W.placement(W.quaternion_to_matrix(tuple(q)), rng.uniform(-spread, spread, 3)))
    return Scene(W.BOX, [mother_half] * 3, ks, ps, np.stack(xf)), (mother_half,) * 3


def run_all_generators(sc, half, seed, n_each):
    rng = np.random.default_rng(seed)
    _, grid = sc.masks(np.zeros((1, 3)), np.array([[0.0, 0.0, 1.0]]))
    hits = kept = rays = 0
    for name, gen in (("random", random_rays), ("aimed", aimed_rays), ("tangent", tangent_rays),
                      ("tiny component", tiny_component_rays), ("grid", lambda s, r, n, h: grid_rays(s, r, n, h, grid))):
        P, D = gen(sc, rng, n_each, half)
        h, k = sc.check(P, D, name)
        hits, kept, rays = hits + h, kept + k, rays + len(P)
    return hits, kept, rays


# -------------------------------------------------------------------------------------------------------- tests

def test_no_hit_is_culled_on_configs4_geometry():
    """>= 10^6 adversarial rays through the 64 daughters of configs[4]; the masks must also prune."""
    sc, half = config4_scene()
    hits, kept, rays = run_all_generators(sc, half, 20261104, 210000)
    assert rays >= 1000000 and hits > 0.5 * rays  # the generators do aim: most rays hit something
    assert kept < 2.5 * hits and kept < 3.0 * rays  # <= 3 of 64 daughters survive per ray: the cull prunes


@pytest.mark.parametrize("nd, mother_half, size, spread", [
    (64, 1e4, 1e-2, 1e4 * 0.9),    # tiny daughters in a huge mother: FP32 cannot resolve them, the bound must cover it
    (64, 1e4, 1e-2, 1.0),          # ... clustered near the origin
    (200, 100.0, 6.0, 90.0),       # four chunks of 64, five kinds
    (100, 50.0, 20.0, 30.0),       # two chunks, heavy overlap: many candidates per cell
    (1, 10.0, 3.0, 5.0),           # one cell
    (2, 10.0, 1.0, 8.0),
    (9, 1e3, 50.0, 900.0),
])
def test_no_hit_is_culled_in_random_scenes(nd, mother_half, size, spread):
    sc, half = random_scene(nd * 1000 + int(size * 7), nd, mother_half, size, spread)
    hits, kept, rays = run_all_generators(sc, half, nd, 20000)
    assert hits > 0


def test_flat_scenes_and_start_points_outside_the_mother():
    """Daughters in one plane / on one line (a grid axis of zero extent before padding), and start points outside the
    mother's bounding sphere: out of contract, every daughter is kept."""
    rng = np.random.default_rng(5)
    for axes in ((1, 1, 0), (1, 0, 0)):
        ks = [W.ORB] * 8
        ps = [[1.0]] * 8
        xf = [W.placement(np.eye(3), rng.uniform(-20, 20, 3) * np.asarray(axes)) for _ in range(8)]
        sc = Scene(W.BOX, [30.0] * 3, ks, ps, np.stack(xf))
        run_all_generators(sc, (30.0,) * 3, 7, 20000)
    sc, half = config4_scene()
    P = isotropic(rng, 1000) * 400.0
    D = unit(rng.uniform(-100, 100, (1000, 3)) - P)
    m, _ = sc.masks(P, D)
    assert np.all(m[:, 0] == np.uint64(0xFFFFFFFFFFFFFFFF)) and np.all(m[:, 1:] == 0)
    tin = sc.oracle_tin(P, D)
    assert np.isfinite(tin).any()


def test_the_cell_of_a_point_lists_every_daughter_that_holds_it():
    """World Locate in a node with many children -- and vg_volume_safety for a point inside a daughter or outside the
    mother -- test only the daughters listed in the point's grid cell: every daughter
    whose Inside (oracle) is INSIDE or SURFACE at the point must be in that mask -- random points, points on the daughters'
    surfaces and points on the grid's own cell planes, edges and corners."""
    rng = np.random.default_rng(11)
    for sc, half in (config4_scene(), random_scene(4242, 40, 50.0, 12.0, 35.0), random_scene(77, 64, 1e3, 60.0, 800.0),
                     random_scene(99, 200, 100.0, 6.0, 90.0)):  # (four chunks of 64: what vg_volume_safety looks up)
        _, grid = sc.masks(np.zeros((1, 3)), np.array([[0.0, 0.0, 1.0]]))
        o, cs, g = grid[:3], grid[3:6], grid[6:9].astype(int)
        n = 200000 if len(sc.kinds) <= 64 else 50000  # (the oracle evaluates every daughter at every point)
        P = rng.uniform(-1, 1, (n, 3)) * np.asarray(half)
        _, Q = surface_points(sc, rng, n)
        node = o + cs * np.stack([rng.integers(0, g[a] + 1, n) for a in range(3)], axis=1)
        snapped = np.where(rng.random((n, 3)) < 0.6, node, rng.uniform(-1, 1, (n, 3)) * np.asarray(half))
        for pts, what in ((P, "random"), (Q, "on a daughter's surface"), (snapped, "on the grid's planes")):
            pts = np.ascontiguousarray(pts)
            m, _ = sc.masks(pts, np.tile([0.0, 0.0, 1.0], (len(pts), 1)), None, 3)
            for k, s in enumerate(sc.o_d):
                L = pts @ sc.R[k].T + sc.b[k]
                holds = s.inside(L[:, 0], L[:, 1], L[:, 2]) != O.OUTSIDE
                bit = (m[:, k // 64] >> np.uint64(k % 64)) & np.uint64(1) == 1
                assert not (holds & ~bit).any(), "%s: daughter %d holds %d points that its cell does not list" % (what, k, (holds & ~bit).sum())


def test_the_safety_cell_of_a_point_lists_its_nearest_daughter():
    """vg_volume_safety / vg_world_safety evaluate only the daughters listed in the point's cell of the safety grid
    (vg_nav_cull.h, nav_safety_cell; stage 4): the minimum over the LISTED daughters of the oracle's SafetyToIn must be
    the minimum over ALL of them, bit for bit -- random points, points on the daughters' surfaces, on the planes, edges
    and corners of the safety grid itself, and points outside the grid's box (every daughter kept).  The lists must
    also prune, and a grid must exist where this test means to exercise one."""
    rng = np.random.default_rng(2027)
    scenes = (config4_scene(), random_scene(4242, 40, 50.0, 12.0, 35.0), random_scene(77, 64, 1e3, 60.0, 800.0),
              random_scene(99, 200, 100.0, 6.0, 90.0), random_scene(5, 100, 50.0, 20.0, 30.0), random_scene(8, 8, 1e4, 1e-2, 0.9e4),
              random_scene(3, 5, 10.0, 2.0, 6.0))
    for si, (sc, half) in enumerate(scenes):
        nd = len(sc.kinds)
        _, grid = sc.masks(np.zeros((1, 3)), np.array([[0.0, 0.0, 1.0]]), None, 4)
        o, ext, gs = grid[:3], grid[3:6] * grid[6:9], int(grid[9])
        assert (gs > 0) == (nd >= 8), "scene %d: %d daughters, safety grid of %d cells per axis" % (si, nd, gs)
        n = 60000 if nd <= 64 else 20000  # (the oracle evaluates every daughter at every point)
        P = rng.uniform(-1, 1, (n, 3)) * np.asarray(half)
        _, Q = surface_points(sc, rng, n)
        g1 = max(gs, 1)
        node = o + ext / g1 * np.stack([rng.integers(0, g1 + 1, n) for a in range(3)], axis=1)
        node = node * (1 + rng.choice([0.0, 1e-16, -1e-16, 1e-13, -1e-13], (n, 1)))
        snapped = np.where(rng.random((n, 3)) < 0.6, node, rng.uniform(-1, 1, (n, 3)) * np.asarray(half))
        outside = (o + ext * rng.uniform(-0.2, 1.2, (n, 3)))
        listed = 0
        for pts, what in ((P, "random"), (Q, "on a daughter's surface"), (snapped, "on the safety grid's planes"), (outside, "around the box")):
            pts = np.ascontiguousarray(pts)
            m, _ = sc.masks(pts, np.tile([0.0, 0.0, 1.0], (len(pts), 1)), None, 4)
            s_all = np.empty((nd, len(pts)))
            bits = np.zeros((nd, len(pts)), dtype=bool)
            for k, s in enumerate(sc.o_d):
                L = pts @ sc.R[k].T + sc.b[k]
                s_all[k] = s.safety_to_in(L[:, 0], L[:, 1], L[:, 2])
                bits[k] = (m[:, k // 64] >> np.uint64(k % 64)) & np.uint64(1) == 1
            assert not (m[:, (nd + 63) // 64:] != 0).any() and bits.any(axis=0).all()
            want = s_all.min(axis=0)
            got = np.where(bits, s_all, np.inf).min(axis=0)
            bad = got != want
            assert not bad.any(), "scene %d, %s: the nearest daughter of %d points is not listed, first %s (listed min %r, min %r)" % (
                si, what, bad.sum(), pts[bad][0].tolist(), got[bad][0], want[bad][0])
            inbox = np.all((pts >= o) & (pts <= o + ext), axis=1)
            if gs == 0:
                assert bits.all()
            else:
                assert bits[:, ~inbox].all()  # outside the box: no cell, every daughter
            if what == "random":
                listed = bits[:, inbox].sum() / max(1, inbox.sum())
        if si == 0:
            assert listed < 12.0, "configs[4]: %.1f of 64 daughters listed per cell: the grid does not prune" % listed


def test_the_walk_lists_every_daughter_whose_bounding_sphere_the_ray_meets():
    """The grid walk on its own (stage 1), against geometry written out here: every daughter whose TRUE bounding sphere
    (centre -R^T b, radius of the solid about its origin, no inflation) is met by the ray between the start point and
    the limit must be in the walk's mask -- a tighter statement than 'no hit is culled' (the spheres are much larger
    than the solids), and the one the walk's rounding margins (FP32 stepping, padded cells) have to deliver.  Rays along
    the grid's planes, edges and diagonals, tangent rays, rays with tiny components, limits set exactly at the sphere."""
    for si, (sc, half) in enumerate((config4_scene(), random_scene(4242, 40, 50.0, 12.0, 35.0), random_scene(8, 64, 1e4, 1e-2, 0.9e4),
                                     random_scene(99, 200, 100.0, 6.0, 90.0), random_scene(5, 100, 50.0, 20.0, 30.0))):
        nd = len(sc.kinds)
        rad = np.zeros(nd)
        for j, (kind, par) in enumerate(zip(sc.kinds, sc.params)):
            if kind == W.BOX:
                rad[j] = np.linalg.norm(par[:3])
            elif kind == W.TRD:
                rad[j] = np.linalg.norm([max(par[0], par[1]), max(par[2], par[3]), par[4]])
            elif kind == W.ORB:
                rad[j] = par[0]
            elif kind == W.TUBE:
                rad[j] = math.hypot(par[1], par[2])
            else:
                rad[j] = math.hypot(max(par[1], par[3]), par[4])
        rng = np.random.default_rng(31 + si)
        _, grid = sc.masks(np.zeros((1, 3)), np.array([[0.0, 0.0, 1.0]]))
        for name, gen in (("random", random_rays), ("aimed", aimed_rays), ("tangent", tangent_rays),
                          ("tiny component", tiny_component_rays), ("grid", lambda s, r, n, h: grid_rays(s, r, n, h, grid))):
            P, D = gen(sc, rng, 40000, half)
            P, D = np.ascontiguousarray(P), np.ascontiguousarray(D)
            inside_mother = sc.o_mother.inside(P[:, 0], P[:, 1], P[:, 2]) != O.OUTSIDE
            P, D = P[inside_mother], D[inside_mother]
            V = sc.centers[:, None, :] - P[None, :, :]                      # (nd, n, 3)
            tca = np.einsum("knj,nj->kn", V, D)
            d2 = np.einsum("knj,knj->kn", V, V) - tca * tca
            r2 = (rad * rad)[:, None]
            thc = np.sqrt(np.maximum(r2 - d2, 0.0))
            t_in, t_out = tca - thc, tca + thc                               # the ray is inside the sphere for t in [t_in, t_out]
            met = (d2 <= r2 * (1 - 1e-12)) & (t_out >= 0)
            first = np.where(met, np.maximum(t_in, 0.0), np.inf)
            for t_lim in (None, np.where(np.isfinite(first.min(axis=0)), first.min(axis=0), 1.0)):
                must = met if t_lim is None else met & (first <= t_lim[None, :])
                m, _ = sc.masks(P, D, t_lim, 1)
                bits = np.zeros((nd, len(P)), dtype=bool)
                for k in range(nd):
                    bits[k] = (m[:, k // 64] >> np.uint64(k % 64)) & np.uint64(1) == 1
                lost = must & ~bits
                assert not lost.any(), "scene %d, %s rays, limit %s: the walk misses %d (daughter, ray) pairs whose sphere the ray meets, first %s" % (
                    si, name, "none" if t_lim is None else "at the nearest sphere", lost.sum(), np.argwhere(lost)[:3].tolist())
