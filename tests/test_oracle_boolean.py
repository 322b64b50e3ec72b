"""Pins of the oracle's boolean solids (readings R27-R29 in oracle/vg_oracle.c and DESIGN.md; "boolean
operations", "logical operations").  Expectations come from the set definitions in tests/geomdefs.py
(membership written out in numpy), from closed-form reductions to a single primitive, and from ray marching."""
import math

import numpy as np
import pytest

import geomdefs as G
import oracle as O
import workloads as W

CASES = {bc.name: bc for bc in W.boolean_cases()}
IDENT = [1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]


def build(bc):
    return O.Boolean(bc.op, O.Shape(bc.kind_a, bc.par_a), O.Shape(bc.kind_b, bc.par_b), bc.xform)


def to_b(xf, x, y, z):
    M = np.asarray(xf, dtype=np.float64).reshape(3, 4)
    L = M[:, :3] @ np.stack([x, y, z]) + M[:, 3:4]
    return L[0], L[1], L[2]


def member(bc, x, y, z):
    """Set definition of C = A op B on the closed sets (c.1 + R27), independent of the oracle."""
    ma = G.member(bc.kind_a, bc.par_a, x, y, z)
    mb = G.member(bc.kind_b, bc.par_b, *to_b(bc.xform, x, y, z))
    return {W.UNION: ma | mb, W.INTERSECTION: ma & mb, W.SUBTRACTION: ma & ~mb}[bc.op]


def tracks(bc, c, n):
    return bc.tracks(n, lambda x, y, z: np.abs(c.sdf(x, y, z)) < W.SURFACE_BAND)


@pytest.mark.parametrize("name", ["tube", "cone_seg", "polycone_step", "box", "trd", "orb"])
def test_all_crossings_alternate_membership(name):
    """Every crossing flips the membership: midpoints between consecutive crossings alternate, the first interval has the
    membership of the start point, the count is even outside / odd inside, and the first entry is Cross."""
    shapes = {"tube": (O.TUBE, [5.0, 10.0, 15.0, 0.0, 4 * math.pi / 3]), "cone_seg": (O.CONE, [2.0, 6.0, 4.0, 12.0, 20.0, 0.3, 5.9]),
              "polycone_step": (O.POLYCONE, [0.0, 7.0, 4, -10, 2, 5, 0, 2, 5, 0, 3, 9, 6, 3, 9]), "box": (O.BOX, [5.0, 5.0, 5.0]),
              "trd": (O.TRD, [5.0, 10.0, 7.0, 3.0, 15.0]), "orb": (O.ORB, [20.0])}
    kind, par = shapes[name]
    s = O.Shape(kind, par)
    c, h = W.bounding_half(kind, par)
    x, y, z, dx, dy, dz = W.draw_tracks(31, 3000, c, tuple(1.5 * v for v in h), lambda x, y, z: np.abs(s.sdf(x, y, z)) < 1e-6)
    first = s.cross(x, y, z, dx, dy, dz)
    counts = []
    for i in range(x.size):
        p, d = np.array([x[i], y[i], z[i]]), np.array([dx[i], dy[i], dz[i]])
        t = s.all_crossings(p, d)
        counts.append(t.size)
        start_in = bool(G.member(kind, par, *p))
        assert t.size % 2 == (1 if start_in else 0)
        assert (t.size == 0 and math.isinf(first[i])) or t[0] == first[i]
        assert np.all(np.diff(t) >= 0)
        if t.size and np.min(np.diff(np.concatenate([[0.0], t]))) > 1e-6:
            mids = 0.5 * (np.concatenate([[0.0], t]) + np.concatenate([t, [t[-1] + 1.0]]))
            mem = G.member(kind, par, *(p[:, None] + mids * d[:, None]))
            want = np.arange(mids.size) % 2 == (0 if start_in else 1)
            assert np.array_equal(mem, want), (i, t, mem)
    assert max(counts) >= (4 if name in ("tube", "cone_seg", "polycone_step") else 2)


@pytest.mark.parametrize("name", list(CASES))
def test_inside_and_sdf_sign_are_the_set_operation(name):
    bc = CASES[name]
    c = build(bc)
    x, y, z = tracks(bc, c, 60000)[:3]
    mem = member(bc, x, y, z)
    cls = c.inside(x, y, z)
    assert np.array_equal(cls == O.INSIDE, mem) and np.array_equal(cls == O.OUTSIDE, ~mem)
    assert np.array_equal(c.sdf(x, y, z) < 0, mem)
    assert 0.01 < mem.mean() < 0.6


@pytest.mark.parametrize("name", list(CASES))
def test_composed_safety_never_overestimates(name):
    """R29: |sdf_C| <= distance to the boundary of C.  Checked against the first boundary crossing in 400 directions per
    point (an upper bound of the true distance that comes close to it) and against a membership probe: the ball of radius
    |sdf_C| around p holds no point of the other membership."""
    bc = CASES[name]
    c = build(bc)
    x, y, z = tracks(bc, c, 300)[:3]
    s = c.sdf(x, y, z)
    mem = member(bc, x, y, z)
    rng = np.random.default_rng(5)
    v = rng.normal(size=(3, 400))
    v /= np.linalg.norm(v, axis=0)
    for i in range(x.size):
        r = abs(s[i]) * (1 - 1e-9)
        q = member(bc, x[i] + r * v[0], y[i] + r * v[1], z[i] + r * v[2])
        assert np.all(q == mem[i]), (name, i)
        t = c.distance_to_out(np.full(400, x[i]), np.full(400, y[i]), np.full(400, z[i]), v[0], v[1], v[2]) if mem[i] else \
            c.distance_to_in(np.full(400, x[i]), np.full(400, y[i]), np.full(400, z[i]), v[0], v[1], v[2])
        assert abs(s[i]) <= t.min() * (1 + 1e-12)


@pytest.mark.parametrize("name", list(CASES))
def test_distances_land_on_the_boundary_and_flip_membership(name):
    bc = CASES[name]
    c = build(bc)
    x, y, z, dx, dy, dz = tracks(bc, c, 40000)
    cls = c.inside(x, y, z)
    din, dout = c.distance_to_in(x, y, z, dx, dy, dz), c.distance_to_out(x, y, z, dx, dy, dz)
    assert np.array_equal(din == -1.0, cls == O.INSIDE) and np.array_equal(dout == -1.0, cls == O.OUTSIDE)
    assert np.all(np.isfinite(dout[cls == O.INSIDE]))
    t = np.where(cls == O.INSIDE, dout, din)
    hit = np.isfinite(t)
    assert 0.02 < hit.mean() < 0.9
    tt = t[hit]
    hx, hy, hz = x[hit] + tt * dx[hit], y[hit] + tt * dy[hit], z[hit] + tt * dz[hit]
    assert np.max(np.abs(c.sdf(hx, hy, hz))) <= 1e-9  # the composed sdf vanishes on the boundary of C
    e = 1e-6
    before = member(bc, hx - e * dx[hit], hy - e * dy[hit], hz - e * dz[hit])
    after = member(bc, hx + e * dx[hit], hy + e * dy[hit], hz + e * dz[hit])
    assert np.mean(before != after) > 0.998
    assert np.array_equal(before[before != after], (cls[hit] == O.INSIDE)[before != after])
    # no earlier change of membership: sample the open segment (0, t) and the rays that miss
    for frac in (0.03, 0.25, 0.5, 0.75, 0.97):
        mid = member(bc, x[hit] + frac * tt * dx[hit], y[hit] + frac * tt * dy[hit], z[hit] + frac * tt * dz[hit])
        assert np.array_equal(mid, cls[hit] == O.INSIDE)
    miss = ~hit
    for far in (1.0, 7.0, 30.0, 100.0):
        assert not member(bc, x[miss] + far * dx[miss], y[miss] + far * dy[miss], z[miss] + far * dz[miss]).any()


@pytest.mark.parametrize("name", list(CASES))
def test_distance_equals_ray_marching(name):
    """Brute force: march the set-definition membership along the ray (step 5e-3), bisect the first flip."""
    bc = CASES[name]
    c = build(bc)
    x, y, z, dx, dy, dz = tracks(bc, c, 1500)
    cls = c.inside(x, y, z)
    t = np.where(cls == O.INSIDE, c.distance_to_out(x, y, z, dx, dy, dz), c.distance_to_in(x, y, z, dx, dy, dz))
    start = member(bc, x, y, z)
    tmax, h = 2.5 * max(bc.half) * math.sqrt(3), 5e-3
    found = np.full(x.size, np.inf)
    lo = np.zeros(x.size)
    for k in range(1, int(tmax / h) + 1):
        tk = k * h
        m = member(bc, x + tk * dx, y + tk * dy, z + tk * dz)
        new = (m != start) & np.isinf(found)
        found[new] = tk
        lo[np.isinf(found)] = tk
        if not np.isinf(found).any():
            break
    fl = np.isfinite(found)
    a, b = lo[fl].copy(), found[fl].copy()
    for _ in range(40):
        mid = 0.5 * (a + b)
        m = member(bc, x[fl] + mid * dx[fl], y[fl] + mid * dy[fl], z[fl] + mid * dz[fl])
        same = m == start[fl]
        a, b = np.where(same, mid, a), np.where(same, b, mid)
    march = np.full(x.size, np.inf)
    march[fl] = 0.5 * (a + b)
    # a feature thinner than the step can hide from the march, never from the oracle: oracle <= march, equal almost always
    assert np.all(t <= march + 1e-7)
    agree = np.isclose(t, march, rtol=0, atol=1e-7) | (np.isinf(t) & np.isinf(march))
    assert agree.mean() > 0.995, agree.mean()


def _five(s, t):
    return [s.inside(*t[:3]), s.distance_to_in(*t), s.distance_to_out(*t), s.safety_to_in(*t[:3]), s.safety_to_out(*t[:3])]


def _same(a, b, tol=1e-12):
    assert np.array_equal(a[0], b[0])
    for u, v in zip(a[1:], b[1:]):
        fin = np.isfinite(v)
        assert np.array_equal(fin, np.isfinite(u)) and np.array_equal(u[~fin], v[~fin])
        assert np.all(np.abs(u[fin] - v[fin]) <= tol * np.maximum(1.0, np.abs(v[fin])))


def test_reductions_to_one_primitive():
    """B inside A: A u B == A.  A inside B: A n B == A.  B apart from A: A - B == A.  All five queries, safeties included
    (the composed bound is exact when only one operand matters)."""
    a = O.Shape(O.TUBE, [5.0, 10.0, 15.0, 0.0, 4 * math.pi / 3])
    t = W.draw_tracks(41, 30000, (0, 0, 0), (15, 15, 22.5), lambda x, y, z: np.abs(a.sdf(x, y, z)) < 1e-6)
    small = O.Shape(O.ORB, [1.0])
    into = W.placement(W.quaternion_to_matrix((0.5, 0.5, 0.5, 0.5)), (-7.5, 0.5, 3.0))  # inside the tube wall
    _same(_five(O.Boolean(O.UNION, a, small, into), t), _five(a, t))
    big = O.Shape(O.BOX, [40.0, 40.0, 40.0])
    _same(_five(O.Boolean(O.INTERSECTION, a, big, W.placement(W.quaternion_to_matrix((0.5, -0.5, 0.5, 0.5)), (1, 2, 3))), t), _five(a, t))
    # subtraction: compare on the points that are not inside the far-away box (its own interior belongs to neither)
    far = W.placement(np.eye(3), (60.0, 0.0, 0.0))
    _same(_five(O.Boolean(O.SUBTRACTION, a, O.Shape(O.BOX, [3.0, 3.0, 3.0]), far), t), _five(a, t))


def test_two_overlapping_boxes_are_a_box():
    """box(5,5,5) n box(5,5,5)@(4,0,0) == box(3,5,5)@(2,0,0); their union == box(7,5,5)@(2,0,0) (coincident side faces)."""
    a = O.Shape(O.BOX, [5.0, 5.0, 5.0])
    shift = W.placement(np.eye(3), (4.0, 0.0, 0.0))
    for op, hx in ((O.INTERSECTION, 3.0), (O.UNION, 7.0)):
        c = O.Boolean(op, a, a, shift)
        ref = O.Shape(O.BOX, [hx, 5.0, 5.0])
        t = W.draw_tracks(43, 30000, (2, 0, 0), (12, 9, 9), lambda x, y, z: np.abs(ref.sdf(x - 2.0, y, z)) < 1e-6)
        tr = (t[0] - 2.0,) + tuple(t[1:])
        got, want = _five(c, t), _five(ref, tr)
        _same(got[:3], want[:3])
        # safeties: exact inside an intersection of convex bodies and outside a union; a lower bound elsewhere
        sdf_c, sdf_r = got[3], want[3]
        exact = (sdf_r < 0) if op == O.INTERSECTION else (sdf_r > 0)
        assert np.max(np.abs(sdf_c[exact] - sdf_r[exact])) < 1e-12
        assert np.all(np.abs(sdf_c) <= np.abs(sdf_r) + 1e-12) and np.array_equal(sdf_c < 0, sdf_r < 0)


@pytest.mark.parametrize("name", list(CASES))
def test_rigid_motion_and_80bit(name):
    bc = CASES[name]
    c = build(bc)
    t = tracks(bc, c, 20000)
    ref = _five(c, t)
    # moving B's placement and nothing else must change results; moving it back restores them (guards a dropped xform)
    moved = O.Boolean(bc.op, c.a, c.b, W.placement(np.eye(3), (0.3, 0.0, 0.0)) if name != "box_union_orb" else W.placement(np.eye(3), (9, 9, 9)))
    assert not np.array_equal(moved.inside(*t[:3]), ref[0])
    ld = O.Boolean(bc.op, O.Shape(bc.kind_a, bc.par_a, long_double=True), O.Shape(bc.kind_b, bc.par_b, long_double=True), bc.xform)
    got = _five(ld, t)
    assert np.array_equal(got[0], ref[0])
    for u, v in zip(got[1:], ref[1:]):
        fin = np.isfinite(v)
        assert np.array_equal(fin, np.isfinite(u))
        assert np.max(np.abs(u[fin] - v[fin])) <= 1e-11


def test_invalid_booleans_are_rejected():
    a = O.Shape(O.BOX, [1, 1, 1])
    with pytest.raises(ValueError):
        O.Boolean(3, a, a, IDENT)
    with pytest.raises(ValueError):
        O.Boolean(O.UNION, a, a, [float("nan")] * 12)


# ------------------------------------------------------------------ nested booleans (reading R31)

CSG = {c.name: c for c in W.csg_cases()}


def csg_member(tree, x, y, z):
    """Set definition of a CSG tree on the closed sets, composed in numpy (independent of the oracle)."""
    if tree[0] == "leaf":
        return G.member(tree[1], tree[2], x, y, z)
    ma = csg_member(tree[2], x, y, z)
    mb = csg_member(tree[3], *to_b(tree[4], x, y, z))
    return {W.UNION: ma | mb, W.INTERSECTION: ma & mb, W.SUBTRACTION: ma & ~mb}[tree[1]]


def csg_band(c):
    """Clear of the surface of EVERY primitive of the tree (the contract of the distances, R7)."""
    leaves = c.leaves()

    def band(x, y, z):
        bad = np.zeros(np.shape(x), dtype=bool)
        for shape, M in leaves:
            L = M[:, :3] @ np.stack([x, y, z]) + M[:, 3:4]
            bad |= np.abs(shape.sdf(L[0], L[1], L[2])) < W.SURFACE_BAND
        return bad
    return band


@pytest.mark.parametrize("name", list(CSG))
def test_nested_boolean_membership_distances_and_safety(name):
    cc = CSG[name]
    c = cc.build(O)
    x, y, z, dx, dy, dz = cc.tracks(30000, csg_band(c))
    mem = csg_member(cc.tree, x, y, z)
    cls = c.inside(x, y, z)
    assert np.array_equal(cls == O.INSIDE, mem) and np.array_equal(cls == O.OUTSIDE, ~mem)
    assert 0.03 < mem.mean() < 0.7
    s = c.sdf(x, y, z)
    assert np.array_equal(s < 0, mem)
    din, dout = c.distance_to_in(x, y, z, dx, dy, dz), c.distance_to_out(x, y, z, dx, dy, dz)
    assert np.array_equal(din == -1.0, mem) and np.array_equal(dout == -1.0, ~mem)
    t = np.where(mem, dout, din)
    hit = np.isfinite(t)
    assert np.all(hit[mem]) and 0.05 < hit.mean() < 0.95
    tt = t[hit]
    hx, hy, hz = x[hit] + tt * dx[hit], y[hit] + tt * dy[hit], z[hit] + tt * dz[hit]
    assert np.max(np.abs(c.sdf(hx, hy, hz))) <= 1e-9
    e = 1e-6
    before = csg_member(cc.tree, hx - e * dx[hit], hy - e * dy[hit], hz - e * dz[hit])
    after = csg_member(cc.tree, hx + e * dx[hit], hy + e * dy[hit], hz + e * dz[hit])
    assert np.mean(before != after) > 0.997
    for frac in (0.03, 0.3, 0.6, 0.97):
        mid = csg_member(cc.tree, x[hit] + frac * tt * dx[hit], y[hit] + frac * tt * dy[hit], z[hit] + frac * tt * dz[hit])
        assert np.array_equal(mid, mem[hit])
    for far in (0.5, 3.0, 12.0, 60.0):
        assert not csg_member(cc.tree, x[~hit] + far * dx[~hit], y[~hit] + far * dy[~hit], z[~hit] + far * dz[~hit]).any()
    assert np.all(np.abs(s)[hit] <= tt * (1 + 1e-12))  # the composed safety never exceeds a distance


def test_nested_boolean_reductions():
    """(A u small-inside-A) - C == A - C; regrouping a union changes nothing; A n (B n C) == (A n B) n C."""
    a = O.Shape(O.BOX, [8, 8, 8])
    small = O.Shape(O.ORB, [1.0])
    tube = O.Shape(O.TUBE, [0, 3, 12, 0, 2 * math.pi])
    orb = O.Shape(O.ORB, [9.5])
    q = W.quaternion_to_matrix((0.5, 0.5, 0.5, 0.5))
    p_small, p_tube, p_orb = W.placement(np.eye(3), (4.0, 4.0, 4.0)), W.placement(q, (1.0, 0.0, -1.0)), W.placement(np.eye(3), (1.0, 1.0, 0.0))
    flat = O.Boolean(O.SUBTRACTION, a, tube, p_tube)
    nested = O.Boolean(O.SUBTRACTION, O.Boolean(O.UNION, a, small, p_small), tube, p_tube)
    t = W.draw_tracks(51, 30000, (0, 0, 0), (12, 12, 12), csg_band(nested))
    _same(_five(nested, t), _five(flat, t))
    # ((a n orb) n tube) == (a n (orb n tube')) with tube' placed relative to the orb's frame
    left = O.Boolean(O.INTERSECTION, O.Boolean(O.INTERSECTION, a, orb, p_orb), tube, p_tube)
    Mo = np.vstack([np.asarray(p_orb).reshape(3, 4), [0, 0, 0, 1]])
    Mt = np.vstack([np.asarray(p_tube).reshape(3, 4), [0, 0, 0, 1]])
    rel = (Mt @ np.linalg.inv(Mo))[:3].reshape(12)  # frame of the orb -> frame of the tube
    right = O.Boolean(O.INTERSECTION, a, O.Boolean(O.INTERSECTION, orb, tube, rel), p_orb)
    t = W.draw_tracks(52, 30000, (0, 0, 0), (12, 12, 12), csg_band(left))
    _same(_five(left, t), _five(right, t), tol=1e-11)
    lu = O.Boolean(O.UNION, O.Boolean(O.UNION, a, orb, p_orb), tube, p_tube)
    ru = O.Boolean(O.UNION, a, O.Boolean(O.UNION, orb, tube, rel), p_orb)
    _same(_five(lu, t), _five(ru, t), tol=1e-11)
    with pytest.raises(ValueError):  # more than eight primitives
        big = a
        for _ in range(8):
            big = O.Boolean(O.UNION, big, small, p_small)
