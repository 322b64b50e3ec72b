"""Pins of the oracle against what the definitions and the mathematics fix.

The paper prints no worked example (PAPER.md:110-120 only states the three questions), so every pin is
a hand-derived closed form (tests/golden/worked_examples.txt), a textbook routine the query reduces to,
an invariant, a reduction between solids, or brute force on tiny inputs.  None of them calls the CUDA path.
"""
import math
import os

import numpy as np
import pytest

import geomdefs as G
import oracle as O
import workloads as W

PI = math.pi
TUBE_P = [5.0, 10.0, 15.0, 0.0, 4 * PI / 3]
CONE_P = [2.0, 6.0, 4.0, 12.0, 20.0, 0.0, 2 * PI]
CONE_SEG_P = [2.0, 6.0, 4.0, 12.0, 20.0, 0.3, 1.9 * PI]
TRD_P = [5.0, 10.0, 7.0, 3.0, 15.0]
PCON_P = W.polycone_params(W.config_seed(3, 0))
PCON_SEG_P = [0.4, 1.2 * PI] + PCON_P[2:]
# polycones with z steps (reading R26): radii jump at z = -4 (outwards, and the bore opens) and at z = 6 (inwards)
PCON_STEP_P = [0.0, 2 * PI, 7, -12.0, 0.0, 6.0, -4.0, 1.0, 8.0, -4.0, 3.0, 12.0, 2.0, 2.0, 10.0, 6.0, 2.0, 11.0, 6.0, 0.0, 5.0,
               14.0, 1.5, 4.0]
PCON_STEP_SEG_P = [-0.7, 1.3 * PI] + PCON_STEP_P[2:]

SHAPES = {
    "box": (O.BOX, [5.0, 5.0, 5.0]),
    "orb": (O.ORB, [20.0]),
    "tube": (O.TUBE, TUBE_P),
    "tube_full_solid": (O.TUBE, [0.0, 8.0, 8.0, 0.0, 2 * PI]),
    "tube_small_wedge": (O.TUBE, [3.0, 9.0, 6.0, -0.5, 0.8]),
    "cone": (O.CONE, CONE_P),
    "cone_seg": (O.CONE, CONE_SEG_P),
    "trd": (O.TRD, TRD_P),
    "polycone": (O.POLYCONE, PCON_P),
    "polycone_seg": (O.POLYCONE, PCON_SEG_P),
    "polycone_step": (O.POLYCONE, PCON_STEP_P),
    "polycone_step_seg": (O.POLYCONE, PCON_STEP_SEG_P),
}


def tracks_for(name, n, seed=11):
    kind, par = SHAPES[name]
    c, h = W.bounding_half(kind, par)
    s = O.Shape(kind, par)
    band = lambda x, y, z: np.abs(s.sdf(x, y, z)) < W.SURFACE_BAND
    return s, W.draw_tracks(seed, n, c, tuple(1.5 * v for v in h), band)


# ------------------------------------------------------------------ worked examples (golden file)

def _parse_golden(name="worked_examples.txt"):
    path = os.path.join(os.path.dirname(__file__), "golden", name)
    names = {"box": O.BOX, "orb": O.ORB, "tube": O.TUBE, "cone": O.CONE, "trd": O.TRD}
    val = lambda t: {"4PI3": 4 * PI / 3, "2PI": 2 * PI, "inf": math.inf}.get(t, None) if t in ("4PI3", "2PI", "inf") else float(t)
    rows = []
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        eid, shape, p, d, res = [f.strip() for f in line.split("|")]
        st = shape.split()
        rows.append((eid, names[st[0]], [val(t) for t in st[1:]], [val(t) for t in p.split()],
                     None if d == "-" else [val(t) for t in d.split()],
                     {k: val(v) for k, v in (kv.split("=") for kv in res.split())}))
    return rows


@pytest.mark.parametrize("row", _parse_golden(), ids=lambda r: r[0])
def test_worked_examples(row):
    eid, kind, par, p, d, res = row
    s = O.Shape(kind, par)
    for q, want in res.items():
        if q == "inside":
            got = float(s.inside(*p)[0])
        elif q.startswith("safety"):
            got = float(getattr(s, q)(*p)[0])
        else:
            got = float(getattr(s, q)(*p, *d, 1e30)[0])
        if math.isinf(want):
            assert got == want, (eid, q, got)
        else:
            assert abs(got - want) <= 1e-12 * max(1.0, abs(want)), (eid, q, got, want)


# ------------------------------------------------------------------ sdf: brute force, sign, eikonal

@pytest.mark.parametrize("name", list(SHAPES))
def test_sdf_sign_is_membership(name):
    kind, par = SHAPES[name]
    s, (x, y, z, *_) = tracks_for(name, 20000)
    sd = s.sdf(x, y, z)
    mem = G.member(kind, par, x, y, z)
    assert np.array_equal(sd < 0, mem)
    cls = s.inside(x, y, z)
    assert np.array_equal(cls == O.INSIDE, mem) and np.array_equal(cls == O.OUTSIDE, ~mem)
    # Inside agrees with the sign of both safeties (BASELINE.json north_star)
    assert np.array_equal(s.safety_to_in(x, y, z), sd) and np.array_equal(s.safety_to_out(x, y, z), -sd)
    frac = mem.mean()
    assert 0.02 < frac < 0.6


@pytest.mark.parametrize("name", list(SHAPES))
def test_sdf_brute_force_surface_sampling(name):
    kind, par = SHAPES[name]
    s, (x, y, z, *_) = tracks_for(name, 24, seed=5)
    sd = s.sdf(x, y, z)
    for i in range(x.size):
        bf = G.brute_distance(kind, par, (x[i], y[i], z[i]))
        assert abs(abs(sd[i]) - bf) < 2e-4 * max(1.0, bf), (name, i, sd[i], bf)


@pytest.mark.parametrize("name", list(SHAPES))
def test_sdf_eikonal(name):
    """|sdf(p) - sdf(q)| <= |p - q| everywhere; |grad sdf| = 1 away from medial sets.  A lower-bound
    'safety' (max of surface distances) fails the gradient part."""
    s, (x, y, z, dx, dy, dz) = tracks_for(name, 20000, seed=3)
    step = 0.37
    a = s.sdf(x, y, z)
    b = s.sdf(x + step * dx, y + step * dy, z + step * dz)
    assert np.all(np.abs(a - b) <= step * (1 + 1e-12) + 1e-12)
    h = 1e-5
    g = [(s.sdf(x + h * (k == 0), y + h * (k == 1), z + h * (k == 2)) -
          s.sdf(x - h * (k == 0), y - h * (k == 1), z - h * (k == 2))) / (2 * h) for k in range(3)]
    gn = np.sqrt(g[0] ** 2 + g[1] ** 2 + g[2] ** 2)
    assert np.all(gn <= 1 + 1e-6)
    assert np.mean(np.abs(gn - 1) < 1e-5) > 0.97     # the rest sit on medial sets within h


def test_box_safety_closed_form():
    s, (x, y, z, *_) = tracks_for("box", 5000)
    q = np.stack([np.abs(x) - 5, np.abs(y) - 5, np.abs(z) - 5])
    want = np.linalg.norm(np.maximum(q, 0), axis=0) + np.minimum(q.max(axis=0), 0)
    assert np.allclose(s.sdf(x, y, z), want, rtol=0, atol=1e-14)


def test_tube_full_solid_safety_is_2d_box_sdf():
    s, (x, y, z, *_) = tracks_for("tube_full_solid", 5000)
    q = np.stack([np.hypot(x, y) - 8.0, np.abs(z) - 8.0])
    want = np.linalg.norm(np.maximum(q, 0), axis=0) + np.minimum(q.max(axis=0), 0)
    assert np.allclose(s.sdf(x, y, z), want, rtol=0, atol=1e-13)


def test_cone_slant_distance_closed_form():
    # near the outer surface mid-height the safety is (rmax(z) - rho) / sqrt(1 + B^2)
    s = O.Shape(O.CONE, CONE_P)
    B = (12.0 - 6.0) / 40.0
    z = np.linspace(-5, 5, 11)
    rho = 9.0 + B * z - 0.5
    got = s.safety_to_out(rho * math.cos(0.7), rho * math.sin(0.7), z)
    assert np.allclose(got, 0.5 / math.sqrt(1 + B * B), rtol=0, atol=1e-13)


# ------------------------------------------------------------------ reductions between solids

def _five(s, t, step_max=1e30):
    x, y, z, dx, dy, dz = t
    return [s.inside(x, y, z).astype(np.float64), s.safety_to_in(x, y, z), s.safety_to_out(x, y, z),
            s.distance_to_in(x, y, z, dx, dy, dz, step_max), s.distance_to_out(x, y, z, dx, dy, dz, step_max)]


def _same(a, b, tol=1e-11):
    for u, v in zip(a, b):
        fin = np.isfinite(u)
        assert np.array_equal(fin, np.isfinite(v))
        assert np.array_equal(u[~fin], v[~fin])
        assert np.all(np.abs(u[fin] - v[fin]) <= tol * np.maximum(1.0, np.abs(v[fin])))


def test_trd_with_equal_ends_is_box():
    box = O.Shape(O.BOX, [5, 7, 9])
    trd = O.Shape(O.TRD, [5, 5, 7, 7, 9])
    t = W.draw_tracks(21, 20000, (0, 0, 0), (9, 12, 15), lambda x, y, z: np.abs(box.sdf(x, y, z)) < 1e-6)
    _same(_five(trd, t), _five(box, t))


def test_cone_with_equal_radii_is_tube():
    tube = O.Shape(O.TUBE, TUBE_P)
    cone = O.Shape(O.CONE, [5, 10, 5, 10, 15, 0, 4 * PI / 3])
    _, t = tracks_for("tube", 20000)
    _same(_five(cone, t), _five(tube, t))


def test_two_plane_polycone_is_cone_and_inserted_plane_changes_nothing():
    _, t = tracks_for("cone_seg", 20000)
    cone = O.Shape(O.CONE, CONE_SEG_P)
    sphi, dphi = CONE_SEG_P[5], CONE_SEG_P[6]
    pc2 = O.Shape(O.POLYCONE, [sphi, dphi, 2, -20, 2, 6, 20, 4, 12])
    # extra plane at z = 4 on the existing generators: rmin = 2 + 2*24/40 = 3.2, rmax = 6 + 6*24/40 = 9.6
    pc3 = O.Shape(O.POLYCONE, [sphi, dphi, 3, -20, 2, 6, 4, 3.2, 9.6, 20, 4, 12])
    ref = _five(cone, t)
    _same(_five(pc2, t), ref)
    _same(_five(pc3, t), ref, tol=1e-9)


def test_three_plane_polycone_with_equal_radii_is_tube():
    tube = O.Shape(O.TUBE, TUBE_P)
    pc = O.Shape(O.POLYCONE, [0, 4 * PI / 3, 3, -15, 5, 10, 2, 5, 10, 15, 5, 10])
    _, t = tracks_for("tube", 20000)
    _same(_five(pc, t), _five(tube, t))


def test_stepped_polycone_of_two_cylinders_is_the_union_of_two_tubes():
    """R26: a polycone whose radii jump at z = 0 is the union of two tubes that share the plane z = 0.  Outside the union
    the distance to it is the smaller of the two tube distances (distance to a union of sets), DistanceToIn the smaller of
    the two DistanceToIn (the first entry into either part), Inside the OR of the memberships."""
    pc = O.Shape(O.POLYCONE, [0, 2 * PI, 4, -10, 2, 5, 0, 2, 5, 0, 3, 9, 6, 3, 9])
    lo = O.Shape(O.TUBE, [2, 5, 5, 0, 2 * PI])   # z in [-10, 0] about z = -5
    hi = O.Shape(O.TUBE, [3, 9, 3, 0, 2 * PI])   # z in [0, 6] about z = 3
    x, y, z, dx, dy, dz = W.draw_tracks(21, 40000, (0, 0, -2), (13.5, 13.5, 12),
                                        lambda x, y, z: np.abs(pc.sdf(x, y, z)) < W.SURFACE_BAND)
    s_lo, s_hi = lo.sdf(x, y, z + 5), hi.sdf(x, y, z - 3)
    out = (s_lo > 0) & (s_hi > 0)
    assert 0.5 < out.mean() < 0.95
    assert np.array_equal(pc.inside(x, y, z) == O.OUTSIDE, out)
    assert np.max(np.abs(pc.sdf(x, y, z)[out] - np.minimum(s_lo, s_hi)[out])) < 1e-12
    want = np.minimum(lo.distance_to_in(x, y, z + 5, dx, dy, dz), hi.distance_to_in(x, y, z - 3, dx, dy, dz))
    got = pc.distance_to_in(x, y, z, dx, dy, dz)
    fin = np.isfinite(want[out])
    assert np.array_equal(np.isfinite(got[out]), fin) and 0.05 < fin.mean() < 0.9
    assert np.max(np.abs(got[out][fin] - want[out][fin])) < 1e-11
    # inside the union the way out passes through both parts: DistanceToOut >= the exit of the part the point is in
    ins = ~out
    t_part = np.where(s_lo < 0, lo.distance_to_out(x, y, z + 5, dx, dy, dz), hi.distance_to_out(x, y, z - 3, dx, dy, dz))
    assert np.all(pc.distance_to_out(x, y, z, dx, dy, dz)[ins] >= t_part[ins] - 1e-11)
    # a hand-worked point: (7, 0, -1) lies 1 below the step annulus 5 <= rho <= 9 at z = 0 and 2 outside the lower tube
    assert abs(pc.sdf(7.0, 0.0, -1.0)[0] - 1.0) < 1e-15
    assert pc.distance_to_in(7.0, 0.0, -1.0, 0.0, 0.0, 1.0)[0] == 1.0
    assert pc.distance_to_in(7.0, 0.0, -1.0, -1.0, 0.0, 0.0)[0] == 2.0
    assert pc.distance_to_out(4.0, 0.0, -1.0, 0.0, 0.0, 1.0)[0] == 7.0   # through the plane z = 0 into the upper part


def test_orb_rotation_invariance():
    s, t = tracks_for("orb", 5000)
    R = G.random_rotation(np.random.default_rng(1))
    P = R @ np.stack(t[:3])
    D = R @ np.stack(t[3:])
    _same(_five(s, (P[0], P[1], P[2], D[0], D[1], D[2])), _five(s, t), tol=1e-10)


def test_revolution_invariance_full_phi():
    for name in ("cone", "polycone", "tube_full_solid"):
        s, t = tracks_for(name, 5000)
        c, sn = math.cos(1.234), math.sin(1.234)
        x, y, z, dx, dy, dz = t
        tr = (c * x - sn * y, sn * x + c * y, z, c * dx - sn * dy, sn * dx + c * dy, dz)
        a, b = _five(s, tr), _five(s, t)
        # Inside may not flip; distances agree to rounding
        _same(a, b, tol=1e-9)


# ------------------------------------------------------------------ first crossing: textbook routines

def test_box_slab_method():
    s, (x, y, z, dx, dy, dz) = tracks_for("box", 20000)
    P, D = np.stack([x, y, z]), np.stack([dx, dy, dz])
    with np.errstate(divide="ignore", invalid="ignore"):
        ta, tb = (-5 - P) / D, (5 - P) / D
    tn, tf = np.minimum(ta, tb).max(axis=0), np.maximum(ta, tb).min(axis=0)
    inside = G.member(O.BOX, [5, 5, 5], x, y, z)
    want_in = np.where(inside, -1.0, np.where((tn < tf) & (tf > 0), tn, np.inf))
    want_out = np.where(inside, tf, -1.0)
    assert np.array_equal(s.distance_to_in(x, y, z, dx, dy, dz), want_in)
    assert np.array_equal(s.distance_to_out(x, y, z, dx, dy, dz), want_out)


def test_box_generic_convex_clip_equals_slabs():
    box = O.Shape(O.BOX, [5, 5, 5])
    trd = O.Shape(O.TRD, [5, 5, 5, 5, 5])
    _, t = tracks_for("box", 20000)
    a, b = box.cross(*t), trd.cross(*t)
    fin = np.isfinite(a)
    assert np.array_equal(fin, np.isfinite(b))
    assert np.all(np.abs(a[fin] - b[fin]) <= 1e-15 * np.abs(a[fin]) + 1e-15)


def test_orb_ray_sphere_quadratic():
    s, (x, y, z, dx, dy, dz) = tracks_for("orb", 20000)
    b = x * dx + y * dy + z * dz
    c = x * x + y * y + z * z - 400.0
    disc = b * b - c
    sq = np.sqrt(np.maximum(disc, 0))
    want_in = np.where(c < 0, -1.0, np.where((disc > 0) & (b < 0), -b - sq, np.inf))
    want_out = np.where(c < 0, -b + sq, -1.0)
    for got, want in ((s.distance_to_in(x, y, z, dx, dy, dz), want_in), (s.distance_to_out(x, y, z, dx, dy, dz), want_out)):
        fin = np.isfinite(want)
        assert np.array_equal(fin, np.isfinite(got))
        assert np.allclose(got[fin], want[fin], rtol=1e-12, atol=1e-12)


def test_long_solid_cylinder_is_ray_cylinder_quadratic():
    # tube rmin=0, full phi, dz so large that the caps never matter: textbook ray-cylinder
    s = O.Shape(O.TUBE, [0, 8, 1e6, 0, 2 * PI])
    rng = np.random.default_rng(2)
    n = 20000
    x, y, z = rng.uniform(-16, 16, n), rng.uniform(-16, 16, n), rng.uniform(-5, 5, n)
    v = rng.normal(size=(3, n))
    v /= np.linalg.norm(v, axis=0)
    dx, dy, dz = v
    a = dx * dx + dy * dy
    b = x * dx + y * dy
    c = x * x + y * y - 64.0
    disc = b * b - a * c
    sq = np.sqrt(np.maximum(disc, 0))
    want_in = np.where(c < 0, -1.0, np.where((disc > 0) & (b < 0), (-b - sq) / a, np.inf))
    want_out = np.where(c < 0, (-b + sq) / a, -1.0)
    for got, want in ((s.distance_to_in(x, y, z, dx, dy, dz), want_in), (s.distance_to_out(x, y, z, dx, dy, dz), want_out)):
        fin = np.isfinite(want)
        assert np.array_equal(fin, np.isfinite(got))
        assert np.allclose(got[fin], want[fin], rtol=1e-11, atol=1e-11)


def test_cone_meridional_rays_reduce_to_2d_lines():
    # radial rays in a meridional plane: the hit on a generator r = A + B z is a 2-D line intersection
    s = O.Shape(O.CONE, CONE_P)
    B, A = 6.0 / 40.0, 9.0
    for z0 in (-10.0, 0.0, 7.0):
        for ang in (0.3, 1.1):
            # from far outside, radially inward and tilted: direction (-cos a, 0, sin a) in the (r, z) plane
            r0 = 40.0
            dr, dzz = -math.cos(ang), math.sin(ang)
            t = (A + B * z0 - r0) / (dr - B * dzz)
            zh = z0 + t * dzz
            got = s.distance_to_in(r0 * math.cos(0.5), r0 * math.sin(0.5), z0, dr * math.cos(0.5), dr * math.sin(0.5), dzz)[0]
            if abs(zh) <= 20.0:
                assert abs(got - t) < 1e-12 * t


# ------------------------------------------------------------------ first crossing: invariants + brute force

@pytest.mark.parametrize("name", list(SHAPES))
def test_distance_lands_on_surface_and_flips_side(name):
    kind, par = SHAPES[name]
    s, (x, y, z, dx, dy, dz) = tracks_for(name, 20000, seed=9)
    cls = s.inside(x, y, z)
    din = s.distance_to_in(x, y, z, dx, dy, dz)
    dout = s.distance_to_out(x, y, z, dx, dy, dz)
    # wrong-side convention (R4) and its equivalence with Inside
    assert np.array_equal(din == -1.0, cls == O.INSIDE)
    assert np.array_equal(dout == -1.0, cls == O.OUTSIDE)
    assert np.all(np.isfinite(dout[cls == O.INSIDE]))          # a bounded solid is always left
    t = np.where(cls == O.INSIDE, dout, din)
    hit = np.isfinite(t)
    assert 0.03 < hit.mean() < 0.9
    tt = t[hit]
    hx, hy, hz = x[hit] + tt * dx[hit], y[hit] + tt * dy[hit], z[hit] + tt * dz[hit]
    # (iv) p + t d lies within kTolerance of the surface
    assert np.max(np.abs(s.sdf(hx, hy, hz))) <= 1e-9
    # (v) safety <= distance for every direction
    assert np.all(np.abs(s.sdf(x, y, z))[hit] <= tt * (1 + 1e-12))
    # (vii) membership differs just before / just after the crossing (skip grazing hits)
    e = 1e-6
    before = G.member(kind, par, hx - e * dx[hit], hy - e * dy[hit], hz - e * dz[hit])
    after = G.member(kind, par, hx + e * dx[hit], hy + e * dy[hit], hz + e * dz[hit])
    assert np.mean(before != after) > 0.999
    assert np.array_equal(before[before != after], (cls[hit] == O.INSIDE)[before != after])


@pytest.mark.parametrize("name", list(SHAPES))
def test_cross_equals_sphere_tracing(name):
    """(vi) no crossing earlier: t <- t + |sdf(p + t d)| converges to Cross, or leaves the bounding sphere
    exactly when Cross is +inf.  Uses only the (separately pinned) sdf."""
    kind, par = SHAPES[name]
    s, (x, y, z, dx, dy, dz) = tracks_for(name, 4000, seed=13)
    want = s.cross(x, y, z, dx, dy, dz)
    c, h = W.bounding_half(kind, par)
    far = 4.0 * math.sqrt(sum((1.5 * v) ** 2 for v in h)) + 10.0
    t = np.zeros_like(x)
    live = np.ones(x.shape, dtype=bool)
    for _ in range(4000):
        idx = np.flatnonzero(live)
        if idx.size == 0:
            break
        d = np.abs(s.sdf(x[idx] + t[idx] * dx[idx], y[idx] + t[idx] * dy[idx], z[idx] + t[idx] * dz[idx]))
        t[idx] += d
        live[idx[(d < 1e-12) | (t[idx] > far)]] = False
    conv = ~live
    escaped = t > far
    # a handful of grazing rays may converge slowly; they must be rare
    assert conv.mean() > 0.995
    assert np.array_equal(np.isinf(want[conv]), escaped[conv])
    ok = conv & ~escaped
    assert np.max(np.abs(t[ok] - want[ok])) < 1e-8


@pytest.mark.parametrize("name", list(SHAPES))
def test_cross_vs_ray_marching_tiny(name):
    """(viii) brute-force marching (step 1e-3 + bisection) on the membership function, tiny input."""
    kind, par = SHAPES[name]
    s, (x, y, z, dx, dy, dz) = tracks_for(name, 60, seed=17)
    want = s.cross(x, y, z, dx, dy, dz)
    c, h = W.bounding_half(kind, par)
    tmax = 4.0 * math.sqrt(sum((1.5 * v) ** 2 for v in h))
    for i in range(x.size):
        tm = G.march_first_flip(kind, par, (x[i], y[i], z[i]), (dx[i], dy[i], dz[i]), tmax)
        if math.isinf(want[i]):
            assert math.isinf(tm), (name, i, tm)
        elif math.isinf(tm) or want[i] < tm - 2e-3:
            # the marcher may step over a clip shorter than its step: the crossing must then be real
            e = 1e-7
            a = G.member(kind, par, *(np.array([x[i], y[i], z[i]]) + (want[i] - e) * np.array([dx[i], dy[i], dz[i]])))
            b = G.member(kind, par, *(np.array([x[i], y[i], z[i]]) + (want[i] + e) * np.array([dx[i], dy[i], dz[i]])))
            assert bool(a) != bool(b), (name, i, want[i], tm)
        else:
            assert abs(want[i] - tm) < 1e-9 * max(1.0, tm) + 1e-10, (name, i, want[i], tm)


@pytest.mark.parametrize("name", ["tube", "cone_seg", "trd", "polycone"])
def test_safety_is_infimum_of_cross_over_directions(name):
    """(iii) inf over many directions of Cross(p, d) decreases to |sdf(p)| and never goes below it."""
    s, (x, y, z, *_) = tracks_for(name, 6, seed=23)
    rng = np.random.default_rng(4)
    v = rng.normal(size=(3, 100000))
    v /= np.linalg.norm(v, axis=0)
    sd = np.abs(s.sdf(x, y, z))
    for i in range(x.size):
        n = v.shape[1]
        t = s.cross(np.full(n, x[i]), np.full(n, y[i]), np.full(n, z[i]), v[0], v[1], v[2])
        assert t.min() >= sd[i] * (1 - 1e-12)
        assert t.min() <= sd[i] * 1.01 + 1e-3


def test_step_max_turns_far_hits_into_misses():
    s, (x, y, z, dx, dy, dz) = tracks_for("tube", 5000)
    full = s.distance_to_in(x, y, z, dx, dy, dz, np.inf)
    cut = s.distance_to_in(x, y, z, dx, dy, dz, 12.0)
    assert np.array_equal(cut, np.where((full > 12.0), np.inf, full))
    assert np.array_equal(s.distance_to_in(x, y, z, dx, dy, dz, 1e30), full)


def test_zero_direction_components_and_tangents():
    box = O.Shape(O.BOX, [5, 5, 5])
    assert box.distance_to_in(10, 6, 0, -1, 0, 0)[0] == np.inf          # parallel, outside the y slab
    assert box.distance_to_in(10, 4, 0, -1, 0, 0)[0] == 5.0
    assert box.distance_to_out(0, 0, 0, 0, 0, -1)[0] == 5.0
    orb = O.Shape(O.ORB, [20])
    assert orb.distance_to_in(30, 20, 0, -1, 0, 0)[0] == np.inf         # tangent: not a crossing (R8)
    tube = O.Shape(O.TUBE, TUBE_P)
    assert tube.distance_to_in(0, 7.5, 30, 0, 0, -1)[0] == 15.0         # along the axis onto the cap
    assert tube.distance_to_in(0, 2.0, 30, 0, 0, -1)[0] == np.inf       # down the bore


def test_invalid_parameters_are_rejected():
    bad = [(O.BOX, [5, 0, 5]), (O.BOX, [5, 5]), (O.ORB, [-1]), (O.TUBE, [10, 5, 15, 0, 1]), (O.TUBE, [5, 10, 15, 0, 0]),
           (O.CONE, [2, 6, 12, 4, 20, 0, 1]), (O.TRD, [5, 10, 7, 3, -1]), (O.POLYCONE, [0, 1, 1, 0, 1, 2]),
           (O.POLYCONE, [0, 1, 2, 0, 1, 2, 0, 1, 2]), (O.BOX, [float("nan"), 1, 1]),
           # z steps (R26): not at an end, not three planes at one z, radial ranges must overlap, z never decreases
           (O.POLYCONE, [0, 7, 3, 0, 1, 2, 0, 1, 3, 5, 1, 3]), (O.POLYCONE, [0, 7, 3, 0, 1, 2, 5, 1, 3, 5, 1, 2]),
           (O.POLYCONE, [0, 7, 5, 0, 1, 2, 3, 1, 2, 3, 1, 3, 3, 1, 4, 6, 1, 4]),
           (O.POLYCONE, [0, 7, 4, 0, 1, 2, 3, 1, 2, 3, 2, 4, 6, 2, 4]), (O.POLYCONE, [0, 7, 3, 0, 1, 2, 3, 1, 2, 2, 1, 2])]
    for kind, par in bad:
        with pytest.raises(ValueError):
            O.Shape(kind, par)


# ------------------------------------------------------------------ the oracle's own rounding

@pytest.mark.parametrize("name", list(SHAPES))
def test_fp64_oracle_agrees_with_80bit_build(name):
    kind, par = SHAPES[name]
    s, t = tracks_for(name, 100000, seed=29)
    sl = O.Shape(kind, par, long_double=True)
    a, b = _five(s, t), _five(sl, t)
    for u, v in zip(a, b):
        fin = np.isfinite(u)
        assert np.array_equal(fin, np.isfinite(v))
        assert np.array_equal(u[~fin], v[~fin])
        assert np.max(np.abs(u[fin] - v[fin])) <= 1e-11
