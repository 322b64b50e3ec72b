"""Pins of reading R32 (oracle/vg_oracle.c: distances from start points in the kTolerance surface band; "the
particle is transported to the border" -- the next step starts ON a surface).  Expectations come from hand-worked points
(tests/golden/surface_examples.txt), from the whole-line crossing list of a start point well away from every surface
(whose alternation is checked against the set definitions of tests/geomdefs.py), from marching the set-definition
membership, and from walking tracks through the trees of volumes border to border with no nudge."""
import math

import numpy as np
import pytest

import geomdefs as G
import oracle as O
import workloads as W
from test_oracle_pins import _parse_golden

PI = math.pi
SHAPES = {
    "box": (O.BOX, [5.0, 5.0, 5.0]),
    "orb": (O.ORB, [20.0]),
    "tube": (O.TUBE, [5.0, 10.0, 15.0, 0.0, 4 * PI / 3]),
    "cone": (O.CONE, [2.0, 6.0, 4.0, 12.0, 20.0, 0.0, 2 * PI]),
    "cone_seg": (O.CONE, [2.0, 6.0, 4.0, 12.0, 20.0, 0.3, 5.9]),
    "trd": (O.TRD, [5.0, 10.0, 7.0, 3.0, 15.0]),
    "polycone": (O.POLYCONE, W.polycone_params(W.config_seed(3, 0))),
    "polycone_step": (O.POLYCONE, list(W.STEPPED_POLYCONE)),
}


@pytest.mark.parametrize("row", _parse_golden("surface_examples.txt"), ids=lambda r: r[0])
def test_surface_examples(row):
    """Hand-worked start points on faces, edges, a corner and the phi planes; and the same results (to the shift along
    the ray) with the point moved 1e-10 to either side of the surface along the direction of motion."""
    eid, kind, par, p, d, res = row
    s = O.Shape(kind, par)
    for shift in (0.0, 1e-10, -1e-10):
        q = [p[i] + shift * d[i] for i in range(3)]
        for name, want in res.items():
            got = float(s.inside(*q)[0]) if name == "inside" else float(getattr(s, name)(*q, *d, 1e30)[0])
            if math.isinf(want):
                assert got == want, (eid, name, shift, got)
            elif name == "inside":
                assert got == want, (eid, name, shift, got)
            else:
                # moving the start by `shift` along the ray moves every crossing by -shift; a result of 0 stays clamped
                lo, hi = (want - abs(shift), want + abs(shift))
                assert lo - 1e-12 * max(1.0, want) <= got <= hi + 1e-12 * max(1.0, want), (eid, name, shift, got, want)


def surface_starts(name, n, seed=77):
    """Tracks transported to a border: seeded tracks of the standard generator (>= 1e-6 from every surface), moved to the
    k-th crossing of their own line.  Kept: crossings that are clear of every other crossing by 1e-3 and are not grazing
    (|d sdf / dt| >= 0.05 across the crossing).  Returns the solid, the start track, its line-crossing list, k."""
    kind, par = SHAPES[name]
    s = O.Shape(kind, par)
    c, h = W.bounding_half(kind, par)
    x, y, z, dx, dy, dz = W.draw_tracks(seed, n, c, tuple(1.5 * v for v in h), lambda x, y, z: np.abs(s.sdf(x, y, z)) < 1e-6)
    rng = np.random.default_rng(seed)
    out = []
    for i in range(n):
        p, d = np.array([x[i], y[i], z[i]]), np.array([dx[i], dy[i], dz[i]])
        t = s.line_crossings(p, d)
        if t.size == 0:
            continue
        k = int(rng.integers(t.size))
        gaps = np.abs(np.delete(t, k) - t[k])
        if gaps.size and gaps.min() < 1e-3:
            continue
        a, b = p + (t[k] - 1e-5) * d, p + (t[k] + 1e-5) * d
        rate = (s.sdf(*b)[0] - s.sdf(*a)[0]) / 2e-5
        if abs(rate) < 0.05:
            continue
        out.append((p, d, t, k))
    assert len(out) > n // 4, (name, len(out))
    return kind, par, s, out


@pytest.mark.parametrize("name", list(SHAPES))
def test_line_crossings_alternate_membership(name):
    """The crossings of the WHOLE line (t of either sign) alternate the set-definition membership, starting outside far
    behind the start point: even-numbered crossings enter, odd-numbered leave (what R32 reads the sense from)."""
    kind, par, s, starts = surface_starts(name, 1500, seed=5)
    for p, d, t, _ in starts:
        assert t.size % 2 == 0
        assert np.all(np.diff(t) >= 0)
        if np.min(np.diff(t)) < 1e-6:
            continue
        mids = np.concatenate([[t[0] - 1.0], 0.5 * (t[:-1] + t[1:]), [t[-1] + 1.0]])
        mem = G.member(kind, par, *(p[:, None] + mids[None, :] * d[:, None]))
        assert np.array_equal(mem, (np.arange(mids.size) % 2) == 1), (p, d, t)
        # and the crossings ahead are the list the first-crossing pins already cover
        ahead = s.all_crossings(p, d)
        assert np.array_equal(ahead, t[t > 0])


@pytest.mark.parametrize("name", list(SHAPES))
def test_surface_start_equals_the_crossing_list_of_the_far_start(name):
    """R32 from a point moved onto its k-th crossing == what the crossing list of the far start point says: 0 for the
    query whose sense the crossing has, the gap to the next crossing for the other one (+inf after the last)."""
    kind, par, s, starts = surface_starts(name, 1500)
    for p, d, t, k in starts:
        h = p + t[k] * d
        assert s.inside(*h)[0] == O.SURFACE
        nxt = (t[k + 1] - t[k]) if k + 1 < t.size else math.inf
        entering = (k % 2 == 0)
        want_in, want_out = (0.0, nxt) if entering else (nxt, 0.0)
        got_in = s.distance_to_in(*h, *d, 1e30)[0]
        got_out = s.distance_to_out(*h, *d, 1e30)[0]
        tol = 1e-9 + 1e-12 * abs(t[k])
        for got, want in ((got_in, want_in), (got_out, want_out)):
            assert (got == want) if math.isinf(want) else abs(got - want) <= tol + 1e-12 * want, (name, p, d, k, got, want)
        # the reversed ray: senses swap, the previous crossing is the next one
        prv = (t[k] - t[k - 1]) if k > 0 else math.inf
        want_in, want_out = (prv, 0.0) if entering else (0.0, prv)
        got_in = s.distance_to_in(*h, *(-d), 1e30)[0]
        got_out = s.distance_to_out(*h, *(-d), 1e30)[0]
        for got, want in ((got_in, want_in), (got_out, want_out)):
            assert (got == want) if math.isinf(want) else abs(got - want) <= tol + 1e-12 * want, (name, p, d, k, "rev", got, want)


@pytest.mark.parametrize("name", list(SHAPES))
def test_surface_start_against_marching_the_set_definition(name):
    """Brute force: from the surface point, march the membership of the closed set (tests/geomdefs.py) in steps of 2e-3 and
    bisect the first flip after the first 1e-4: that flip is DistanceToOut when the ray goes in, DistanceToIn when it goes
    out; the other distance is 0."""
    kind, par, s, starts = surface_starts(name, 400, seed=123)
    c, hh = W.bounding_half(kind, par)
    reach = 4.0 * float(np.linalg.norm(hh)) + float(np.linalg.norm(c))
    for p, d, t, k in starts[:120]:
        h = p + t[k] * d
        ts = np.arange(1e-4, reach, 2e-3)
        mem = G.member(kind, par, *(h[:, None] + ts[None, :] * d[:, None]))
        goes_in = bool(mem[0])
        flips = np.flatnonzero(mem != mem[0])
        got_in, got_out = s.distance_to_in(*h, *d, 1e30)[0], s.distance_to_out(*h, *d, 1e30)[0]
        assert (got_in if goes_in else got_out) <= 1e-9
        other = got_out if goes_in else got_in
        if flips.size == 0:
            assert math.isinf(other), (name, h, d, other)
            continue
        lo, hi = ts[flips[0] - 1], ts[flips[0]]
        for _ in range(50):
            mid = 0.5 * (lo + hi)
            if bool(G.member(kind, par, *(h + mid * d))) == goes_in:
                lo = mid
            else:
                hi = mid
        assert abs(other - 0.5 * (lo + hi)) < 1e-8, (name, h, d, other, lo, hi)


@pytest.mark.parametrize("name", list(SHAPES))
def test_surface_results_do_not_depend_on_the_side_of_the_band(name):
    """Moving the start point +-3e-10 along the surface normal (inside the 1e-9 band on both sides) changes neither the
    zero nor the other distance, beyond what a shift of 3e-10 can do to a crossing that is not grazing."""
    kind, par, s, starts = surface_starts(name, 400, seed=9)
    for p, d, t, k in starts[:150]:
        h = p + t[k] * d
        e = 1e-6
        g = np.array([(s.sdf(*(h + e * u))[0] - s.sdf(*(h - e * u))[0]) / (2 * e) for u in np.eye(3)])
        g /= np.linalg.norm(g)
        base_in, base_out = s.distance_to_in(*h, *d, 1e30)[0], s.distance_to_out(*h, *d, 1e30)[0]
        slack = 1e-7
        for sh in (3e-10, -3e-10):
            q = h + sh * g
            assert s.inside(*q)[0] == O.SURFACE
            gi, go = s.distance_to_in(*q, *d, 1e30)[0], s.distance_to_out(*q, *d, 1e30)[0]
            for got, base in ((gi, base_in), (go, base_out)):
                assert (got == base) if math.isinf(base) else abs(got - base) <= slack, (name, h, d, sh, got, base)


# ------------------------------------------------------------------------------------------------ booleans

IDENT = [1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]


def test_boolean_surface_examples():
    """Hand-worked: A = box(5,5,5), B = orb(3) centred at (4, 0, 0) (B spans x in [1, 7] on the x axis)."""
    a, b = O.Shape(O.BOX, [5.0, 5.0, 5.0]), O.Shape(O.ORB, [3.0])
    xf = [1, 0, 0, -4.0, 0, 1, 0, 0, 0, 0, 1, 0]
    inf = math.inf
    rows = [  # op, p, d, class, DistanceToIn, DistanceToOut
        # on the face of A but deep inside B: inside the union, the face is no border of it
        (O.UNION, (5, 0, 0), (-1, 0, 0), O.INSIDE, -1.0, 10.0),
        (O.UNION, (5, 0, 0), (1, 0, 0), O.INSIDE, -1.0, 2.0),
        # on the surface of B inside A: a border of A - B
        (O.SUBTRACTION, (1, 0, 0), (-1, 0, 0), O.SURFACE, 0.0, 6.0),
        (O.SUBTRACTION, (1, 0, 0), (1, 0, 0), O.SURFACE, inf, 0.0),
        # on the face of A inside B: a border of the intersection (x in [1, 5] on the axis)
        (O.INTERSECTION, (5, 0, 0), (-1, 0, 0), O.SURFACE, 0.0, 4.0),
        (O.INTERSECTION, (5, 0, 0), (1, 0, 0), O.SURFACE, inf, 0.0),
        # on the surface of B outside A (x = 7): a border of the union, not of the intersection
        (O.UNION, (7, 0, 0), (-1, 0, 0), O.SURFACE, 0.0, 12.0),
        (O.UNION, (7, 0, 0), (1, 0, 0), O.SURFACE, inf, 0.0),
        (O.INTERSECTION, (7, 0, 0), (-1, 0, 0), O.OUTSIDE, 2.0, -1.0),
    ]
    for op, p, d, cls, din, dout in rows:
        c = O.Boolean(op, a, b, xf)
        for shift in (0.0, 2e-10, -2e-10):
            q = [p[i] + shift * d[i] for i in range(3)]
            assert c.inside(*q)[0] == cls, (op, p, d, shift)
            for got, want in ((c.distance_to_in(*q, *d, 1e30)[0], din), (c.distance_to_out(*q, *d, 1e30)[0], dout)):
                assert (got == want) if (math.isinf(want) or want == -1.0) else abs(got - want) <= 2e-10 + 1e-12, (op, p, d, shift, got, want)


@pytest.mark.parametrize("bc", W.boolean_cases(), ids=lambda b: b.name)
def test_boolean_events_alternate_the_set_expression(bc):
    """R28 on the whole line: the flips of C alternate the membership of the set expression composed in numpy over
    tests/geomdefs.py, starting outside far behind the start point; the first flip ahead is the distance the query for
    the point's own side returns."""
    from test_oracle_boolean import build, member, tracks
    c = build(bc)
    x, y, z, dx, dy, dz = tracks(bc, c, 600)
    din, dout = c.distance_to_in(x, y, z, dx, dy, dz), c.distance_to_out(x, y, z, dx, dy, dz)
    for i in range(x.size):
        p, d = np.array([x[i], y[i], z[i]]), np.array([dx[i], dy[i], dz[i]])
        t = c.events(p, d)
        assert t.size % 2 == 0
        ahead = t[t > 0]
        first = ahead[0] if ahead.size else math.inf
        assert first == (dout[i] if din[i] == -1.0 else din[i])
        if t.size == 0 or np.min(np.diff(t)) < 1e-6:
            continue
        mids = np.concatenate([[t[0] - 1.0], 0.5 * (t[:-1] + t[1:]), [t[-1] + 1.0]])
        mem = member(bc, *(p[:, None] + mids[None, :] * d[:, None]))
        assert np.array_equal(mem, (np.arange(mids.size) % 2) == 1), (bc.name, p, d, t)


@pytest.mark.parametrize("bc", W.boolean_cases(), ids=lambda b: b.name)
def test_boolean_surface_start_equals_the_event_list_of_the_far_start(bc):
    """A track moved onto the k-th crossing of EITHER operand (whether or not that crossing is a border of C): the class
    and both distances are what the far start point's event list of C says."""
    from test_oracle_boolean import build, tracks, to_b
    c = build(bc)
    x, y, z, dx, dy, dz = tracks(bc, c, 500)
    rng = np.random.default_rng(3)
    M = np.asarray(bc.xform, dtype=np.float64).reshape(3, 4)
    checked = 0
    for i in range(x.size):
        p, d = np.array([x[i], y[i], z[i]]), np.array([dx[i], dy[i], dz[i]])
        ta = c.a.line_crossings(p, d)
        tb = c.b.line_crossings(M[:, :3] @ p + M[:, 3], M[:, :3] @ d)
        tc = c.events(p, d)
        allt = np.concatenate([ta, tb])
        if allt.size == 0:
            continue
        ts = float(allt[rng.integers(allt.size)])
        if np.sort(np.abs(allt - ts))[1:2].min(initial=1.0) < 1e-3:
            continue
        h = p + ts * d
        sa = c.a.sdf(*h)[0]
        sb = c.b.sdf(*to_b(bc.xform, *[np.array([v]) for v in h]))[0]
        on_a = abs(sa) < abs(sb)
        lo, hi = h - 1e-5 * d, h + 1e-5 * d
        f = (lambda q: c.a.sdf(*q)[0]) if on_a else (lambda q: c.b.sdf(*to_b(bc.xform, *[np.array([v]) for v in q]))[0])
        if abs(f(hi) - f(lo)) / 2e-5 < 0.05:
            continue
        k = np.flatnonzero(np.abs(tc - ts) < 1e-9)
        got_in, got_out = c.distance_to_in(*h, *d, 1e30)[0], c.distance_to_out(*h, *d, 1e30)[0]
        tol = 1e-9 + 1e-12 * abs(ts)
        if k.size:  # a border of C
            k = int(k[0])
            assert c.inside(*h)[0] == O.SURFACE
            nxt = (tc[k + 1] - ts) if k + 1 < tc.size else math.inf
            want_in, want_out = (0.0, nxt) if k % 2 == 0 else (nxt, 0.0)
        else:  # an operand's surface hidden in, or outside of, the other: the class of C is strict there
            after = tc[tc > ts]
            nxt = (after[0] - ts) if after.size else math.inf
            inside_c = (np.searchsorted(tc, ts) % 2) == 1
            assert c.inside(*h)[0] == (O.INSIDE if inside_c else O.OUTSIDE)
            want_in, want_out = (-1.0, nxt) if inside_c else (nxt, -1.0)
        for got, want in ((got_in, want_in), (got_out, want_out)):
            assert (got == want) if (math.isinf(want) or want == -1.0) else abs(got - want) <= tol + 1e-12 * want, (bc.name, h, d, got, want)
        checked += 1
    assert checked > 100


# ------------------------------------------------------------------------------- border-to-border transport

def walk(world, node, p, d, max_steps=400):
    """Step, move exactly onto the border (no nudge), take the node Step returned; until the root is left."""
    n = p.shape[1]
    path = np.zeros(n)
    alive = node >= 0
    steps = np.zeros(n, dtype=np.int64)
    trace = []
    for _ in range(max_steps):
        if not alive.any():
            break
        idx = np.flatnonzero(alive)
        st, nx = world.step(node[idx], *p[:, idx], *d[:, idx], 1e30)
        assert np.all(np.isfinite(st)) and np.all(st >= 0), (st[~np.isfinite(st) | (st < 0)][:5])
        trace.append((idx, node[idx].copy(), p[:, idx].copy(), st.copy()))
        p[:, idx] += st * d[:, idx]
        path[idx] += st
        steps[idx] += 1
        node[idx] = nx
        alive[idx] = nx >= 0
    assert not alive.any(), "tracks still inside after %d steps" % max_steps
    return path, steps, trace


@pytest.mark.parametrize("which", ["world", "mixed"])
def test_transport_through_the_tree_border_to_border(which):
    """Tracks walk through the tree of volumes from border to border with NO nudge (every step starts exactly where the
    last one ended, in the node Step returned): the walk ends, no step repeats a border (no zero-length ping-pong: at
    most one zero step in a row), the steps add up to the straight path out of the root box, and half-way along every
    step Locate finds the node the step was taken in."""
    from test_oracle_world import build_mixed
    if which == "world":
        wc = W.world_case()
        shapes = [O.Shape(k, q) for k, q in zip(wc.kinds, wc.params)]
        wo = O.World(shapes, wc.parents, wc.xforms)
    else:
        wc = W.mixed_world_case()
        shapes, wo = build_mixed(wc)

    def band(x, y, z):
        nd = wo.locate(x, y, z)
        return (nd < 0) | (wo.safety(np.maximum(nd, 0), x, y, z) < W.SURFACE_BAND)

    n = 3000
    t = wc.tracks(n, band)
    p, d = np.array(t[:3]), np.array(t[3:])
    node = wo.locate(*p)
    root = shapes[0]
    R = np.asarray(wc.xforms, dtype=np.float64).reshape(-1, 12)[0].reshape(3, 4)
    pl, dl = R[:, :3] @ p + R[:, 3:4], R[:, :3] @ d
    straight = root.distance_to_out(*pl, *dl, 1e30)
    path, steps, trace = walk(wo, node.copy(), p.copy(), d)
    assert np.allclose(path, straight, rtol=0, atol=1e-8), np.abs(path - straight).max()
    assert steps.max() < 60
    for idx, nd, ps, st in trace:
        big = st > 1e-6
        mid = ps[:, big] + 0.5 * st[big] * d[:, idx[big]]
        assert np.array_equal(wo.locate(*mid), nd[big])
    # no two zero-length steps in a row for any track
    last_zero = np.zeros(n, dtype=bool)
    for idx, nd, ps, st in trace:
        z = st <= 1e-9
        assert not np.any(z & last_zero[idx])
        last_zero[idx] = z
