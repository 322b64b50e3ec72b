"""GPU parity of the boolean solids (include/vg.h vg_boolean_create; readings R27-R29) against the oracle on the same
seeded inputs: classes bit-exact, -1 / +inf sentinels bit-exact, distances and safeties within max(1e-9, 1e-12 |oracle|)."""
import os

import numpy as np
import pytest
import torch

import oracle as O
import workloads as W
from parity import assert_int_equal, assert_real_close

pytestmark = pytest.mark.gpu

CASES = {bc.name: bc for bc in W.boolean_cases()}


@pytest.fixture(scope="module")
def vg():
    import paper_1512_06637_b200 as vg
    return vg


def dev(arrs):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs]


def build(vg, bc):
    co = O.Boolean(bc.op, O.Shape(bc.kind_a, bc.par_a), O.Shape(bc.kind_b, bc.par_b), bc.xform)
    cg = vg.Boolean(bc.op, vg.Shape(bc.kind_a, bc.par_a), vg.Shape(bc.kind_b, bc.par_b), bc.xform)
    return co, cg


def clear_of_both(co, bc):
    """Redraw points within 1e-6 of the surface of C or of either operand (a point ON an operand's surface but deep inside
    the other is a surface-band case of R7 for the state machine, outside the parity contract)."""
    M = np.asarray(bc.xform).reshape(3, 4)

    def band(x, y, z):
        L = M[:, :3] @ np.stack([x, y, z]) + M[:, 3:4]
        return (np.abs(co.a.sdf(x, y, z)) < W.SURFACE_BAND) | (np.abs(co.b.sdf(L[0], L[1], L[2])) < W.SURFACE_BAND)
    return band


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("n", [1, 20001, 200003])
def test_boolean_queries_match_the_oracle(vg, name, n):
    bc = CASES[name]
    co, cg = build(vg, bc)
    t = bc.tracks(n, clear_of_both(co, bc))
    dt = dev(t)
    assert_int_equal(cg.inside(*dt[:3]).cpu().numpy(), co.inside(*t[:3]), "%s inside" % name)
    for q in ("distance_to_in", "distance_to_out"):
        for step_max in (W.STEP_MAX, 6.0):
            assert_real_close(getattr(cg, q)(*dt, step_max).cpu().numpy(), getattr(co, q)(*t, step_max), "%s %s" % (name, q))
    for q in ("safety_to_in", "safety_to_out"):
        assert_real_close(getattr(cg, q)(*dt[:3]).cpu().numpy(), getattr(co, q)(*t[:3]), "%s %s" % (name, q))
    if n > 1000:
        cls = co.inside(*t[:3])
        assert (cls == O.INSIDE).any() and (cls == O.OUTSIDE).any()


def test_boolean_query_all_and_host_entry(vg):
    bc = CASES["box_minus_tube"]
    co, cg = build(vg, bc)
    t = bc.tracks(70001, clear_of_both(co, bc))
    dt = dev(t)
    cls, din, dout, sin, sout = cg.query_all(*dt, W.STEP_MAX)
    assert_int_equal(cls.cpu().numpy(), co.inside(*t[:3]), "fused inside")
    assert_real_close(din.cpu().numpy(), co.distance_to_in(*t, W.STEP_MAX), "fused din")
    assert_real_close(dout.cpu().numpy(), co.distance_to_out(*t, W.STEP_MAX), "fused dout")
    assert_real_close(sin.cpu().numpy(), co.safety_to_in(*t[:3]), "fused sin")
    assert_real_close(sout.cpu().numpy(), co.safety_to_out(*t[:3]), "fused sout")
    ht = [torch.from_numpy(a).pin_memory() for a in t]
    g = cg.query_host("distance_to_out", *ht, step_max=W.STEP_MAX).numpy()
    assert_real_close(g, co.distance_to_out(*t, W.STEP_MAX), "host dout")


def test_axis_aligned_rays_and_degenerate_directions(vg):
    """Zero direction components (R9) through the state machine: box faces, tube caps and axis-parallel rays."""
    for name in ("box_union_orb", "box_minus_tube", "tube_minus_cone"):
        bc = CASES[name]
        co, cg = build(vg, bc)
        x, y, z, dx, dy, dz = bc.tracks(60000, clear_of_both(co, bc))
        rng = np.random.default_rng(3)
        mode = rng.integers(0, 6, x.size)
        sgn = rng.choice([-1.0, 1.0], x.size)
        for m, (a, b, c) in enumerate([(1, 0, 0), (0, 1, 0), (0, 0, 1)]):
            k = mode == m
            dx[k], dy[k], dz[k] = a * sgn[k], b * sgn[k], c * sgn[k]
        t = (x, y, z, dx, dy, dz)
        dt = dev(t)
        for q in ("distance_to_in", "distance_to_out"):
            assert_real_close(getattr(cg, q)(*dt, W.STEP_MAX).cpu().numpy(), getattr(co, q)(*t, W.STEP_MAX), "%s %s axis rays" % (name, q))


def test_boolean_create_rejects_bad_input(vg):
    a = vg.Shape(W.BOX, [1, 1, 1])
    ident = [1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]
    with pytest.raises(vg.VgError):
        vg.Boolean(3, a, a, ident)
    with pytest.raises(vg.VgError):
        vg.Boolean(vg.UNION, a, a, [2, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0])
    pc = vg.Shape(W.POLYCONE, W.polycone_params(1))
    c = vg.Boolean(vg.UNION, a, a, ident)
    bp = vg.Boolean(vg.UNION, a, pc, ident)  # a polycone may be an operand of a boolean of two solids ...
    assert bp.kind == vg.BOOLEAN
    for bad in ((c, pc), (pc, c), (bp, a), (a, bp)):  # ... but not a leaf of a nested tree
        with pytest.raises(vg.VgError):
            vg.Boolean(vg.UNION, bad[0], bad[1], ident)
    vg.Volume(vg.Shape(W.BOX, [100, 100, 100]), [bp], [ident])  # ... but it is a placed solid like any other (R30)
    assert vg.Boolean(vg.UNION, a, c, ident).kind == vg.BOOLEAN  # a boolean operand makes a nested boolean (R31)
    vg.Volume(vg.Shape(W.BOX, [10, 10, 10]), [c], [ident])  # a boolean daughter is served by the world kernels (R30)


@pytest.mark.parametrize("name", ["tube_union_box", "cone_intersection_orb", "box_minus_tube"])
def test_full_size_as_benchmarked_every_track(vg, name):
    """4,194,304 tracks (the size bench.py times); the oracle checks every track."""
    bc = CASES[name]
    co, cg = build(vg, bc)
    t = bc.tracks(4194304, clear_of_both(co, bc))
    dt = dev(t)
    cls = cg.inside(*dt[:3])
    din, dout = cg.distance_to_in(*dt, W.STEP_MAX), cg.distance_to_out(*dt, W.STEP_MAX)
    sin = cg.safety_to_in(*dt[:3])
    sel = np.arange(4194304)
    ts = [np.ascontiguousarray(a[sel]) for a in t]
    assert_int_equal(cls.cpu().numpy()[sel], co.inside(*ts[:3]), name + " full-size inside")
    assert_real_close(din.cpu().numpy()[sel], co.distance_to_in(*ts, W.STEP_MAX), name + " full-size din")
    assert_real_close(dout.cpu().numpy()[sel], co.distance_to_out(*ts, W.STEP_MAX), name + " full-size dout")
    assert_real_close(sin.cpu().numpy()[sel], co.safety_to_in(*ts[:3]), name + " full-size safety")
    # every track: wrong-side sentinels follow the class, and the composed safety never exceeds the distance
    assert bool(((din == -1.0) == (cls == vg.INSIDE)).all()) and bool(((dout == -1.0) == (cls == vg.OUTSIDE)).all())
    outside = cls == vg.OUTSIDE
    assert bool((sin[outside] <= din[outside] * (1 + 1e-12)).all())


def _random_primitive(rng):
    kind = int(rng.integers(0, 5))
    two_pi = 2 * np.pi
    if kind == W.BOX:
        return kind, [float(v) for v in rng.uniform(1.0, 10.0, 3)]
    if kind == W.ORB:
        return kind, [float(rng.uniform(2.0, 10.0))]
    if kind == W.TUBE:
        rmin = float(rng.choice([0.0, rng.uniform(0.5, 4.0)]))
        return kind, [rmin, rmin + float(rng.uniform(1.0, 6.0)), float(rng.uniform(1.0, 10.0)), float(rng.uniform(-3, 3)),
                      float(rng.choice([two_pi, rng.uniform(0.5, 6.0)]))]
    if kind == W.CONE:
        a, b = float(rng.choice([0.0, rng.uniform(0.5, 3.0)])), float(rng.choice([0.0, rng.uniform(0.5, 3.0)]))
        return kind, [a, a + float(rng.uniform(1.0, 6.0)), b, b + float(rng.uniform(1.0, 6.0)), float(rng.uniform(1.0, 10.0)),
                      float(rng.uniform(-3, 3)), float(rng.choice([two_pi, rng.uniform(0.5, 6.0)]))]
    return kind, [float(v) for v in rng.uniform(1.0, 8.0, 5)]


def test_random_booleans(vg):
    """Random operand kinds, parameters, operations and placements (all 25 kind pairs are specialised kernels)."""
    rng = np.random.default_rng(4711)
    pairs = set()
    for rep in range(int(os.environ.get("VG_STRESS_REPS", "60"))):
        ka, pa = _random_primitive(rng)
        kb, pb = _random_primitive(rng)
        op = int(rng.integers(0, 3))
        q = rng.normal(size=4)
        q /= np.linalg.norm(q)
        off = tuple(float(v) for v in rng.uniform(-5, 5, 3))
        bc = W.BooleanCase("random%d" % rep, op, ka, pa, kb, pb, off, tuple(q), 9100 + rep)
        co, cg = build(vg, bc)
        t = bc.tracks(20011, clear_of_both(co, bc))
        dt = dev(t)
        what = "%s %s%r %s%r @%r" % (W.OP_NAME[op], W.KIND_NAME[ka], pa, W.KIND_NAME[kb], pb, off)
        assert_int_equal(cg.inside(*dt[:3]).cpu().numpy(), co.inside(*t[:3]), what)
        assert_real_close(cg.distance_to_in(*dt, W.STEP_MAX).cpu().numpy(), co.distance_to_in(*t, W.STEP_MAX), what + " din")
        assert_real_close(cg.distance_to_out(*dt, W.STEP_MAX).cpu().numpy(), co.distance_to_out(*t, W.STEP_MAX), what + " dout")
        assert_real_close(cg.safety_to_in(*dt[:3]).cpu().numpy(), co.safety_to_in(*t[:3]), what + " safety")
        pairs.add((ka, kb))
    assert len(pairs) >= 20


# ------------------------------------------------------------------ nested booleans (reading R31)

CSG = {c.name: c for c in W.csg_cases()}


def csg_band(co):
    leaves = co.leaves()

    def band(x, y, z):
        bad = np.zeros(np.shape(x), dtype=bool)
        for shape, M in leaves:
            L = M[:, :3] @ np.stack([x, y, z]) + M[:, 3:4]
            bad |= np.abs(shape.sdf(L[0], L[1], L[2])) < W.SURFACE_BAND
        return bad
    return band


@pytest.mark.parametrize("name", list(CSG))
@pytest.mark.parametrize("n", [1, 30011, 300007])
def test_nested_booleans_match_the_oracle(vg, name, n):
    cc = CSG[name]
    co, cg = cc.build(O), cc.build(vg)
    t = cc.tracks(n, csg_band(co))
    dt = dev(t)
    assert_int_equal(cg.inside(*dt[:3]).cpu().numpy(), co.inside(*t[:3]), name + " inside")
    for q in ("distance_to_in", "distance_to_out"):
        for step_max in (W.STEP_MAX, 4.0):
            assert_real_close(getattr(cg, q)(*dt, step_max).cpu().numpy(), getattr(co, q)(*t, step_max), "%s %s" % (name, q))
    for q in ("safety_to_in", "safety_to_out"):
        assert_real_close(getattr(cg, q)(*dt[:3]).cpu().numpy(), getattr(co, q)(*t[:3]), "%s %s" % (name, q))
    if n > 1000:
        cls = co.inside(*t[:3])
        assert (cls == O.INSIDE).mean() > 0.03 and (cls == O.OUTSIDE).mean() > 0.03
    assert cg.kind == vg.BOOLEAN


def test_random_nested_booleans(vg):
    """Random trees of 3 to 8 primitives: random grouping (left-deep, right-deep, balanced), operations and placements."""
    rng = np.random.default_rng(815)

    def tree(nleaf):
        if nleaf == 1:
            k, p = _random_primitive(rng)
            return ("leaf", k, p)
        nl = int(rng.integers(1, nleaf))
        q = rng.normal(size=4)
        q /= np.linalg.norm(q)
        xf = W.placement(W.quaternion_to_matrix(tuple(q)), tuple(float(v) for v in rng.uniform(-4, 4, 3)))
        return ("op", int(rng.integers(0, 3)), tree(nl), tree(nleaf - nl), xf)
    done = 0
    for rep in range(int(os.environ.get("VG_STRESS_REPS", "40"))):
        cc = W.CsgCase("random%d" % rep, tree(int(rng.integers(3, 9))), (0, 0, 0), (14, 14, 14), 9300 + rep)
        co, cg = cc.build(O), cc.build(vg)
        t = cc.tracks(12007, csg_band(co))
        cls = co.inside(*t[:3])
        dt = dev(t)
        what = repr(cc.tree)[:200]
        assert_int_equal(cg.inside(*dt[:3]).cpu().numpy(), cls, what)
        assert_real_close(cg.distance_to_in(*dt, W.STEP_MAX).cpu().numpy(), co.distance_to_in(*t, W.STEP_MAX), what + " din")
        assert_real_close(cg.distance_to_out(*dt, W.STEP_MAX).cpu().numpy(), co.distance_to_out(*t, W.STEP_MAX), what + " dout")
        assert_real_close(cg.safety_to_in(*dt[:3]).cpu().numpy(), co.safety_to_in(*t[:3]), what + " safety")
        done += int((cls == O.INSIDE).any())
    assert done >= 15  # most random trees are not empty


def test_nested_boolean_limits(vg):
    a = vg.Shape(W.BOX, [1, 1, 1])
    ident = [1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]
    c = a
    for _ in range(7):
        c = vg.Boolean(vg.UNION, c, a, ident)  # 8 primitives: the limit
    with pytest.raises(vg.VgError):
        vg.Boolean(vg.UNION, c, a, ident)


def test_nested_boolean_as_a_world_node_and_a_daughter(vg):
    """A tree placed in a box: node of a world (R30 + R31) and daughter of a volume, against the oracle's world."""
    cc = CSG["twice_drilled_block_in_a_sphere"]
    q = np.array([0.3, -0.4, 0.5, 0.7])
    xf = [W.placement(np.eye(3), (0, 0, 0)), W.placement(W.quaternion_to_matrix(tuple(q / np.linalg.norm(q))), (3.0, -2.0, 4.0))]
    wo = O.World([O.Shape(W.BOX, [30, 30, 30]), cc.build(O)], [-1, 0], xf)
    wg = vg.World([vg.Shape(W.BOX, [30, 30, 30]), cc.build(vg)], [-1, 0], xf)
    leaves = wo.shapes[1].leaves()
    M1 = np.asarray(xf[1]).reshape(3, 4)

    def band(x, y, z):
        L1 = M1[:, :3] @ np.stack([x, y, z]) + M1[:, 3:4]
        bad = np.abs(wo.shapes[0].sdf(x, y, z)) < W.SURFACE_BAND
        for shape, M in leaves:
            L = M[:, :3] @ L1 + M[:, 3:4]
            bad |= np.abs(shape.sdf(L[0], L[1], L[2])) < W.SURFACE_BAND
        return bad
    t = W.draw_tracks(61, 200003, (3, -2, 4), (16, 16, 16), band)
    dt = dev(t)
    node_o, node_g = wo.locate(*t[:3]), wg.locate(*dt[:3])
    assert_int_equal(node_g.cpu().numpy(), node_o, "tree node locate")
    assert (node_o == 1).mean() > 0.05
    so, no = wo.step(node_o, *t, W.STEP_MAX)
    sg, ng = wg.step(node_g, *dt, W.STEP_MAX)
    assert_int_equal(ng.cpu().numpy(), no, "tree node next")
    assert_real_close(sg.cpu().numpy(), so, "tree node step")
    assert_real_close(wg.safety(node_g, *dt[:3]).cpu().numpy(), wo.safety(node_o, *t[:3]), "tree node safety")
    vol = vg.Volume(vg.Shape(W.BOX, [30, 30, 30]), [cc.build(vg)], [xf[1]])
    root = node_o == 0
    tr = [np.ascontiguousarray(a[root]) for a in t]
    sv, hv = vol.compute_step(*dev(tr), W.STEP_MAX)
    assert_real_close(sv.cpu().numpy(), so[root], "tree daughter step")
    assert_int_equal(hv.cpu().numpy(), np.where(no[root] < 0, -1, no[root] - 1), "tree daughter hit")


# ---------------------------------------------------------------------------------- polycone operands (vg_boolx.cu)

def _pcon_cases():
    two_pi = 2 * np.pi
    pc10 = W.polycone_params(W.config_seed(3, 0))                       # the configs[3] polycone, rmax 10..30, z in +-50
    pcw = [0.4, 4.0] + pc10[2:]                                        # the same with a phi cut
    small = [0.0, two_pi, 4.0, -8.0, 1.0, 4.0, -2.0, 2.0, 7.0, 3.0, 0.5, 5.0, 9.0, 0.0, 3.0]
    q = np.array([0.18, -0.31, 0.22, 0.9])
    Q = W.quaternion_to_matrix(tuple(q / np.linalg.norm(q)))
    return [
        ("pcon_minus_box", W.SUBTRACTION, (W.POLYCONE, pc10), (W.BOX, [12.0, 40.0, 30.0]), W.placement(Q, (8.0, 3.0, -5.0)), 60.0),
        ("box_intersection_pcon", W.INTERSECTION, (W.BOX, [25.0, 18.0, 45.0]), (W.POLYCONE, pc10), W.placement(Q, (4.0, -3.0, 6.0)), 60.0),
        ("pcon_union_pcon", W.UNION, (W.POLYCONE, small), (W.POLYCONE, small), W.placement(Q, (3.0, 2.0, 4.0)), 16.0),
        ("tube_minus_pcon_wedge", W.SUBTRACTION, (W.TUBE, [0.0, 28.0, 45.0, 0.0, two_pi]), (W.POLYCONE, pcw), W.placement(np.eye(3), (0.0, 0.0, 0.0)), 60.0),
        ("pcon_step_union_orb", W.UNION, (W.POLYCONE, W.STEPPED_POLYCONE), (W.ORB, [7.0]), W.placement(Q, (6.0, 0.0, 9.0)), 22.0),
    ]


@pytest.mark.parametrize("case", _pcon_cases(), ids=lambda c: c[0])
def test_boolean_with_polycone_operands_matches_the_oracle(vg, case):
    """boolean operations over the elementary bodies -- the polycone included.  All five queries, a finite
    physics step, the fused call and tracks that start ON the boolean's surface (R32), against the oracle."""
    name, op, (ka, pa), (kb, pb), xf, half = case
    co = O.Boolean(op, O.Shape(ka, pa), O.Shape(kb, pb), xf)
    cg = vg.Boolean(op, vg.Shape(ka, pa), vg.Shape(kb, pb), xf)
    assert cg.kind == vg.BOOLEAN
    M = np.asarray(xf).reshape(3, 4)

    def band(x, y, z):
        L = M[:, :3] @ np.stack([x, y, z]) + M[:, 3:4]
        return (np.abs(co.a.sdf(x, y, z)) < W.SURFACE_BAND) | (np.abs(co.b.sdf(L[0], L[1], L[2])) < W.SURFACE_BAND)

    t = W.draw_tracks(900 + len(name), 100003, (0.0, 0.0, 0.0), (half, half, half), band)
    dt = dev(t)
    cls = co.inside(*t[:3])
    assert (cls == O.INSIDE).any() and (cls == O.OUTSIDE).any()
    assert_int_equal(cg.inside(*dt[:3]).cpu().numpy(), cls, name + " inside")
    for q in ("distance_to_in", "distance_to_out"):
        for step_max in (W.STEP_MAX, 9.0):
            assert_real_close(getattr(cg, q)(*dt, step_max).cpu().numpy(), getattr(co, q)(*t, step_max), "%s %s" % (name, q))
    for q in ("safety_to_in", "safety_to_out"):
        assert_real_close(getattr(cg, q)(*dt[:3]).cpu().numpy(), getattr(co, q)(*t[:3]), "%s %s" % (name, q))
    fused = cg.query_all(*dt, W.STEP_MAX)
    assert_int_equal(fused[0].cpu().numpy(), cls, name + " fused inside")
    assert_real_close(fused[1].cpu().numpy(), co.distance_to_in(*t, W.STEP_MAX), name + " fused din")
    # border starts: move the outside tracks that hit onto their crossing and ask again (no nudge)
    x, y, z, dx, dy, dz = t
    din = co.distance_to_in(x, y, z, dx, dy, dz)
    hit = np.isfinite(din) & (din > 0)
    ts = tuple(np.ascontiguousarray(a) for a in (x[hit] + din[hit] * dx[hit], y[hit] + din[hit] * dy[hit], z[hit] + din[hit] * dz[hit],
                                                 dx[hit], dy[hit], dz[hit]))
    ds = dev(ts)
    assert_int_equal(cg.inside(*ds[:3]).cpu().numpy(), co.inside(*ts[:3]), name + " border inside")
    for q in ("distance_to_in", "distance_to_out"):
        assert_real_close(getattr(cg, q)(*ds, W.STEP_MAX).cpu().numpy(), getattr(co, q)(*ts, W.STEP_MAX), "%s border %s" % (name, q))


@pytest.mark.parametrize("eps", [2e-8, 7e-8, 2e-7, 3e-7, 1e-6, 1e-3])
def test_a_chord_shorter_than_the_ray_tolerance_does_not_stall_the_state_machine(vg, eps):
    """A ray that clips an edge of an operand through a chord of ~1e-7 (shorter than VG_KRAYTOL) leaves that operand with
    its entering crossing still 'at the start' (R32): asked for its next entering crossing it answered 0, and the state
    machines of the booleans entered and left it on the spot until their event limit and returned +inf (found by the
    8000-tree soak: one track in 10^8).  B = the unit cube, clipped at its edge x = y = 1 along d = (1, -1, 0) / sqrt 2;
    A = a box 8 further along the ray; E = a large box around everything; D = an orb far away.  The clip must not decide
    anything: DistanceToIn of A - B, (A - B) u D and (B n D) u A is A's entry; DistanceToOut of E u B and (E u B) u D from
    a start inside E is E's exit."""
    s0 = 5.0
    d = np.array([1.0, -1.0, 0.0]) / np.sqrt(2.0)
    mid = np.array([1.0 - eps / 2, 1.0 - eps / 2, 0.0])   # middle of the chord: the line x + y = 2 - eps cuts the corner
    n = 64
    z0 = np.random.default_rng(3).uniform(-0.5, 0.5, n)    # the same clip at 64 heights
    P = mid[None, :] - s0 * d[None, :] + np.stack([0 * z0, 0 * z0, z0], axis=1)
    ca = mid + 8.0 * d                                     # centre of A

    def tracks(origin):  # the rays in the frame whose origin sits at `origin` (no rotation)
        Q = P - np.asarray(origin)[None, :]
        return tuple(np.ascontiguousarray(a) for a in (Q[:, 0], Q[:, 1], Q[:, 2], np.full(n, d[0]), np.full(n, d[1]), np.full(n, d[2])))
    to_b_from_a = W.placement(np.eye(3), tuple(-ca))       # B as seen from the frame of A: centred at -ca (B sits at the world's origin)
    far = W.placement(np.eye(3), (0.0, 0.0, -40.0))
    ident = W.placement(np.eye(3), (0.0, 0.0, 0.0))

    def build(mod):
        A, B, D, E = (lambda: mod.Shape(W.BOX, [1.0, 1.0, 2.0])), (lambda: mod.Shape(W.BOX, [1.0, 1.0, 1.0])), \
                     (lambda: mod.Shape(W.ORB, [1.0])), (lambda: mod.Shape(W.BOX, [30.0, 30.0, 30.0]))
        a_minus_b = lambda: mod.Boolean(W.SUBTRACTION, A(), B(), to_b_from_a)
        return {  # name: (solid, origin of its frame, query)
            "A - B": (a_minus_b(), ca, "distance_to_in"),
            "(A - B) u D": (mod.Boolean(W.UNION, a_minus_b(), D(), far), ca, "distance_to_in"),
            "(B n D) u A": (mod.Boolean(W.UNION, mod.Boolean(W.INTERSECTION, B(), D(), far), A(), W.placement(np.eye(3), tuple(ca))), (0, 0, 0), "distance_to_in"),
            "E u B": (mod.Boolean(W.UNION, E(), B(), ident), (0, 0, 0), "distance_to_out"),
            "(E u B) u D": (mod.Boolean(W.UNION, mod.Boolean(W.UNION, E(), B(), ident), D(), far), (0, 0, 0), "distance_to_out"),
        }
    so, sg = build(O), build(vg)
    for name, (co, origin, q) in so.items():
        t = tracks(origin)
        want = getattr(co, q)(*t, W.STEP_MAX)
        assert np.isfinite(want).all() and (want > s0 + 1.0).all(), name  # the answer lies beyond the clip
        got = getattr(sg[name][0], q)(*dev(t), W.STEP_MAX).cpu().numpy()
        assert_real_close(got, want, "%s %s, chord %g" % (name, q, eps * np.sqrt(2.0)))
