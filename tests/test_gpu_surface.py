"""GPU parity for start points ON surfaces (reading R32; "the particle is transported to
the border": the next step starts on a surface) against the oracle, through the C ABI: Inside == SURFACE, both distances,
both safeties; the hand-worked points of tests/golden/surface_examples.txt; tracks moved onto crossings of primitives,
booleans and CSG trees (both directions, and +-3e-10 / +-1e-16 off the surface); border-to-border walks through the trees
of volumes with no nudge.  Grazing starts (|d sdf / dt| < 0.05) and starts within 1e-3 of another crossing are not
generated (R32: the kernels' ray-parameter tolerance equals the oracle's definition away from those)."""
import math

import numpy as np
import pytest
import torch

import oracle as O
import workloads as W
from parity import assert_int_equal, assert_real_close
from test_oracle_pins import _parse_golden

pytestmark = pytest.mark.gpu

PI = math.pi
SHAPES = {
    "box": (O.BOX, [5.0, 5.0, 5.0]),
    "orb": (O.ORB, [20.0]),
    "tube": (O.TUBE, [5.0, 10.0, 15.0, 0.0, 4 * PI / 3]),
    "tube_full": (O.TUBE, [0.0, 8.0, 8.0, 0.0, 2 * PI]),
    "tube_narrow": (O.TUBE, [3.0, 9.0, 12.0, 0.4, 2.1]),
    "cone": (O.CONE, [2.0, 6.0, 4.0, 12.0, 20.0, 0.0, 2 * PI]),
    "cone_seg": (O.CONE, [2.0, 6.0, 4.0, 12.0, 20.0, 0.3, 5.9]),
    "cone_solid": (O.CONE, [0.0, 6.0, 0.0, 12.0, 20.0, 0.0, 2 * PI]),
    "trd": (O.TRD, [5.0, 10.0, 7.0, 3.0, 15.0]),
    "polycone": (O.POLYCONE, W.polycone_params(W.config_seed(3, 0))),
    "polycone_seg": (O.POLYCONE, [0.0, 4 * PI / 3] + W.polycone_params(W.config_seed(3, 0))[2:]),
    "polycone_step": (O.POLYCONE, list(W.STEPPED_POLYCONE)),
}


@pytest.fixture(scope="module")
def vg():
    import paper_1512_06637_b200 as vg
    return vg


def dev(arrs):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs]


def check_all(so, sg, t, what, classes=None):
    """All five queries on the same tracks, GPU against oracle."""
    dt = dev(t)
    cls_o = so.inside(*t[:3])
    if classes is not None:
        assert np.all(cls_o == classes), what
    assert_int_equal(sg.inside(*dt[:3]).cpu().numpy(), cls_o, what + " inside")
    for q in ("distance_to_in", "distance_to_out"):
        assert_real_close(getattr(sg, q)(*dt, W.STEP_MAX).cpu().numpy(), getattr(so, q)(*t, W.STEP_MAX), what + " " + q)
    for q in ("safety_to_in", "safety_to_out"):
        assert_real_close(getattr(sg, q)(*dt[:3]).cpu().numpy(), getattr(so, q)(*t[:3]), what + " " + q)


@pytest.mark.parametrize("row", _parse_golden("surface_examples.txt"), ids=lambda r: r[0])
def test_hand_worked_surface_points(vg, row):
    """S1-S31 against their hand-derived values (not against the oracle), also 1e-10 before and beyond the point."""
    eid, kind, par, p, d, res = row
    sg = vg.Shape(kind, par)
    for shift in (0.0, 1e-10, -1e-10):
        q = [np.array([p[i] + shift * d[i]]) for i in range(3)]
        dd = [np.array([float(v)]) for v in d]
        dt = dev(q + dd)
        for name, want in res.items():
            got = float(sg.inside(*dt[:3])[0]) if name == "inside" else float(getattr(sg, name)(*dt, 1e30)[0])
            if math.isinf(want) or name == "inside":
                assert got == want, (eid, name, shift, got)
            else:
                assert want - abs(shift) - 1e-9 <= got <= want + abs(shift) + 1e-9, (eid, name, shift, got, want)


def surface_tracks(so, kind, par, n, seed):
    """Tracks of the standard generator moved onto a crossing of their own line (the oracle's crossing list), both ways
    along the line; crossings within 1e-3 of another one and grazing ones are skipped."""
    c, h = W.bounding_half(kind, par)
    x, y, z, dx, dy, dz = W.draw_tracks(seed, n, c, tuple(1.5 * v for v in h), lambda x, y, z: np.abs(so.sdf(x, y, z)) < 1e-6)
    rng = np.random.default_rng(seed)
    P, D = [], []
    for i in range(n):
        p, d = np.array([x[i], y[i], z[i]]), np.array([dx[i], dy[i], dz[i]])
        t = so.line_crossings(p, d)
        if t.size == 0:
            continue
        k = int(rng.integers(t.size))
        gaps = np.abs(np.delete(t, k) - t[k])
        if gaps.size and gaps.min() < 1e-3:
            continue
        a, b = p + (t[k] - 1e-5) * d, p + (t[k] + 1e-5) * d
        if abs(so.sdf(*b)[0] - so.sdf(*a)[0]) / 2e-5 < 0.05:
            continue
        h_ = p + t[k] * d
        P += [h_, h_]
        D += [d, -d]
    P, D = np.array(P).T, np.array(D).T
    return [np.ascontiguousarray(a) for a in (*P, *D)]


@pytest.mark.parametrize("name", list(SHAPES))
def test_tracks_on_a_border_match_the_oracle(vg, name):
    kind, par = SHAPES[name]
    so, sg = O.Shape(kind, par), vg.Shape(kind, par)
    t = surface_tracks(so, kind, par, 6000, seed=1000 + len(name))
    assert t[0].size > 2000
    check_all(so, sg, t, name + " on the border", classes=O.SURFACE)
    # every such track goes either in (DistanceToIn 0) or out (DistanceToOut 0), never both
    dt = dev(t)
    din, dout = sg.distance_to_in(*dt, W.STEP_MAX).cpu().numpy(), sg.distance_to_out(*dt, W.STEP_MAX).cpu().numpy()
    assert np.all((din <= 1e-9) != (dout <= 1e-9))
    # the same points moved off the surface along the ray, inside the band (3e-10, 1e-16) and just out of it (5e-9)
    for sh in (3e-10, -3e-10, 1e-16, -1e-16, 5e-9, -5e-9):
        ts = [t[i] + sh * t[3 + i] for i in range(3)] + t[3:]
        check_all(so, sg, ts, "%s %g along the ray from the border" % (name, sh))


def test_configs1_tube_surface_starts_in_every_kernel_form(vg):
    """The direct, streaming and pipelined forms and the fused five-query call on border starts (a ragged size)."""
    kind, par = SHAPES["tube"]
    so, sg = O.Shape(kind, par), vg.Shape(kind, par)
    t = surface_tracks(so, kind, par, 4000, seed=4)
    dt = dev(t)
    want = {q: getattr(so, q)(*t, W.STEP_MAX) for q in ("distance_to_in", "distance_to_out")}
    try:
        for form in (vg.FORM_DIRECT, vg.FORM_STREAMING, vg.FORM_PIPELINED):
            vg.vg_set_option(vg.OPT_FORM, form)
            for q in want:
                assert_real_close(getattr(sg, q)(*dt, W.STEP_MAX).cpu().numpy(), want[q], "form %d %s" % (form, q))
    finally:
        vg.vg_set_option(vg.OPT_FORM, vg.FORM_AUTO)
    cls, din, dout, sin, sout = sg.query_all(*dt, W.STEP_MAX)
    assert_int_equal(cls.cpu().numpy(), so.inside(*t[:3]), "fused inside")
    assert_real_close(din.cpu().numpy(), want["distance_to_in"], "fused distance_to_in")
    assert_real_close(dout.cpu().numpy(), want["distance_to_out"], "fused distance_to_out")


def test_polycone_fused_call_on_border_starts(vg):
    for name in ("polycone", "polycone_seg", "polycone_step"):
        kind, par = SHAPES[name]
        so, sg = O.Shape(kind, par), vg.Shape(kind, par)
        t = surface_tracks(so, kind, par, 3000, seed=8)
        dt = dev(t)
        cls, din, dout, sin, sout = sg.query_all(*dt, W.STEP_MAX)
        assert_int_equal(cls.cpu().numpy(), so.inside(*t[:3]), name + " fused inside")
        assert_real_close(din.cpu().numpy(), so.distance_to_in(*t, W.STEP_MAX), name + " fused distance_to_in")
        assert_real_close(dout.cpu().numpy(), so.distance_to_out(*t, W.STEP_MAX), name + " fused distance_to_out")


# ------------------------------------------------------------------------------------------------ booleans

def boolean_surface_tracks(co, leaves, n_tracks, draw, seed):
    """Tracks moved onto a crossing of ANY primitive of the boolean (a border of it, or a surface hidden inside / outside
    the other operands), both ways along the line.  `leaves` = [(oracle Shape, 3x4 frame of the boolean -> primitive)]."""
    x, y, z, dx, dy, dz = draw(n_tracks)
    rng = np.random.default_rng(seed)
    P, D = [], []
    for i in range(x.size):
        p, d = np.array([x[i], y[i], z[i]]), np.array([dx[i], dy[i], dz[i]])
        per = [s.line_crossings(M[:, :3] @ p + M[:, 3], M[:, :3] @ d) for s, M in leaves]
        allt = np.concatenate(per)
        if allt.size == 0:
            continue
        j = int(rng.integers(allt.size))
        ts = float(allt[j])
        if np.sort(np.abs(np.delete(allt, j) - ts))[:1].min(initial=1.0) < 1e-3:
            continue
        owner = int(np.searchsorted(np.cumsum([q.size for q in per]), j, side="right"))
        s, M = leaves[owner]
        f = lambda q: s.sdf(*(M[:, :3] @ q + M[:, 3]))[0]
        if abs(f(p + (ts + 1e-5) * d) - f(p + (ts - 1e-5) * d)) / 2e-5 < 0.05:
            continue
        h = p + ts * d
        P += [h, h]
        D += [d, -d]
    P, D = np.array(P).T, np.array(D).T
    return [np.ascontiguousarray(a) for a in (*P, *D)]


@pytest.mark.parametrize("bc", W.boolean_cases(), ids=lambda b: b.name)
def test_boolean_tracks_on_operand_surfaces_match_the_oracle(vg, bc):
    co = O.Boolean(bc.op, O.Shape(bc.kind_a, bc.par_a), O.Shape(bc.kind_b, bc.par_b), bc.xform)
    cg = vg.Boolean(bc.op, vg.Shape(bc.kind_a, bc.par_a), vg.Shape(bc.kind_b, bc.par_b), bc.xform)
    draw = lambda n: bc.tracks(n, lambda x, y, z: np.abs(co.sdf(x, y, z)) < W.SURFACE_BAND)
    t = boolean_surface_tracks(co, co.leaves(), 4000, draw, seed=21)
    assert t[0].size > 1500
    cls = co.inside(*t[:3])
    assert (cls == O.SURFACE).sum() > 300 and (cls != O.SURFACE).sum() > 100  # borders of C and hidden surfaces
    check_all(co, cg, t, bc.name + " on an operand's surface")
    for sh in (3e-10, -3e-10, 1e-16, -1e-16):
        ts = [t[i] + sh * t[3 + i] for i in range(3)] + t[3:]
        check_all(co, cg, ts, "%s %g along the ray from an operand's surface" % (bc.name, sh))


@pytest.mark.parametrize("cc", W.csg_cases(), ids=lambda c: c.name)
def test_csg_tree_tracks_on_primitive_surfaces_match_the_oracle(vg, cc):
    co, cg = cc.build(O), cc.build(vg)
    draw = lambda n: cc.tracks(n, lambda x, y, z: np.abs(co.sdf(x, y, z)) < W.SURFACE_BAND)
    t = boolean_surface_tracks(co, co.leaves(), 3000, draw, seed=22)
    assert t[0].size > 1000
    check_all(co, cg, t, cc.name + " on a primitive's surface")


# ------------------------------------------------------------------------------- border-to-border transport

def build_world(vg, which):
    from test_oracle_world import build_mixed
    if which == "world":
        wc = W.world_case()
        so = [O.Shape(k, p) for k, p in zip(wc.kinds, wc.params)]
        wo = O.World(so, wc.parents, wc.xforms)
        wg = vg.World([vg.Shape(k, p) for k, p in zip(wc.kinds, wc.params)], wc.parents, wc.xforms)
    else:
        wc = W.mixed_world_case()
        so, wo = build_mixed(wc)
        _, wg = build_mixed(wc, vg)
    return wc, so, wo, wg


@pytest.mark.parametrize("which", ["world", "mixed"])
def test_border_to_border_walk_in_lockstep_with_the_oracle(vg, which):
    """Every step starts exactly where the last one ended, in the node Step returned (NO nudge).  The oracle walks; at every
    state the GPU's Step (next node bit-exact, step within tolerance) and Safety are compared with the oracle's."""
    wc, so, wo, wg = build_world(vg, which)

    def band(x, y, z):
        nd = wo.locate(x, y, z)
        return (nd < 0) | (wo.safety(np.maximum(nd, 0), x, y, z) < W.SURFACE_BAND)

    t = wc.tracks(20000, band)
    p, d = np.array(t[:3]), np.array(t[3:])
    node = wo.locate(*p)
    steps = 0
    while (node >= 0).any():
        idx = np.flatnonzero(node >= 0)
        cur = [np.ascontiguousarray(a) for a in (*p[:, idx], *d[:, idx])]
        st_o, nx_o = wo.step(node[idx], *cur, W.STEP_MAX)
        dn = torch.from_numpy(node[idx]).cuda()
        st_g, nx_g = wg.step(dn, *dev(cur), W.STEP_MAX)
        assert_int_equal(nx_g.cpu().numpy(), nx_o, "%s walk step %d next" % (which, steps))
        assert_real_close(st_g.cpu().numpy(), st_o, "%s walk step %d" % (which, steps))
        p[:, idx] += st_o * d[:, idx]
        node[idx] = nx_o
        steps += 1
        assert steps < 80
    assert steps > 5


@pytest.mark.parametrize("which", ["world", "mixed"])
def test_border_to_border_walk_on_the_gpu_alone(vg, which):
    """The same walk with the GPU's own steps and nodes: it ends, the steps add up to the straight way out of the root box,
    and half-way along every step the oracle's Locate finds the node the GPU was in."""
    wc, so, wo, wg = build_world(vg, which)

    def band(x, y, z):
        nd = wo.locate(x, y, z)
        return (nd < 0) | (wo.safety(np.maximum(nd, 0), x, y, z) < W.SURFACE_BAND)

    t = wc.tracks(40000, band)
    x, y, z, dx, dy, dz = dev(t)
    node = wg.locate(x, y, z)
    R = np.asarray(wc.xforms, dtype=np.float64).reshape(-1, 12)[0].reshape(3, 4)
    pl = R[:, :3] @ np.array(t[:3]) + R[:, 3:4]
    dl = R[:, :3] @ np.array(t[3:])
    straight = so[0].distance_to_out(*pl, *dl, 1e30)
    path = torch.zeros_like(x)
    zero_before = torch.zeros_like(x, dtype=torch.bool)
    for it in range(80):
        alive = node >= 0
        if not bool(alive.any()):
            break
        step, nxt = wg.step(node, x, y, z, dx, dy, dz)
        assert bool((step[alive] >= 0).all()) and bool(torch.isfinite(step[alive]).all())
        big = (alive & (step > 1e-6)).cpu().numpy()
        mid = [(c + 0.5 * step * dc).cpu().numpy()[big] for c, dc in ((x, dx), (y, dy), (z, dz))]
        assert np.array_equal(wo.locate(*mid), node.cpu().numpy()[big]), "step %d" % it
        zero = alive & (step <= 1e-9)
        assert not bool((zero & zero_before).any()), "two zero-length steps in a row"
        zero_before = zero
        x = torch.where(alive, x + step * dx, x)
        y = torch.where(alive, y + step * dy, y)
        z = torch.where(alive, z + step * dz, z)
        path = torch.where(alive, path + step, path)
        node = torch.where(alive, nxt, node)
    assert not bool((node >= 0).any())
    assert np.abs(path.cpu().numpy() - straight).max() < 1e-8


def test_compute_step_from_the_border_of_a_daughter(vg):
    """configs[4]: tracks taken to the daughter ComputeStep reported, then asked again in the mother from that point:
    moving on into the daughter the step is 0 with the same hit; moving back out the daughter is not hit again."""
    nav = W.navigator_case()
    vo = O.Volume(O.Shape(nav.mother_kind, nav.mother_params),
                  [O.Shape(k, p) for k, p in zip(nav.daughter_kinds, nav.daughter_params)], nav.xforms)
    vgv = vg.Volume(vg.Shape(nav.mother_kind, nav.mother_params),
                    [vg.Shape(k, p) for k, p in zip(nav.daughter_kinds, nav.daughter_params)], nav.xforms)
    t = nav.tracks(200000, band=lambda x, y, z: vo.safety(x, y, z) < W.SURFACE_BAND)
    step, hit = vo.compute_step(*t, W.STEP_MAX)
    sel = hit >= 0
    p = np.array(t[:3])[:, sel] + step[sel] * np.array(t[3:])[:, sel]
    d = np.array(t[3:])[:, sel]
    for sign in (1.0, -1.0):
        cur = [np.ascontiguousarray(a) for a in (*p, *(sign * d))]
        so_, ho_ = vo.compute_step(*cur, W.STEP_MAX)
        sg_, hg_ = vgv.compute_step(*dev(cur), W.STEP_MAX)
        assert_int_equal(hg_.cpu().numpy(), ho_, "compute_step from a daughter's border, sign %g" % sign)
        assert_real_close(sg_.cpu().numpy(), so_, "compute_step from a daughter's border, sign %g" % sign)
        if sign > 0:
            assert np.all(ho_ == hit[sel]) and np.all(so_ <= 1e-9)
        else:
            assert np.all(ho_ != hit[sel])
