"""GPU parity, part 2: the hand-worked examples through the CUDA path, degenerate rays, step_max, the navigation
step of BASELINE.json configs[4], the host-buffer entry points, streams."""
import math
import os

import numpy as np
import pytest

import oracle as O
import workloads as W
from parity import assert_int_equal, assert_real_close

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TWO_PI = 2 * math.pi
PI = math.pi


@pytest.fixture(scope="module")
def vg():
    import paper_1512_06637_b200 as m
    assert torch.cuda.is_available(), "the CUDA path needs a GPU; there is no fallback"
    return m


def dev(arrs):
    return [torch.from_numpy(np.ascontiguousarray(np.asarray(a, dtype=np.float64))).cuda() for a in arrs]


def oracle_band(s):
    return lambda x, y, z: np.abs(s.sdf(x, y, z)) < W.SURFACE_BAND


# ------------------------------------------------------------- worked examples E1-E21 (tests/golden) on the GPU

def _parse_golden():
    path = os.path.join(os.path.dirname(__file__), "golden", "worked_examples.txt")
    names = {"box": W.BOX, "orb": W.ORB, "tube": W.TUBE, "cone": W.CONE, "trd": W.TRD}
    sym = {"4PI3": 4 * PI / 3, "2PI": 2 * PI, "inf": math.inf}
    val = lambda t: sym[t] if t in sym else float(t)
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
def test_worked_examples_on_gpu(vg, row):
    eid, kind, par, p, d, res = row
    s = vg.Shape(kind, par)
    pt = dev([[v] for v in p])
    dt = dev([[v] for v in d]) if d is not None else None
    for q, want in res.items():
        if q == "inside":
            got = float(s.inside(*pt).cpu()[0])
        elif q.startswith("safety"):
            got = float(getattr(s, q)(*pt).cpu()[0])
        else:
            got = float(getattr(s, q)(*pt, *dt, 1e30).cpu()[0])
        if math.isinf(want):
            assert got == want, (eid, q, got)
        else:
            assert abs(got - want) <= max(1e-9, 1e-12 * abs(want)), (eid, q, got, want)


# ------------------------------------------------------------------------------------------- degenerate rays

SHAPES = {
    "box": (W.BOX, [5.0, 5.0, 5.0]),
    "orb": (W.ORB, [20.0]),
    "tube": (W.TUBE, [5.0, 10.0, 15.0, 0.0, 4 * PI / 3]),
    "cone": (W.CONE, [2.0, 6.0, 4.0, 12.0, 20.0, 0.0, TWO_PI]),
    "trd": (W.TRD, [5.0, 10.0, 7.0, 3.0, 15.0]),
    "polycone": (W.POLYCONE, W.polycone_params(W.config_seed(3, 0))),
    # cylindrical patches (B = 0) seen from the axis: b = -0.0 in the quadratic (the root selection reads the sign bit)
    "cone_cylinder": (W.CONE, [3.0, 8.0, 3.0, 8.0, 10.0, 0.0, TWO_PI]),
    "polycone_step": (W.POLYCONE, [0.0, TWO_PI, 7.0, -12.0, 0.0, 6.0, -4.0, 1.0, 8.0, -4.0, 3.0, 12.0, 2.0, 2.0, 10.0, 6.0, 2.0, 11.0,
                                   6.0, 0.0, 5.0, 14.0, 1.5, 4.0]),
}


@pytest.mark.parametrize("name", list(SHAPES))
def test_axis_aligned_and_planar_directions(vg, name):
    """Directions with one or two components exactly zero (hard part H4): the select-based
    kernels must give what the oracle's explicit branches give."""
    kind, par = SHAPES[name]
    so, sg = O.Shape(kind, par), vg.Shape(kind, par)
    c, h = W.bounding_half(kind, par)
    x, y, z, dx, dy, dz = W.draw_tracks(5, 60000, c, tuple(1.5 * v for v in h), oracle_band(so))
    n = len(x)
    rng = np.random.default_rng(1)
    mode = rng.integers(0, 9, n)
    sgn = rng.choice([-1.0, 1.0], n)
    ang = rng.uniform(0, TWO_PI, n)
    for m, (a, b, c_) in enumerate([(1, 0, 0), (0, 1, 0), (0, 0, 1)]):
        k = mode == m
        dx[k], dy[k], dz[k] = a * sgn[k], b * sgn[k], c_ * sgn[k]
    k = mode == 3
    dx[k], dy[k], dz[k] = np.cos(ang[k]), np.sin(ang[k]), 0.0
    k = mode == 4
    dx[k], dy[k], dz[k] = np.cos(ang[k]), 0.0, np.sin(ang[k])
    k = mode == 5
    dx[k], dy[k], dz[k] = 0.0, np.cos(ang[k]), np.sin(ang[k])
    k = mode == 6  # negative zeros
    dx[k], dy[k], dz[k] = -0.0, sgn[k], -0.0
    t = (x, y, z, dx, dy, dz)
    dt = dev(t)
    for q in ("distance_to_in", "distance_to_out"):
        o = getattr(so, q)(*t, W.STEP_MAX)
        g = getattr(sg, q)(*dt, W.STEP_MAX).cpu().numpy()
        assert_real_close(g, o, "%s %s degenerate directions" % (name, q))


@pytest.mark.parametrize("name", list(SHAPES))
def test_points_on_symmetry_axes_and_planes(vg, name):
    """Points with exactly zero coordinates (rho = 0 on the axis of a solid of revolution, the mid-planes)."""
    kind, par = SHAPES[name]
    so, sg = O.Shape(kind, par), vg.Shape(kind, par)
    c, h = W.bounding_half(kind, par)
    x, y, z, dx, dy, dz = W.draw_tracks(6, 40000, c, tuple(1.5 * v for v in h))
    rng = np.random.default_rng(2)
    mode = rng.integers(0, 6, len(x))
    x[(mode == 0) | (mode == 3)] = 0.0
    y[(mode == 1) | (mode == 3)] = 0.0
    z[mode == 2] = c[2]
    keep = np.abs(so.sdf(x, y, z)) >= W.SURFACE_BAND
    t = tuple(a[keep] for a in (x, y, z, dx, dy, dz))
    dt = dev(t)
    for q in W.QUERIES5:
        if q.startswith("distance"):
            o = getattr(so, q)(*t, W.STEP_MAX)
            g = getattr(sg, q)(*dt, W.STEP_MAX).cpu().numpy()
            assert_real_close(g, o, "%s %s axis points" % (name, q))
        elif q == "inside":
            assert_int_equal(sg.inside(*dt[:3]).cpu().numpy(), so.inside(*t[:3]), "%s inside axis points" % name)
        else:
            assert_real_close(getattr(sg, q)(*dt[:3]).cpu().numpy(), getattr(so, q)(*t[:3]), "%s %s axis points" % (name, q))


@pytest.mark.parametrize("name", list(SHAPES))
def test_step_max_turns_far_hits_into_misses(vg, name):
    kind, par = SHAPES[name]
    so, sg = O.Shape(kind, par), vg.Shape(kind, par)
    c, h = W.bounding_half(kind, par)
    t = W.draw_tracks(8, 50001, c, tuple(1.5 * v for v in h), oracle_band(so))
    dt = dev(t)
    for step_max in (0.0, 3.0, 11.5, math.inf):
        for q in ("distance_to_in", "distance_to_out"):
            o = getattr(so, q)(*t, step_max)
            g = getattr(sg, q)(*dt, step_max).cpu().numpy()
            assert_real_close(g, o, "%s %s step_max=%r" % (name, q, step_max))


def test_permuting_tracks_permutes_results(vg):
    """the geometry calculations of different particles are independent of each other."""
    kind, par = SHAPES["tube"]
    sg = vg.Shape(kind, par)
    c, h = W.bounding_half(kind, par)
    t = W.draw_tracks(9, 70001, c, tuple(1.5 * v for v in h))
    perm = np.random.default_rng(3).permutation(len(t[0]))
    a = sg.distance_to_in(*dev(t), 1e30).cpu().numpy()
    b = sg.distance_to_in(*dev([v[perm] for v in t]), 1e30).cpu().numpy()
    assert np.array_equal(a[perm], b)


def test_non_default_stream_and_concurrent_handles(vg):
    kind, par = SHAPES["cone"]
    so, sg = O.Shape(kind, par), vg.Shape(kind, par)
    c, h = W.bounding_half(kind, par)
    t = W.draw_tracks(10, 300001, c, tuple(1.5 * v for v in h), oracle_band(so))
    dt = dev(t)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    with torch.cuda.stream(s1):
        a = sg.distance_to_in(*dt, 1e30)
    with torch.cuda.stream(s2):
        b = sg.safety_to_in(*dt[:3])
    c_ = sg.distance_to_out(*dt, 1e30, stream=s1)
    torch.cuda.synchronize()
    assert_real_close(a.cpu().numpy(), so.distance_to_in(*t, 1e30), "stream s1")
    assert_real_close(b.cpu().numpy(), so.safety_to_in(*t[:3]), "stream s2")
    assert_real_close(c_.cpu().numpy(), so.distance_to_out(*t, 1e30), "explicit stream")


def test_bad_arguments_raise(vg):
    sg = vg.Shape(W.BOX, [5, 5, 5])
    x = torch.zeros(8, dtype=torch.float64, device="cuda")
    with pytest.raises(TypeError):
        sg.inside(x.float(), x, x)
    with pytest.raises(ValueError):
        sg.inside(x, x[:4], x)
    with pytest.raises(TypeError):
        sg.inside(x.cpu(), x.cpu(), x.cpu())
    with pytest.raises(vg.VgError):
        sg.distance_to_in(x, x, x, x, x, x, step_max=-1.0)
    with pytest.raises(vg.VgError):
        sg.distance_to_in(x, x, x, x, x, x, step_max=float("nan"))


# ------------------------------------------------------------------------------ navigation (configs[4])

def build_volumes(vg, nav, order=None, nd=None):
    idx = list(range(len(nav.daughter_kinds))) if order is None else list(order)
    if nd is not None:
        idx = idx[:nd]
    mo = O.Shape(nav.mother_kind, nav.mother_params)
    mg = vg.Shape(nav.mother_kind, nav.mother_params)
    do = [O.Shape(nav.daughter_kinds[i], nav.daughter_params[i]) for i in idx]
    dg = [vg.Shape(nav.daughter_kinds[i], nav.daughter_params[i]) for i in idx]
    xf = nav.xforms[idx] if idx else np.zeros((0, 12))
    return O.Volume(mo, do, xf), vg.Volume(mg, dg, xf)


def nav_tracks(nav, vol, n, seed=None):
    band = lambda x, y, z: vol.safety(x, y, z) < W.SURFACE_BAND
    return W.draw_tracks(nav.seed if seed is None else seed, n, nav.center, nav.half, band)


def check_step(vo, vgv, t, step_max, what):
    so, ho = vo.compute_step(*t, step_max)
    sg, hg = vgv.compute_step(*dev(t), step_max)
    torch.cuda.synchronize()
    assert_int_equal(hg.cpu().numpy(), ho, what + " hit")
    assert_real_close(sg.cpu().numpy(), so, what + " step")
    return so, ho


def test_config4_full_size(vg):
    nav = W.navigator_case()
    vo, vgv = build_volumes(vg, nav)
    t = nav_tracks(nav, vo, nav.sizes[-1])
    so, ho = check_step(vo, vgv, t, W.STEP_MAX, "cfg4")
    frac = (ho >= 0).mean()
    assert 0.15 < frac < 0.30 and len(set(ho.tolist())) == 65  # every daughter and the mother are hit


@pytest.mark.parametrize("n", [1, 2, 127, 128, 129, 100003])
def test_config4_ragged(vg, n):
    nav = W.navigator_case()
    vo, vgv = build_volumes(vg, nav)
    t = nav_tracks(nav, vo, n, seed=nav.seed + 1)
    check_step(vo, vgv, t, W.STEP_MAX, "cfg4 n=%d" % n)


@pytest.mark.parametrize("step_max", [0.0, 5.0, 40.0, 150.0, math.inf])
def test_physics_step_limits_the_geometric_step(vg, step_max):
    """the smaller of the physics step and the distance to the border wins (hit = -2)."""
    nav = W.navigator_case()
    vo, vgv = build_volumes(vg, nav)
    t = nav_tracks(nav, vo, 200001, seed=nav.seed + 2)
    so, ho = check_step(vo, vgv, t, step_max, "cfg4 step_max=%r" % step_max)
    if step_max < 100:
        assert (ho == -2).any()


@pytest.mark.parametrize("nd", [0, 1, 2, 7, 33])
def test_fewer_daughters_and_permuted_order(vg, nd):
    nav = W.navigator_case()
    order = np.random.default_rng(4).permutation(64)
    vo, vgv = build_volumes(vg, nav, order=order, nd=nd)
    t = nav_tracks(nav, vo, 150001, seed=nav.seed + 3)
    check_step(vo, vgv, t, W.STEP_MAX, "nd=%d" % nd)


def test_tracks_that_break_the_contract(vg):
    """Tracks outside the mother get (-1, -1); a daughter the track is inside of is skipped (R13)."""
    nav = W.navigator_case()
    vo, vgv = build_volumes(vg, nav)
    x, y, z, dx, dy, dz = W.draw_tracks(99, 120001, (0, 0, 0), (130, 130, 130))
    keep = (np.abs(vo.mother.sdf(x, y, z)) >= 1e-6)
    for d, xf in zip(vo.daughters, vo.xforms):
        M = xf.reshape(3, 4)
        lx, ly, lz = (M[i, 0] * x + M[i, 1] * y + M[i, 2] * z + M[i, 3] for i in range(3))
        keep &= np.abs(d.sdf(lx, ly, lz)) >= 1e-6
    t = tuple(a[keep] for a in (x, y, z, dx, dy, dz))
    so, ho = check_step(vo, vgv, t, W.STEP_MAX, "contract violations")
    assert (so == -1.0).any()


def test_mixed_daughter_kinds_and_mothers(vg):
    """Daughters of every supported kind (box, orb, tube segment, cone segment, trd) in a tube mother."""
    rng = np.random.default_rng(12)
    kinds = [W.BOX, W.ORB, W.TUBE, W.CONE, W.TRD, W.TUBE, W.CONE, W.ORB]
    pars = [[3, 4, 5], [5], [2, 5, 4, 0.3, 4.0], [1, 3, 2, 5, 4, 0.0, TWO_PI], [2, 4, 3, 1, 5], [0, 4, 6, 0, TWO_PI],
            [0, 3, 2, 5, 4, 1.0, 2.5], [3]]
    centers = [(-20, -20, -20), (20, -20, -20), (-20, 20, -20), (20, 20, -20), (-20, -20, 20), (20, -20, 20),
               (-20, 20, 20), (20, 20, 20)]
    xf = []
    for c in centers:
        u1, u2, u3 = rng.random(3)
        q = (math.sqrt(1 - u1) * math.sin(TWO_PI * u2), math.sqrt(1 - u1) * math.cos(TWO_PI * u2),
             math.sqrt(u1) * math.sin(TWO_PI * u3), math.sqrt(u1) * math.cos(TWO_PI * u3))
        xf.append(W.placement(W.quaternion_to_matrix(q), c))
    xf = np.stack(xf)
    for mk, mp in ((W.TUBE, [0, 45, 40, 0, TWO_PI]), (W.ORB, [50]), (W.TRD, [40, 45, 42, 38, 40]),
                   (W.CONE, [0, 45, 0, 50, 40, 0, TWO_PI])):
        vo = O.Volume(O.Shape(mk, mp), [O.Shape(k, p) for k, p in zip(kinds, pars)], xf)
        vgv = vg.Volume(vg.Shape(mk, mp), [vg.Shape(k, p) for k, p in zip(kinds, pars)], xf)
        t = W.draw_tracks(31, 120001, (0, 0, 0), (36, 36, 36), lambda x, y, z: vo.safety(x, y, z) < 1e-6)
        so, ho = check_step(vo, vgv, t, W.STEP_MAX, "mixed kinds mother=%d" % mk)
        assert len(set(ho.tolist())) == 9
        sg = vgv.safety(*dev(t[:3])).cpu().numpy()
        assert_real_close(sg, vo.safety(*t[:3]), "volume safety mother=%d" % mk)


@pytest.mark.parametrize("nd, size, spread", [(65, 6.0, 40.0), (100, 20.0, 30.0), (130, 8.0, 45.0), (256, 12.0, 40.0),
                                              (64, 30.0, 10.0)])
def test_many_overlapping_daughters_of_all_kinds(vg, nd, size, spread):
    """More than one chunk of 64 daughters (two- and four-chunk kernels), five kinds, heavy overlap: a track has many
    candidates of one kind, so the warp's shared work list takes several passes; tracks start anywhere in the mother
    (inside a daughter: that daughter is skipped, R13).  Every step and hit index against the oracle."""
    rng = np.random.default_rng(nd * 31 + int(size))
    kinds, pars, xf = [], [], []
    for _ in range(nd):
        kind = [W.BOX, W.ORB, W.TUBE, W.CONE, W.TRD][rng.integers(0, 5)]
        a, b, c = size * rng.uniform(0.3, 1.0, 3)
        par = {W.BOX: [a, b, c], W.ORB: [a], W.TUBE: [0.3 * a, a, b, 0.5, 4.0],
               W.CONE: [0.2 * a, a, 0.3 * b, 1.2 * b, c, 0.0, TWO_PI], W.TRD: [a, 0.5 * a, b, 1.3 * b, c]}[kind]
        q = rng.normal(size=4)
        q /= np.linalg.norm(q)
        kinds.append(kind)
        pars.append(par)
        xf.append(W.placement(W.quaternion_to_matrix(tuple(q)), rng.uniform(-spread, spread, 3)))
    xf = np.stack(xf)
    vo = O.Volume(O.Shape(W.BOX, [60, 60, 60]), [O.Shape(k, p) for k, p in zip(kinds, pars)], xf)
    vgv = vg.Volume(vg.Shape(W.BOX, [60, 60, 60]), [vg.Shape(k, p) for k, p in zip(kinds, pars)], xf)

    def band(x, y, z):
        near = np.abs(vo.mother.sdf(x, y, z)) < 1e-6
        for d, m in zip(vo.daughters, vo.xforms):
            M = m.reshape(3, 4)
            lx, ly, lz = (M[i, 0] * x + M[i, 1] * y + M[i, 2] * z + M[i, 3] for i in range(3))
            near |= np.abs(d.sdf(lx, ly, lz)) < 1e-6
        return near

    t = W.draw_tracks(77 + nd, 100003, (0, 0, 0), (60, 60, 60), band)
    try:
        for form in (1, 2, 0):  # every lane walks its own candidates / the warp pools them / the library's choice
            vg.vg_set_option(vg.OPT_NAV_FORM, form)
            for step_max in (W.STEP_MAX, 25.0):
                so, ho = check_step(vo, vgv, t, step_max, "nd=%d step_max=%g form=%d" % (nd, step_max, form))
    finally:
        vg.vg_set_option(vg.OPT_NAV_FORM, 0)
    assert len(set(ho.tolist())) > min(nd, 40) // 2
    # vg_volume_safety is the plain minimum over the mother and EVERY daughter whatever the containment contract says:
    # points inside several overlapping daughters, and points up to 1.3 half-lengths out (beyond the mother, beyond the
    # safety grid's box and, for some, beyond the bounding box of the daughters' spheres)
    assert_real_close(vgv.safety(*dev(t[:3])).cpu().numpy(), vo.safety(*t[:3]), "volume safety nd=%d, anywhere in the mother" % nd)
    p = W.draw_tracks(78 + nd, 100003, (0, 0, 0), (78, 78, 78), band)[:3]
    so_ = vo.safety(*p)
    assert (so_ < -1.0).sum() > 1000 and (so_ > 1.0).sum() > 1000
    assert_real_close(vgv.safety(*dev(p)).cpu().numpy(), so_, "volume safety nd=%d, beyond the mother" % nd)


def test_random_volumes_step_and_safety_soak(vg):
    """Seeded random volumes (VG_STRESS_REPS of them, default 12): 1..256 daughters of the five kinds, sizes from a
    hundredth to a third of the mother, clustered or spread, in a box / orb / tube mother -- every geometry gives the
    candidate grid and the safety grid other cells, lists and margins.  ComputeStep (steps, hit indices) for tracks
    anywhere in the mother, the volume safety for points up to 1.3 half-lengths out, against the oracle."""
    reps = int(os.environ.get("VG_STRESS_REPS", "12"))
    for rep in range(reps):
        rng = np.random.default_rng(9000 + rep)
        nd = int(rng.choice([1, 2, 7, 8, 9, 13, 40, 63, 64, 65, 128, 129, 200, 256]))
        H = float(rng.choice([10.0, 60.0, 1000.0]))
        size = H * float(rng.choice([0.01, 0.05, 0.15, 0.33]))
        spread = H * float(rng.choice([0.2, 0.6, 0.85]))
        kinds, pars, xf = [], [], []
        for _ in range(nd):
            kind = [W.BOX, W.ORB, W.TUBE, W.CONE, W.TRD][rng.integers(0, 5)]
            a, b, c = size * rng.uniform(0.3, 1.0, 3)
            par = {W.BOX: [a, b, c], W.ORB: [a], W.TUBE: [0.3 * a, a, b, 0.5, 4.0],
                   W.CONE: [0.2 * a, a, 0.3 * b, 1.2 * b, c, 0.0, TWO_PI], W.TRD: [a, 0.5 * a, b, 1.3 * b, c]}[kind]
            q = rng.normal(size=4)
            kinds.append(kind)
            pars.append(par)
            xf.append(W.placement(W.quaternion_to_matrix(tuple(q / np.linalg.norm(q))), rng.uniform(-spread, spread, 3)))
        xf = np.stack(xf)
        mk, mp = [(W.BOX, [H, H, H]), (W.ORB, [1.6 * H]), (W.TUBE, [0.0, 1.5 * H, H, 0.0, TWO_PI])][rep % 3]
        vo = O.Volume(O.Shape(mk, mp), [O.Shape(k, p) for k, p in zip(kinds, pars)], xf)
        vgv = vg.Volume(vg.Shape(mk, mp), [vg.Shape(k, p) for k, p in zip(kinds, pars)], xf)
        band_w = 1e-6 * max(1.0, H / 60.0)

        def band(x, y, z):
            near = np.abs(vo.mother.sdf(x, y, z)) < band_w
            for d, m in zip(vo.daughters, vo.xforms):
                M = m.reshape(3, 4)
                lx, ly, lz = (M[i, 0] * x + M[i, 1] * y + M[i, 2] * z + M[i, 3] for i in range(3))
                near |= np.abs(d.sdf(lx, ly, lz)) < band_w
            return near
        what = "soak %d: nd=%d H=%g size=%g spread=%g mother=%d" % (rep, nd, H, size, spread, mk)
        t = W.draw_tracks(9100 + rep, 20011, (0, 0, 0), (H, H, H), lambda x, y, z: band(x, y, z) | (vo.mother.sdf(x, y, z) > 0))
        for step_max in (W.STEP_MAX, 0.4 * H):
            check_step(vo, vgv, t, step_max, what + " step_max=%g" % step_max)
        p = W.draw_tracks(9200 + rep, 30011, (0, 0, 0), (1.3 * H,) * 3, band)[:3]
        assert_real_close(vgv.safety(*dev(p)).cpu().numpy(), vo.safety(*p), what + " safety")
        # ... and around the daughters, where the lists of the safety grid's cells matter most
        k = rng.integers(0, nd, 20011)
        c = -np.einsum("nji,nj->ni", xf.reshape(-1, 3, 4)[k][:, :, :3], xf.reshape(-1, 3, 4)[k][:, :, 3])
        q3 = c + rng.uniform(-2.5 * size, 2.5 * size, (20011, 3))
        q3 = tuple(np.ascontiguousarray(q3[:, a]) for a in range(3))
        keep = ~band(*q3)
        q3 = tuple(np.ascontiguousarray(a[keep]) for a in q3)
        assert_real_close(vgv.safety(*dev(q3)).cpu().numpy(), vo.safety(*q3), what + " safety around the daughters")


@pytest.mark.parametrize("form", [1, 2])
def test_config4_both_forms_of_phase_two(vg, form):
    nav = W.navigator_case()
    vo, vgv = build_volumes(vg, nav)
    t = nav_tracks(nav, vo, 300007, seed=nav.seed + 9)
    try:
        vg.vg_set_option(vg.OPT_NAV_FORM, form)
        check_step(vo, vgv, t, W.STEP_MAX, "cfg4 form=%d" % form)
        check_step(vo, vgv, t, 30.0, "cfg4 form=%d step_max=30" % form)
    finally:
        vg.vg_set_option(vg.OPT_NAV_FORM, 0)


def test_volume_safety_config4(vg):
    nav = W.navigator_case()
    vo, vgv = build_volumes(vg, nav)
    t = nav_tracks(nav, vo, 300001, seed=nav.seed + 5)
    assert_real_close(vgv.safety(*dev(t[:3])).cpu().numpy(), vo.safety(*t[:3]), "volume safety")


def test_volume_create_rejects_bad_input(vg):
    m = vg.Shape(W.BOX, [10, 10, 10])
    d = vg.Shape(W.BOX, [1, 1, 1])
    bad = [[2, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]]
    with pytest.raises(vg.VgError):
        vg.Volume(m, [d], bad)


def test_volume_with_polycone_and_boolean_solids(vg):
    """A one-level volume whose solids are not all primitives (reading R30) is served by the world kernels behind
    vg_compute_step / vg_volume_safety: same conventions (hit = daughter index, -1 mother exit, -2 physics step)."""
    bools = {b.name: b for b in W.boolean_cases()}
    b1 = bools["box_minus_tube"]
    specs = [("shape", W.POLYCONE, W.STEPPED_POLYCONE, (-40.0, -40.0, 0.0)), ("boolean", b1, None, (40.0, -40.0, 5.0)),
             ("shape", W.TUBE, [5.0, 10.0, 15.0, 0.0, 4 * PI / 3], (-40.0, 40.0, -5.0)),
             ("shape", W.POLYCONE, [0.5, 4.0] + W.STEPPED_POLYCONE[2:], (40.0, 40.0, 0.0)),
             # a boolean with a polycone operand (vg_boolx.cu) as a placed solid: stepped polycone minus an off-centre box
             # (faces at z = -2.9 and 5.5: none in a plane of the polycone, where the two operands' crossings would tie)
             ("pair", (W.SUBTRACTION, W.POLYCONE, W.STEPPED_POLYCONE, W.BOX, [3.0, 20.0, 4.2], W.placement(np.eye(3), (5.0, 0.0, 1.3))),
              None, (0.0, 0.0, 0.0))]
    rng = np.random.default_rng(12)

    def mk(mod, sp):
        if sp[0] == "shape":
            return mod.Shape(sp[1], sp[2])
        if sp[0] == "pair":
            op, ka, pa, kb, pb, xb = sp[1]
            return mod.Boolean(op, mod.Shape(ka, pa), mod.Shape(kb, pb), xb)
        b = sp[1]
        return mod.Boolean(b.op, mod.Shape(b.kind_a, b.par_a), mod.Shape(b.kind_b, b.par_b), b.xform)
    xf = []
    for sp in specs:
        q = rng.normal(size=4)
        xf.append(W.placement(W.quaternion_to_matrix(tuple(q / np.linalg.norm(q))), sp[3]))
    ident = W.placement(np.eye(3), (0, 0, 0))
    for mother in (("shape", W.BOX, [80.0, 80.0, 40.0]), ("boolean", bools["box_union_orb"].__class__(
            "m", W.SUBTRACTION, W.BOX, [80.0, 80.0, 40.0], W.ORB, [6.0], (0.0, 0.0, 0.0), (0.0, 0.0, 0.0, 1.0), 1), None)):
        wo = O.World([mk(O, mother)] + [mk(O, sp) for sp in specs], [-1] + [0] * len(specs), [ident] + xf)
        vgv = vg.Volume(mk(vg, mother), [mk(vg, sp) for sp in specs], xf)

        def band(x, y, z):
            nd = wo.locate(x, y, z)
            zero = np.zeros(x.size, dtype=np.int32)
            return (nd != 0) | (wo.safety(zero, x, y, z) < 1e-4)  # in the mother, outside every daughter, clear of operands too
        t = W.draw_tracks(91, 150001, (0, 0, 0), (80, 80, 40), band)
        zero = np.zeros(t[0].size, dtype=np.int32)
        for step_max in (W.STEP_MAX, 20.0):
            so, no = wo.step(zero, *t, step_max)
            sg, hg = vgv.compute_step(*dev(t), step_max)
            want_hit = np.where(no == 0, -2, np.where(no < 0, -1, no - 1))
            assert_int_equal(hg.cpu().numpy(), want_hit, "general volume hit")
            assert_real_close(sg.cpu().numpy(), so, "general volume step")
        assert set(np.unique(want_hit)) >= {-2, -1, 0, 1, 2, 3, 4}
        assert_real_close(vgv.safety(*dev(t[:3])).cpu().numpy(), wo.safety(zero, *t[:3]), "general volume safety")
        # the same solids as a world: Locate of points anywhere (inside the daughters too), node indices bit-exact
        wg = vg.World([mk(vg, mother)] + [mk(vg, sp) for sp in specs], [-1] + [0] * len(specs), [ident] + xf)
        p = W.draw_tracks(92, 150001, (0, 0, 0), (80, 80, 40), lambda x, y, z: np.zeros(x.size, dtype=bool))[:3]
        node_o = wo.locate(*p)
        clear = np.ones(p[0].size, dtype=bool)
        for nd in range(len(specs) + 1):  # keep points clear of every node's surface band (R7)
            clear &= np.abs(wo.safety(np.full(p[0].size, nd, dtype=np.int32), *p)) > 1e-6
        pc = tuple(np.ascontiguousarray(a[clear]) for a in p)
        assert_int_equal(wg.locate(*dev(pc)).cpu().numpy(), node_o[clear], "world locate with a polycone-operand boolean")
        assert (node_o[clear] == len(specs)).any()


def test_volume_of_many_mixed_solids_uses_the_grids(vg):
    """27 daughters on a 3 x 3 x 3 lattice -- primitives, polycones, booleans, CSG trees and EMPTY booleans of all three record kinds (a solid minus
    a far larger box: SafetyToIn > 0 everywhere and larger than |p - c| + r, so it must not bound the nearest-daughter
    search) -- in one volume: more than 12 children, so the world kernels behind it take the candidate grid (Step, Locate)
    and the safety grid (Safety).  Steps, hit indices, safeties and Locate against the oracle."""
    bools = {b.name: b for b in W.boolean_cases()}
    rng = np.random.default_rng(2718)
    # (B far larger than A: the empty solid's SafetyToIn is ~500 everywhere, far above |p - c| + r of its bounding sphere)
    empty = ("pair", (W.SUBTRACTION, W.BOX, [3.0, 3.0, 3.0], W.BOX, [500.0, 500.0, 500.0], W.placement(np.eye(3), (0.5, 0.0, 0.0))))
    menu = [("shape", W.BOX, [5.0, 7.0, 4.0]), ("shape", W.ORB, [7.0]), ("shape", W.TUBE, [2.0, 6.0, 7.0, 0.3, 4.0]),
            ("shape", W.CONE, [1.0, 4.0, 2.0, 7.0, 6.0, 0.0, TWO_PI]), ("shape", W.TRD, [3.0, 6.0, 5.0, 2.0, 6.0]),
            ("shape", W.POLYCONE, [0.0, TWO_PI, 4.0, -7.0, 0.0, 3.0, -2.0, 1.0, 7.0, 3.0, 2.0, 5.0, 7.0, 0.0, 2.0]),
            ("boolean", bools["box_union_orb"]), ("pair", (W.SUBTRACTION, W.ORB, [8.0], W.TUBE, [0.0, 3.0, 9.0, 0.0, TWO_PI],
                                                              W.placement(np.eye(3), (1.0, 0.5, 0.0)))), empty,
            ("tree", bools["box_union_orb"], (W.SUBTRACTION, W.TUBE, [0.0, 2.5, 12.0, 0.0, TWO_PI], W.placement(np.eye(3), (-1.0, 0.0, 0.0)))),
            # ... an empty CSG tree and an empty boolean with a polycone operand (other record kinds inside the library)
            # (small, so that their bounding spheres would be a tight -- and wrong -- upper bound)
            ("tree", W.BooleanCase("tiny", W.UNION, W.BOX, [2.0, 2.0, 2.0], W.ORB, [2.0], (1.0, 0.0, 0.0), (0.0, 0.0, 0.0, 1.0), 1),
             (W.SUBTRACTION, W.BOX, [500.0, 500.0, 500.0], W.placement(np.eye(3), (0.0, 0.0, 0.0)))),
            ("pair", (W.SUBTRACTION, W.POLYCONE, [0.0, TWO_PI, 3.0, -2.0, 0.0, 1.0, 0.0, 0.5, 2.0, 2.0, 0.0, 1.0], W.BOX, [500.0, 500.0, 500.0],
                      W.placement(np.eye(3), (0.0, 0.0, 0.0))))]
    specs, xf = [], []
    k = 0
    for ix in (-1, 0, 1):
        for iy in (-1, 0, 1):
            for iz in (-1, 0, 1):
                specs.append(menu[k % len(menu)])
                k += 1
                q = rng.normal(size=4)
                c = np.array([ix, iy, iz]) * 26.0 + rng.uniform(-2.0, 2.0, 3)
                xf.append(W.placement(W.quaternion_to_matrix(tuple(q / np.linalg.norm(q))), tuple(c)))

    def mk(mod, sp):
        if sp[0] == "shape":
            return mod.Shape(sp[1], sp[2])
        if sp[0] == "pair":
            op, ka, pa, kb, pb, xb = sp[1]
            return mod.Boolean(op, mod.Shape(ka, pa), mod.Shape(kb, pb), xb)
        b = sp[1]
        inner = mod.Boolean(b.op, mod.Shape(b.kind_a, b.par_a), mod.Shape(b.kind_b, b.par_b), b.xform)
        if sp[0] == "tree":  # (A op B) op2 C: a CSG tree of three primitives (R31)
            op2, kc, pc, xc = sp[2]
            return mod.Boolean(op2, inner, mod.Shape(kc, pc), xc)
        return inner
    ident = W.placement(np.eye(3), (0, 0, 0))
    mother = ("shape", W.BOX, [60.0, 60.0, 60.0])  # well clear of the lattice: near a daughter, its neighbours are nearer than the mother
    wo = O.World([mk(O, mother)] + [mk(O, sp) for sp in specs], [-1] + [0] * len(specs), [ident] + xf)
    vgv = vg.Volume(mk(vg, mother), [mk(vg, sp) for sp in specs], xf)
    wg = vg.World([mk(vg, mother)] + [mk(vg, sp) for sp in specs], [-1] + [0] * len(specs), [ident] + xf)
    n_nodes = len(specs) + 1

    def near_a_surface(x, y, z):
        near = np.zeros(x.size, dtype=bool)
        for nd in range(n_nodes):
            near |= np.abs(wo.safety(np.full(x.size, nd, dtype=np.int32), x, y, z)) < 1e-4
        return near
    t = W.draw_tracks(93, 120001, (0, 0, 0), (60, 60, 60), lambda x, y, z: (wo.locate(x, y, z) != 0) | near_a_surface(x, y, z))
    zero = np.zeros(t[0].size, dtype=np.int32)
    for step_max in (W.STEP_MAX, 15.0):
        so, no = wo.step(zero, *t, step_max)
        sg, hg = vgv.compute_step(*dev(t), step_max)
        want_hit = np.where(no == 0, -2, np.where(no < 0, -1, no - 1))
        assert_int_equal(hg.cpu().numpy(), want_hit, "many mixed solids hit step_max=%g" % step_max)
        assert_real_close(sg.cpu().numpy(), so, "many mixed solids step step_max=%g" % step_max)
    hits = set(np.unique(want_hit).tolist())
    is_empty = lambda sp: sp is empty or (sp[0] in ("pair", "tree") and 500.0 in (sp[1][4] if sp[0] == "pair" else sp[2][2]))
    assert sum(is_empty(sp) for sp in specs) >= 6
    assert len(hits) >= 17 and not any(is_empty(specs[h]) for h in hits if h >= 0)  # nothing ever hits an empty solid
    assert_real_close(vgv.safety(*dev(t[:3])).cpu().numpy(), wo.safety(zero, *t[:3]), "many mixed solids safety")
    # points anywhere (inside the daughters, outside the mother): Locate bit-exact, per-node safety of the mother
    p = W.draw_tracks(94, 120001, (0, 0, 0), (70, 70, 70), near_a_surface)[:3]
    assert_int_equal(wg.locate(*dev(p)).cpu().numpy(), wo.locate(*p), "many mixed solids locate")
    zp = np.zeros(p[0].size, dtype=np.int32)
    assert_real_close(wg.safety(torch.from_numpy(zp).cuda(), *dev(p)).cpu().numpy(), wo.safety(zp, *p), "many mixed solids safety anywhere")
    # points around the centres of the empty solids: the nearest daughter is a NEIGHBOUR, 15-20 away, although the empty
    # solid's bounding sphere is right there
    rng = np.random.default_rng(5)
    cs = np.stack([-(np.asarray(m).reshape(3, 4)[:, :3].T @ np.asarray(m).reshape(3, 4)[:, 3]) for sp, m in zip(specs, xf) if is_empty(sp)])
    q = cs[rng.integers(0, len(cs), 60000)] + rng.uniform(-9.0, 9.0, (60000, 3))
    q = tuple(np.ascontiguousarray(q[:, a]) for a in range(3))
    zq = np.zeros(60000, dtype=np.int32)
    want = wo.safety(zq, *q)
    assert (want > 5.0).sum() > 20000
    assert_real_close(vgv.safety(*dev(q)).cpu().numpy(), want, "safety around the empty solids (volume)")
    assert_real_close(wg.safety(torch.from_numpy(zq).cuda(), *dev(q)).cpu().numpy(), want, "safety around the empty solids (world)")


# ------------------------------------------------------------------------------- host-buffer entry points

@pytest.mark.parametrize("n", [1, 4097, 65536, 1048576 + 3, 3 * 1048576 + 11])
def test_host_entry_points_match_the_oracle(vg, n):
    sc = W.shape_cases(1)[0]
    so, sg = O.Shape(sc.kind, sc.params), vg.Shape(sc.kind, sc.params)
    t = sc.tracks(n, band=oracle_band(so))
    ht = [torch.from_numpy(a).pin_memory() for a in t]
    for q in W.QUERIES5:
        g = sg.query_host(q, *ht, step_max=W.STEP_MAX).numpy()
        if q.startswith("distance"):
            assert_real_close(g, getattr(so, q)(*t, W.STEP_MAX), "host %s" % q)
        elif q == "inside":
            assert_int_equal(g, so.inside(*t[:3]), "host inside")
        else:
            assert_real_close(g, getattr(so, q)(*t[:3]), "host %s" % q)
    # the fused host call: one pass of the tracks over the host link for all five answers
    fused = sg.query_all_host(*ht, step_max=W.STEP_MAX)
    for q, g in zip(W.QUERIES5, fused):
        if q.startswith("distance"):
            assert_real_close(g.numpy(), getattr(so, q)(*t, W.STEP_MAX), "host fused %s" % q)
        elif q == "inside":
            assert_int_equal(g.numpy(), so.inside(*t[:3]), "host fused inside")
        else:
            assert_real_close(g.numpy(), getattr(so, q)(*t[:3]), "host fused %s" % q)
    # pageable memory works as well
    g = sg.query_host("distance_to_in", *[torch.from_numpy(a) for a in t], step_max=W.STEP_MAX,
                      out=torch.empty(n, dtype=torch.float64)).numpy()
    assert_real_close(g, so.distance_to_in(*t, W.STEP_MAX), "host pageable")


def test_host_entry_points_with_one_block_baskets(vg):
    """Equally spaced host arrays (rows of one [6][n] allocation, results in one [4][n]) travel as strided 2-D copies: same
    answers as separately allocated arrays; rows of a block with a larger pitch and pageable blocks work as well."""
    sc = W.shape_cases(1)[0]
    so, sg = O.Shape(sc.kind, sc.params), vg.Shape(sc.kind, sc.params)
    for n in (1, 1000, 70001, 1048576 + 3):
        t = sc.tracks(n, band=oracle_band(so))
        for pitch, pin in ((n, True), (n + 13, True), (n, False)):
            blk = torch.empty((6, pitch), dtype=torch.float64)
            blk = blk.pin_memory() if pin else blk
            for i in range(6):
                blk[i, :n].copy_(torch.from_numpy(t[i]))
            rows = [blk[i, :n] for i in range(6)]
            oblk = torch.empty((4, pitch), dtype=torch.float64)
            oblk = oblk.pin_memory() if pin else oblk
            out = [torch.empty(n, dtype=torch.int32)] + [oblk[i, :n] for i in range(4)]
            fused = sg.query_all_host(*rows, step_max=W.STEP_MAX, out=out)
            for q, g in zip(W.QUERIES5, fused):
                if q.startswith("distance"):
                    assert_real_close(g.numpy(), getattr(so, q)(*t, W.STEP_MAX), "block host fused %s" % q)
                elif q == "inside":
                    assert_int_equal(g.numpy(), so.inside(*t[:3]), "block host fused inside")
                else:
                    assert_real_close(g.numpy(), getattr(so, q)(*t[:3]), "block host fused %s" % q)
            g = sg.query_host("safety_to_in", *rows[:3]).numpy()
            assert_real_close(g, so.safety_to_in(*t[:3]), "block host safety")


def test_host_compute_step(vg):
    nav = W.navigator_case()
    vo, vgv = build_volumes(vg, nav)
    t = nav_tracks(nav, vo, 2 * 1048576 + 5, seed=nav.seed + 6)
    so, ho = vo.compute_step(*t, W.STEP_MAX)
    sg, hg = vgv.compute_step_host(*[torch.from_numpy(a).pin_memory() for a in t], step_max=W.STEP_MAX)
    assert_int_equal(hg.numpy(), ho, "host compute_step hit")
    assert_real_close(sg.numpy(), so, "host compute_step step")


def test_library_launch_counter_counts_kernels(vg):
    sg = vg.Shape(W.BOX, [5, 5, 5])
    x = torch.zeros(1000, dtype=torch.float64, device="cuda")
    before = vg.vg_launch_count()
    for _ in range(7):
        sg.safety_to_in(x, x, x)
    assert vg.vg_launch_count() - before == 7


# ------------------------------------------------------------- candidate-grid safeties of the full-phi polycone

def _random_polycone(seed, nz, rmin_hi=5.0):
    rng = np.random.default_rng(seed)
    z = np.sort(rng.uniform(-50.0, 50.0, nz))
    z += np.arange(nz) * 1e-3  # strictly increasing even if two draws coincide
    rmin = rng.uniform(0.0, rmin_hi, nz) if rmin_hi > 0 else np.zeros(nz)
    rmax = rng.uniform(10.0, 30.0, nz)
    out = [0.0, TWO_PI, float(nz)]
    for i in range(nz):
        out += [float(z[i]), float(rmin[i]), float(rmax[i])]
    return out


@pytest.mark.parametrize("wedge", [None, (0.3, 4.0), (-2.0, 1.1), (1.0, math.pi)], ids=["full", "wide", "narrow", "half"])
@pytest.mark.parametrize("seed,nz,rmin_hi", [(1, 2, 5.0), (2, 3, 0.0), (3, 10, 5.0), (4, 17, 9.0), (5, 32, 5.0), (6, 32, 0.0)])
def test_polycone_grid_safeties_match_the_oracle(vg, seed, nz, rmin_hi, wedge):
    """vg_pcon_grid.h: the per-cell candidate masks must hold the nearest segment of every point of the cell.  Points are
    drawn in 3x the bounding box (so some fall off the grid and take the ordered walk inside the same kernel), plus
    points on a lattice that lands exactly on cell corners and edges (rho = i / inv_cr, z = zg0 + j / inv_cz)."""
    par = _random_polycone(seed, nz, rmin_hi)
    if wedge is not None:  # a phi cut: the surface grid plus the face grid (u in [-R, R), every outline edge)
        par[0], par[1] = wedge
    so, sg = O.Shape(W.POLYCONE, par), vg.Shape(W.POLYCONE, par)
    c, h = W.bounding_half(W.POLYCONE, par)
    x, y, z = W.draw_tracks(100 + seed, 300001, c, tuple(3.0 * v for v in h))[:3]
    # cell corners: the grid spans rho in [0, 2.25 rmax), z in [zlo - zl/2, zhi + zl/2) with 64 x 128 cells
    rmax = h[0]
    zl = 2.0 * h[2]
    ii, jj = np.meshgrid(np.arange(65), np.arange(129))
    rho_c = (ii * (2.25 * rmax / 64)).ravel()
    z_c = (c[2] - h[2] - 0.5 * zl + jj * (2.0 * zl / 128)).ravel()
    ang = np.random.default_rng(seed).uniform(0, TWO_PI, rho_c.size)
    x = np.concatenate([x, rho_c * np.cos(ang)])
    y = np.concatenate([y, rho_c * np.sin(ang)])
    z = np.concatenate([z, z_c])
    keep = np.abs(so.sdf(x, y, z)) >= W.SURFACE_BAND
    t = tuple(np.ascontiguousarray(a[keep]) for a in (x, y, z))
    dt = dev(t)
    assert_real_close(sg.safety_to_in(*dt).cpu().numpy(), so.safety_to_in(*t), "grid safety_to_in nz=%d" % nz)
    assert_real_close(sg.safety_to_out(*dt).cpu().numpy(), so.safety_to_out(*t), "grid safety_to_out nz=%d" % nz)
    # the generic kernel (forced direct form) evaluates every segment: same answers
    vg.vg_set_option(vg.OPT_FORM, vg.FORM_DIRECT)
    try:
        g2 = sg.safety_to_in(*dt).cpu().numpy()
    finally:
        vg.vg_set_option(vg.OPT_FORM, vg.FORM_AUTO)
    assert_real_close(g2, so.safety_to_in(*t), "generic safety_to_in nz=%d" % nz)


def test_exercise_all_kernels_script(vg):
    """tests/exercise_all_kernels.py: every kernel once on odd sizes with guard words around the results (the pool has
    no compute-sanitizer), each compared with the oracle."""
    import exercise_all_kernels
    exercise_all_kernels.main()
