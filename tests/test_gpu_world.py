"""GPU parity of the world queries (tree of placed solids; include/vg.h vg_world_*; readings R22-R25) against the
oracle on the same seeded inputs: node indices bit-exact, steps and safeties within max(1e-9, 1e-12 |oracle|)."""
import numpy as np
import pytest
import torch

import oracle as O
import workloads as W
from parity import assert_int_equal, assert_real_close

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vg():
    import paper_1512_06637_b200 as vg
    return vg


def dev(arrs):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs]


@pytest.fixture(scope="module")
def worlds(vg):
    wc = W.world_case()
    so = [O.Shape(k, p) for k, p in zip(wc.kinds, wc.params)]
    sg = [vg.Shape(k, p) for k, p in zip(wc.kinds, wc.params)]
    wo = O.World(so, wc.parents, wc.xforms)
    wg = vg.World(sg, wc.parents, wc.xforms)

    def band(x, y, z):
        nd = wo.locate(x, y, z)
        return (nd < 0) | (wo.safety(nd, x, y, z) < W.SURFACE_BAND)

    return wc, wo, wg, band


@pytest.mark.parametrize("n", [1, 129, 20001, 300007])
def test_locate_step_safety_match_the_oracle(vg, worlds, n):
    wc, wo, wg, band = worlds
    t = wc.tracks(n, band)
    dt = dev(t)
    node_o = wo.locate(*t[:3])
    node_g = wg.locate(*dt[:3])
    assert_int_equal(node_g.cpu().numpy(), node_o, "world locate n=%d" % n)
    for step_max in (W.STEP_MAX, 7.5):
        so, no = wo.step(node_o, *t, step_max)
        sg, ng = wg.step(node_g, *dt, step_max)
        assert_int_equal(ng.cpu().numpy(), no, "world step next n=%d" % n)
        assert_real_close(sg.cpu().numpy(), so, "world step n=%d" % n)
    assert_real_close(wg.safety(node_g, *dt[:3]).cpu().numpy(), wo.safety(node_o, *t[:3]), "world safety n=%d" % n)
    if n > 1000:
        depth = np.where(node_o == 0, 0, np.where(node_o <= 64, 1, 2))
        assert len(set(depth.tolist())) == 3


def test_points_outside_the_world_and_bad_nodes(vg, worlds):
    wc, wo, wg, band = worlds
    x, y, z, dx, dy, dz = W.draw_tracks(77, 50000, (0, 0, 0), (130, 130, 130))
    keep = np.abs(wo.shapes[0].sdf(x, y, z)) > 1e-6
    t = [a[keep] for a in (x, y, z, dx, dy, dz)]
    node_o = wo.locate(*t[:3])
    # keep clear of every surface below the root as well
    ok = (node_o < 0) | (wo.safety(np.maximum(node_o, 0), *t[:3]) >= W.SURFACE_BAND)
    t = [np.ascontiguousarray(a[ok]) for a in t]
    node_o = node_o[ok]
    assert (node_o < 0).any() and (node_o >= 0).any()
    dt = dev(t)
    node_g = wg.locate(*dt[:3])
    assert_int_equal(node_g.cpu().numpy(), node_o, "locate incl. outside")
    so, no = wo.step(node_o, *t)
    sg, ng = wg.step(node_g, *dt)
    assert_int_equal(ng.cpu().numpy(), no, "step next incl. outside")
    assert_real_close(sg.cpu().numpy(), so, "step incl. outside")
    bad = torch.full_like(node_g, 100000)
    sg, ng = wg.step(bad, *dt)
    assert bool((sg == -1).all()) and bool((ng == -1).all())
    assert bool((wg.safety(bad, *dt[:3]) == -1).all())


# The walk through the world (step, move onto the border, take `next` as the new node) lives in tests/test_gpu_surface.py
# now: it is exact (no nudge beyond the border), in lockstep with the oracle and on the GPU alone (reading R32).


def test_world_create_rejects_bad_input(vg):
    b = vg.Shape(W.BOX, [1, 1, 1])
    ident = [1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]
    with pytest.raises(vg.VgError):
        vg.World([b, b], [0, 0], [ident, ident])
    with pytest.raises(vg.VgError):
        vg.World([b, b], [-1, 1], [ident, ident])
    with pytest.raises(vg.VgError):
        vg.World([b, b], [-1, 0], [ident, [2, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]])
    w = vg.World([b], [-1], [ident])
    x = torch.zeros(5, dtype=torch.float64, device="cuda")
    assert w.locate(x, x, x).tolist() == [0] * 5


def test_full_size_as_benchmarked_every_track(vg, worlds):
    """4,194,304 tracks (the size and launch configuration bench.py times); the oracle checks every track."""
    wc, wo, wg, band = worlds
    t = wc.tracks(4194304, band)
    dt = dev(t)
    node_g = wg.locate(*dt[:3])
    step_g, next_g = wg.step(node_g, *dt, W.STEP_MAX)
    safe_g = wg.safety(node_g, *dt[:3])
    sel = np.arange(4194304)
    ts = [np.ascontiguousarray(a[sel]) for a in t]
    node_o = wo.locate(*ts[:3])
    assert_int_equal(node_g.cpu().numpy()[sel], node_o, "full-size locate")
    so, no = wo.step(node_o, *ts, W.STEP_MAX)
    assert_int_equal(next_g.cpu().numpy()[sel], no, "full-size next")
    assert_real_close(step_g.cpu().numpy()[sel], so, "full-size step")
    assert_real_close(safe_g.cpu().numpy()[sel], wo.safety(node_o, *ts[:3]), "full-size safety")
    # a property that holds for every track: the safety never exceeds the step
    assert bool((safe_g <= step_g * (1 + 1e-12)).all())


# ------------------------------------------------- nodes that are polycones and booleans (reading R30)

def _build_mixed(mod, mc):
    def mk(nd):
        if nd[0] == "shape":
            return mod.Shape(nd[1], nd[2])
        b = nd[1]
        return mod.Boolean(b.op, mod.Shape(b.kind_a, b.par_a), mod.Shape(b.kind_b, b.par_b), b.xform)
    objs = [mk(nd) for nd in mc.nodes]
    return objs, mod.World(objs, mc.parents, mc.xforms)


@pytest.fixture(scope="module")
def mixed_worlds(vg):
    mc = W.mixed_world_case()
    objs_o, wo = _build_mixed(O, mc)
    objs_g, wg = _build_mixed(vg, mc)
    # clear of every surface of every node AND of every boolean operand (the state machine's contract, R7)
    G = np.zeros((len(mc.nodes), 4, 4))
    for i in range(len(mc.nodes)):
        X = np.eye(4)
        X[:3, :] = mc.xforms[i].reshape(3, 4)
        G[i] = X if mc.parents[i] < 0 else X @ G[mc.parents[i]]

    def band(x, y, z):
        nd = wo.locate(x, y, z)
        bad = (nd < 0) | (wo.safety(np.maximum(nd, 0), x, y, z) < W.SURFACE_BAND)
        P = np.stack([x, y, z, np.ones_like(x)])
        for i, o in enumerate(objs_o):
            if isinstance(o, O.Boolean):
                L = G[i] @ P
                B = np.asarray(o.xform).reshape(3, 4)
                LB = B[:, :3] @ L[:3] + B[:, 3:4]
                bad |= (np.abs(o.a.sdf(L[0], L[1], L[2])) < W.SURFACE_BAND) | (np.abs(o.b.sdf(LB[0], LB[1], LB[2])) < W.SURFACE_BAND)
        return bad

    return mc, wo, wg, band


@pytest.mark.parametrize("n", [1, 4099, 400003])
def test_mixed_world_matches_the_oracle(vg, mixed_worlds, n):
    mc, wo, wg, band = mixed_worlds
    t = mc.tracks(n, band)
    dt = dev(t)
    node_o = wo.locate(*t[:3])
    node_g = wg.locate(*dt[:3])
    assert_int_equal(node_g.cpu().numpy(), node_o, "mixed world locate n=%d" % n)
    for step_max in (W.STEP_MAX, 9.0):
        so, no = wo.step(node_o, *t, step_max)
        sg, ng = wg.step(node_g, *dt, step_max)
        assert_int_equal(ng.cpu().numpy(), no, "mixed world next n=%d" % n)
        assert_real_close(sg.cpu().numpy(), so, "mixed world step n=%d" % n)
    assert_real_close(wg.safety(node_g, *dt[:3]).cpu().numpy(), wo.safety(node_o, *t[:3]), "mixed world safety n=%d" % n)
    if n > 100000:
        counts = np.bincount(node_o, minlength=13)
        assert np.all(counts[:9] > 1000) and counts[9:].sum() > 50


# ------------------------------------------------------------------------------------- random trees (soak)

def _random_tree(rng):
    """Root box (100) > k1 children of random kinds, sizes and rotations (they may overlap: Locate takes the first in index
    order, Step and Safety are minima) > for some box / orb children, k2 grand-children inside them."""
    TWO_PI = 2 * np.pi
    H = 100.0

    def solid(size):
        kind = [W.BOX, W.ORB, W.TUBE, W.CONE, W.TRD, W.POLYCONE][rng.integers(0, 6)]
        a, b, c = size * rng.uniform(0.4, 1.0, 3)
        par = {W.BOX: [a, b, c], W.ORB: [a], W.TUBE: [0.3 * a, a, b, 0.5, 4.0],
               W.CONE: [0.2 * a, a, 0.3 * b, 1.2 * b, c, 0.0, TWO_PI], W.TRD: [a, 0.5 * a, b, 1.3 * b, c],
               W.POLYCONE: [0.0, TWO_PI, 4.0, -c, 0.0, 0.5 * a, -0.3 * c, 0.2 * a, a, 0.3 * c, 0.2 * a, 0.6 * a, c, 0.0, 0.4 * a]}[kind]
        return kind, [float(v) for v in par]

    def place(spread):
        q = rng.normal(size=4)
        return W.placement(W.quaternion_to_matrix(tuple(q / np.linalg.norm(q))), rng.uniform(-spread, spread, 3))
    kinds, pars, parents, xf = [W.BOX], [[H, H, H]], [-1], [W.placement(np.eye(3), (0, 0, 0))]
    k1 = int(rng.choice([3, 11, 12, 13, 30, 64, 70]))
    size = H * float(rng.choice([0.06, 0.12, 0.2]))
    for _ in range(k1):
        k, p = solid(size)
        kinds.append(k), pars.append(p), parents.append(0), xf.append(place(H - 1.8 * size))
    for i in range(1, k1 + 1):
        if kinds[i] in (W.BOX, W.ORB) and rng.random() < 0.5:
            inner = min(pars[i])
            for _ in range(int(rng.choice([1, 2, 12, 20]))):
                k, p = solid(0.22 * inner)
                kinds.append(k), pars.append(p), parents.append(i), xf.append(place(0.45 * inner))
    return kinds, pars, parents, np.stack(xf)


def test_random_trees_soak(vg):
    """VG_STRESS_REPS seeded random trees (default 8): Locate of points anywhere, Step and Safety in the located nodes and
    in the root, against the oracle.  Nodes with 12..64 children take the candidate and safety grids, the others the
    sphere loops."""
    import os
    for rep in range(int(os.environ.get("VG_STRESS_REPS", "8"))):
        rng = np.random.default_rng(7000 + rep)
        kinds, pars, parents, xf = _random_tree(rng)
        nn = len(kinds)
        wo = O.World([O.Shape(k, p) for k, p in zip(kinds, pars)], parents, xf)
        wg = vg.World([vg.Shape(k, p) for k, p in zip(kinds, pars)], parents, xf)

        def band(x, y, z):  # clear of the surface of EVERY node (children overlap: a point may be near a sibling's surface)
            bad = wo.locate(x, y, z) < 0
            for nd in range(nn):
                bad |= np.abs(wo.safety(np.full(x.size, nd, dtype=np.int32), x, y, z)) < 1e-6
            return bad
        t = W.draw_tracks(7100 + rep, 20011, (0, 0, 0), (100, 100, 100), band)
        dt = dev(t)
        what = "random tree %d (%d nodes, %d under the root)" % (rep, nn, parents.count(0))
        node_o = wo.locate(*t[:3])
        node_g = wg.locate(*dt[:3])
        assert_int_equal(node_g.cpu().numpy(), node_o, what + " locate")
        for nodes in (node_o, np.zeros_like(node_o)):
            ng_in = torch.from_numpy(nodes).cuda()
            for step_max in (W.STEP_MAX, 12.0):
                so, no = wo.step(nodes, *t, step_max)
                sg, ng = wg.step(ng_in, *dt, step_max)
                assert_int_equal(ng.cpu().numpy(), no, what + " next")
                assert_real_close(sg.cpu().numpy(), so, what + " step")
            assert_real_close(wg.safety(ng_in, *dt[:3]).cpu().numpy(), wo.safety(nodes, *t[:3]), what + " safety")
