"""Pins of the oracle's world queries (tree of placed solids; readings R22-R25 in oracle/vg_oracle.c and DESIGN.md;
PAPER.md:104 "hierarchical connections", "transported to the border").

Nothing here re-calls the world functions to check themselves: every expectation is composed in numpy from the
per-solid oracle functions (pinned in test_oracle_pins.py) and the one-level ComputeStep (pinned in test_oracle_nav.py).
"""
import numpy as np
import pytest

import oracle as O
import workloads as W


@pytest.fixture(scope="module")
def world():
    wc = W.world_case()
    shapes = [O.Shape(k, p) for k, p in zip(wc.kinds, wc.params)]
    w = O.World(shapes, wc.parents, wc.xforms)

    def band(x, y, z):
        nd = w.locate(x, y, z)
        return (nd < 0) | (w.safety(nd, x, y, z) < W.SURFACE_BAND)

    t = wc.tracks(60000, band)
    return wc, shapes, w, t


def global_transforms(wc):
    """4x4 world -> local matrices, composed in numpy (independent of the oracle's one-at-a-time chain)."""
    nn = len(wc.kinds)
    G = np.zeros((nn, 4, 4))
    for i in range(nn):
        X = np.eye(4)
        X[:3, :] = wc.xforms[i].reshape(3, 4)
        G[i] = X if wc.parents[i] < 0 else X @ G[wc.parents[i]]
    return G


def to_node(G, i, x, y, z):
    P = np.stack([x, y, z, np.ones_like(x)])
    L = G[i] @ P
    return L[0], L[1], L[2]


def dir_to_node(G, i, dx, dy, dz):
    L = G[i][:3, :3] @ np.stack([dx, dy, dz])
    return L[0], L[1], L[2]


def test_world_layout(world):
    wc, shapes, w, t = world
    assert len(wc.kinds) == 193 and wc.parents[0] == -1
    assert np.all(wc.parents[1:65] == 0) and np.all(wc.parents[65:] >= 1) and np.all(wc.parents[65:] <= 64)
    assert np.all(wc.parents[1:] < np.arange(1, 193))
    R = wc.xforms.reshape(-1, 3, 4)[:, :, :3]
    assert np.max(np.abs(R @ np.transpose(R, (0, 2, 1)) - np.eye(3))) < 1e-14
    assert {W.BOX, W.ORB, W.TUBE, W.CONE, W.TRD} == set(wc.kinds)


def test_locate_is_the_deepest_node_that_holds_the_point(world):
    """Brute force over all nodes: a node holds p iff p is inside its solid and inside every ancestor's; siblings do
    not overlap, so exactly one chain holds p and Locate is its deepest member."""
    wc, shapes, w, t = world
    x, y, z = t[:3]
    G = global_transforms(wc)
    nn = len(shapes)
    own = np.zeros((nn, x.size), dtype=bool)
    for i in range(nn):
        own[i] = shapes[i].inside(*to_node(G, i, x, y, z)) == O.INSIDE
    held = own.copy()
    for i in range(1, nn):  # parents come first
        held[i] &= held[wc.parents[i]]
    depth = np.zeros(nn, dtype=int)
    for i in range(1, nn):
        depth[i] = depth[wc.parents[i]] + 1
    assert held.sum(axis=0).max() <= 3 and np.all(held[0])
    # exactly one node per depth at most (no overlapping siblings)
    for dlev in (1, 2):
        assert held[depth == dlev].sum(axis=0).max() <= 1
    expect = np.array([np.flatnonzero(held[:, j])[-1] for j in range(x.size)])  # deepest = highest index on the chain
    expect_depth = depth[expect]
    assert np.array_equal(held.sum(axis=0) - 1, expect_depth)
    got = w.locate(x, y, z)
    assert np.array_equal(got, expect)
    frac = np.bincount(depth[got], minlength=3) / x.size
    assert frac[0] > 0.4 and frac[1] > 0.3 and frac[2] > 0.005
    # outside the world
    assert np.array_equal(w.locate([150.0, 0.0], [0.0, 0.0], [0.0, 101.0]), [-1, -1])


def test_step_is_the_one_level_step_of_the_node(world):
    """World step == ComputeStep of a Volume built from the node and its children, on coordinates transformed in numpy."""
    wc, shapes, w, t = world
    x, y, z, dx, dy, dz = t
    G = global_transforms(wc)
    node = w.locate(x, y, z)
    step, nxt = w.step(node, x, y, z, dx, dy, dz)
    checked = 0
    for nd in [0, 1, 2, 17, 40, 64, 65, 66, 130, 192]:
        sel = np.flatnonzero(node == nd)
        if sel.size == 0:
            continue
        kids = np.flatnonzero(wc.parents == nd)
        vol = O.Volume(shapes[nd], [shapes[c] for c in kids], wc.xforms[kids] if kids.size else np.zeros((0, 12)))
        lx, ly, lz = to_node(G, nd, x[sel], y[sel], z[sel])
        ldx, ldy, ldz = dir_to_node(G, nd, dx[sel], dy[sel], dz[sel])
        s1, hit = vol.compute_step(lx, ly, lz, ldx, ldy, ldz)
        want_next = np.where(hit < 0, wc.parents[nd], kids[np.maximum(hit, 0)] if kids.size else wc.parents[nd])
        assert np.array_equal(nxt[sel], want_next), nd
        assert np.max(np.abs(step[sel] - s1)) < 1e-10, nd
        checked += sel.size
    assert checked > 0.5 * x.size
    # the root: exit leaves the world
    root = node == 0
    assert set(np.unique(nxt[root])) <= set(range(-1, 65)) and (nxt[root] == -1).any() and (nxt[root] > 0).any()


def test_step_lands_on_the_border_between_node_and_next(world):
    """Marching through Locate: just before the step the track is still in `node`, just after it is in `next`
    (the particle is transported to the border and changes volume)."""
    wc, shapes, w, t = world
    x, y, z, dx, dy, dz = t
    node = w.locate(x, y, z)
    step, nxt = w.step(node, x, y, z, dx, dy, dz)
    assert np.all(step > 0) and np.all(np.isfinite(step))
    eps = 1e-6
    ok = step > 2 * eps
    before = w.locate(x + (step - eps) * dx, y + (step - eps) * dy, z + (step - eps) * dz)
    after = w.locate(x + (step + eps) * dx, y + (step + eps) * dy, z + (step + eps) * dz)
    # grazing hits (within eps of an edge) may skip a volume: allow a handful
    assert (before[ok] != node[ok]).mean() < 1e-3
    assert (after[ok] != nxt[ok]).mean() < 1e-3
    # halfway there nothing has changed either
    mid = w.locate(x + 0.5 * step * dx, y + 0.5 * step * dy, z + 0.5 * step * dz)
    assert np.array_equal(mid, node)


def test_physics_step_and_bad_nodes(world):
    wc, shapes, w, t = world
    x, y, z, dx, dy, dz = (a[:5000] for a in t)
    node = w.locate(x, y, z)
    s_inf, n_inf = w.step(node, x, y, z, dx, dy, dz)
    s, n = w.step(node, x, y, z, dx, dy, dz, step_max=5.0)
    lim = s_inf > 5.0
    assert lim.any() and (~lim).any()
    assert np.all(s[lim] == 5.0) and np.array_equal(n[lim], node[lim])
    assert np.array_equal(s[~lim], s_inf[~lim]) and np.array_equal(n[~lim], n_inf[~lim])
    s, n = w.step(np.full(10, -1, dtype=np.int32), x[:10], y[:10], z[:10], dx[:10], dy[:10], dz[:10])
    assert np.all(s == -1) and np.all(n == -1)


def test_world_safety_is_the_distance_to_the_nearest_surface_of_any_node(world):
    """R25 in the located node == min over ALL nodes of |sdf| (surfaces of other nodes are farther than the node's own)."""
    wc, shapes, w, t = world
    x, y, z = (a[:20000] for a in t[:3])
    G = global_transforms(wc)
    node = w.locate(x, y, z)
    got = w.safety(node, x, y, z)
    brute = np.full(x.size, np.inf)
    for i in range(len(shapes)):
        brute = np.minimum(brute, np.abs(shapes[i].sdf(*to_node(G, i, x, y, z))))
    assert np.max(np.abs(got - brute)) < 1e-10
    assert np.all(got >= W.SURFACE_BAND)


def test_rigid_motion_of_the_whole_world(world):
    """Moving the root placement and the tracks by the same rigid motion changes nothing."""
    wc, shapes, w, t = world
    x, y, z, dx, dy, dz = (a[:20000] for a in t)
    Q = W.quaternion_to_matrix((0.5, -0.5, 0.5, 0.5))
    c = np.array([3.0, -7.0, 11.0])
    P = Q @ np.stack([x, y, z]) + c[:, None]  # moved points
    D = Q @ np.stack([dx, dy, dz])
    xf = wc.xforms.copy()
    xf[0] = W.placement(Q, c)  # world -> root local undoes the motion
    w2 = O.World(shapes, wc.parents, xf)
    n1 = w.locate(x, y, z)
    n2 = w2.locate(P[0], P[1], P[2])
    assert np.array_equal(n1, n2)
    s1, k1 = w.step(n1, x, y, z, dx, dy, dz)
    s2, k2 = w2.step(n2, P[0], P[1], P[2], D[0], D[1], D[2])
    assert np.array_equal(k1, k2) and np.max(np.abs(s1 - s2)) < 1e-10


def test_world_create_rejects_bad_trees():
    b = O.Shape(O.BOX, [1, 1, 1])
    ident = [1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]
    with pytest.raises(ValueError):
        O.World([b, b], [0, 0], [ident, ident])  # root must have parent -1
    with pytest.raises(ValueError):
        O.World([b, b], [-1, 1], [ident, ident])  # parent must come first


# ------------------------------------------------- nodes that are polycones and booleans (reading R30)

def build_mixed(mc, mod=O):
    def mk(nd):
        if nd[0] == "shape":
            return mod.Shape(nd[1], nd[2])
        b = nd[1]
        return mod.Boolean(b.op, mod.Shape(b.kind_a, b.par_a), mod.Shape(b.kind_b, b.par_b), b.xform)
    objs = [mk(nd) for nd in mc.nodes]
    return objs, mod.World(objs, mc.parents, mc.xforms)


@pytest.fixture(scope="module")
def mixed():
    mc = W.mixed_world_case()
    objs, w = build_mixed(mc)

    def band(x, y, z):
        nd = w.locate(x, y, z)
        return (nd < 0) | (w.safety(nd, x, y, z) < W.SURFACE_BAND)

    return mc, objs, w, mc.tracks(60000, band)


def test_mixed_world_locate_is_the_deepest_holder(mixed):
    mc, objs, w, t = mixed
    x, y, z = t[:3]
    nn = len(objs)
    G = np.zeros((nn, 4, 4))
    for i in range(nn):
        X = np.eye(4)
        X[:3, :] = mc.xforms[i].reshape(3, 4)
        G[i] = X if mc.parents[i] < 0 else X @ G[mc.parents[i]]
    held = np.zeros((nn, x.size), dtype=bool)
    for i in range(nn):
        held[i] = objs[i].inside(*to_node(G, i, x, y, z)) == O.INSIDE
        if i > 0:
            held[i] &= held[mc.parents[i]]
    expect = np.array([np.flatnonzero(held[:, j])[-1] for j in range(x.size)])
    got = w.locate(x, y, z)
    assert np.array_equal(got, expect)
    counts = np.bincount(got, minlength=nn)
    assert np.all(counts[1:9] > 100) and counts[9:].sum() > 5


def test_mixed_world_step_and_safety_properties(mixed):
    mc, objs, w, t = mixed
    x, y, z, dx, dy, dz = t
    node = w.locate(x, y, z)
    step, nxt = w.step(node, x, y, z, dx, dy, dz)
    assert np.all(step > 0) and np.all(np.isfinite(step))
    eps = 1e-6
    ok = step > 2 * eps
    before = w.locate(x + (step - eps) * dx, y + (step - eps) * dy, z + (step - eps) * dz)
    after = w.locate(x + (step + eps) * dx, y + (step + eps) * dy, z + (step + eps) * dz)
    assert (before[ok] != node[ok]).mean() < 2e-3 and (after[ok] != nxt[ok]).mean() < 2e-3
    for frac in (0.1, 0.5, 0.9):
        mid = w.locate(x + frac * step * dx, y + frac * step * dy, z + frac * step * dz)
        assert (mid != node).mean() < 1e-3
    # safety: never beyond the step, and the ball of that radius stays in the node (probe 60 directions per point)
    s = w.safety(node, x, y, z)
    assert np.all(s >= W.SURFACE_BAND) and np.all(s <= step * (1 + 1e-12))
    rng = np.random.default_rng(8)
    sel = rng.choice(x.size, 3000, replace=False)
    for _ in range(60):
        v = rng.normal(size=3)
        v /= np.linalg.norm(v)
        r = s[sel] * (1 - 1e-9)
        assert np.array_equal(w.locate(x[sel] + r * v[0], y[sel] + r * v[1], z[sel] + r * v[2]), node[sel])
    # and no direction reaches a border sooner than the safety; in nodes without booleans (polycones, the orbs inside
    # them) the safety is exact, so the nearest border over 4000 directions comes close to it for most points
    idx = np.flatnonzero(np.isin(node, [1, 3, 5, 7, 9, 11]))[:200]
    v = rng.normal(size=(3, 4000))
    v /= np.linalg.norm(v, axis=0)
    ratio = []
    for j in idx:
        tt, _ = w.step(np.full(4000, node[j], dtype=np.int32), np.full(4000, x[j]), np.full(4000, y[j]), np.full(4000, z[j]), v[0], v[1], v[2])
        assert s[j] <= tt.min() * (1 + 1e-12)
        ratio.append(tt.min() / s[j])
    assert np.median(ratio) < 1.02
