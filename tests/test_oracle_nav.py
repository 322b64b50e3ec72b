"""Pins of the oracle's navigation step (ComputeStep)
and of the seeded workloads (BASELINE.json configs)."""
import math

import numpy as np
import pytest

import geomdefs as G
import oracle as O
import workloads as W


def build_volume(nav, order=None, xforms=None):
    mother = O.Shape(nav.mother_kind, nav.mother_params)
    idx = list(range(len(nav.daughter_kinds))) if order is None else list(order)
    ds = [O.Shape(nav.daughter_kinds[i], nav.daughter_params[i]) for i in idx]
    xf = (nav.xforms if xforms is None else xforms)[idx]
    return O.Volume(mother, ds, xf)


def nav_tracks(nav, vol, n, seed=None):
    band = lambda x, y, z: vol.safety(x, y, z) < W.SURFACE_BAND
    return W.draw_tracks(nav.seed if seed is None else seed, n, nav.center, nav.half, band)


def test_transforms_are_rigid_and_layout_matches_reading():
    nav = W.navigator_case()
    assert nav.xforms.shape == (64, 12)
    M = nav.xforms.reshape(64, 3, 4)
    R, b = M[:, :, :3], M[:, :, 3]
    assert np.max(np.abs(R @ np.transpose(R, (0, 2, 1)) - np.eye(3))) < 1e-15
    assert np.allclose(np.linalg.det(R), 1.0, atol=1e-14)
    # R c + b = 0: the daughter's centre maps to its local origin (R12)
    assert np.max(np.abs(np.einsum("nij,nj->ni", R, nav.centers) + b)) < 1e-12
    assert sorted(set(nav.centers[:, 0])) == [-75.0, -25.0, 25.0, 75.0]
    assert nav.daughter_kinds.count(W.BOX) == 32 and nav.daughter_kinds.count(W.TUBE) == 32
    assert nav.daughter_kinds[0] == W.BOX and nav.daughter_kinds[1] == W.TUBE and nav.daughter_kinds[5] == W.BOX
    # rotations differ between daughters and are not the identity
    assert np.linalg.norm(R[0] - np.eye(3)) > 0.1 and np.linalg.norm(R[0] - R[1]) > 0.1


def test_single_daughter_identity_is_min_of_the_two_distances():
    mother = O.Shape(O.BOX, [100, 100, 100])
    d = O.Shape(O.TUBE, [0, 8, 8, 0, 2 * math.pi])
    ident = np.array([[1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]], dtype=np.float64)
    vol = O.Volume(mother, [d], ident)
    x, y, z, dx, dy, dz = W.draw_tracks(3, 20000, (0, 0, 0), (30, 30, 30), lambda x, y, z: vol.safety(x, y, z) < 1e-6)
    step, hit = vol.compute_step(x, y, z, dx, dy, dz)
    tout = mother.distance_to_out(x, y, z, dx, dy, dz)
    tin = d.distance_to_in(x, y, z, dx, dy, dz)
    assert np.array_equal(step, np.minimum(tout, tin))
    assert np.array_equal(hit, np.where(tin < tout, 0, -1))
    assert 0.02 < (hit == 0).mean() < 0.5


def test_config4_statistics_and_physics_step():
    nav = W.navigator_case()
    vol = build_volume(nav)
    x, y, z, dx, dy, dz = nav_tracks(nav, vol, 50000)
    assert np.all(vol.safety(x, y, z) >= W.SURFACE_BAND)
    step, hit = vol.compute_step(x, y, z, dx, dy, dz, W.STEP_MAX)
    assert np.all(step > 0) and np.all(np.isfinite(step)) and hit.min() == -1 and hit.max() == 63
    # about 22 % of the tracks hit a daughter, mean step about 72
    assert 0.19 < (hit >= 0).mean() < 0.25
    assert 65 < step.mean() < 80
    # the physics step wins: (stepMax, -2)
    s2, h2 = vol.compute_step(x, y, z, dx, dy, dz, 40.0)
    assert np.array_equal(s2, np.where(step > 40.0, 40.0, step))
    assert np.array_equal(h2, np.where(step > 40.0, -2, hit))
    # safety <= step
    assert np.all(vol.safety(x, y, z) <= step * (1 + 1e-12))


def test_permuting_daughters_permutes_hit():
    nav = W.navigator_case()
    vol = build_volume(nav)
    perm = np.random.default_rng(5).permutation(64)
    volp = build_volume(nav, order=perm)
    t = nav_tracks(nav, vol, 20000)
    s0, h0 = vol.compute_step(*t)
    s1, h1 = volp.compute_step(*t)
    assert np.array_equal(s0, s1)
    assert np.array_equal(np.where(h1 >= 0, perm[np.maximum(h1, 0)], h1), h0)


def test_rigid_motion_invariance():
    """Moving every daughter and every track by the same rigid motion (inside a large mother orb, which is
    itself invariant under rotation) leaves step and hit unchanged.  Catches R vs R^T and the sign of b."""
    nav = W.navigator_case()
    mother = O.Shape(O.ORB, [400.0])
    ds = [O.Shape(k, p) for k, p in zip(nav.daughter_kinds, nav.daughter_params)]
    vol = O.Volume(mother, ds, nav.xforms)
    x, y, z, dx, dy, dz = nav_tracks(nav, vol, 20000, seed=8)
    s0, h0 = vol.compute_step(x, y, z, dx, dy, dz)
    G_rot = G.random_rotation(np.random.default_rng(6))
    # p' = G p  =>  local = R p + b = (R G^T) p' + b
    M = nav.xforms.reshape(64, 3, 4).copy()
    M[:, :, :3] = M[:, :, :3] @ G_rot.T
    vol2 = O.Volume(mother, ds, M.reshape(64, 12))
    P = G_rot @ np.stack([x, y, z])
    D = G_rot @ np.stack([dx, dy, dz])
    s1, h1 = vol2.compute_step(P[0], P[1], P[2], D[0], D[1], D[2])
    assert np.array_equal(h0, h1)
    assert np.max(np.abs(s0 - s1)) < 1e-10
    assert 0.05 < (h0 >= 0).mean()


def test_compute_step_brute_force_marching():
    """Independent numpy membership of the mother and of every daughter (own transform code) marched along
    the ray: first parameter at which the track leaves the mother or enters any daughter."""
    nav = W.navigator_case()
    vol = build_volume(nav)
    x, y, z, dx, dy, dz = nav_tracks(nav, vol, 40, seed=12)
    step, hit = vol.compute_step(x, y, z, dx, dy, dz)
    M = nav.xforms.reshape(64, 3, 4)
    for i in range(x.size):
        t = np.arange(0.0, 360.0, 2e-3)
        P = np.stack([x[i] + t * dx[i], y[i] + t * dy[i], z[i] + t * dz[i]])
        first, who = np.inf, -1
        out = ~G.member(G.BOX, nav.mother_params, P[0], P[1], P[2])
        if out.any():
            first = t[np.argmax(out)]
        for k in range(64):
            L = M[k, :, :3] @ P + M[k, :, 3:4]
            m = G.member(nav.daughter_kinds[k], nav.daughter_params[k], L[0], L[1], L[2])
            if m.any() and t[np.argmax(m)] < first:
                first, who = t[np.argmax(m)], k
        if who != hit[i]:
            # a clipped corner shorter than the marching step can be stepped over: then the oracle's hit
            # must be real (the point just past its step lies in that daughter)
            assert hit[i] >= 0 and step[i] < first
            q = np.array([x[i], y[i], z[i]]) + (step[i] + 1e-7) * np.array([dx[i], dy[i], dz[i]])
            L = M[hit[i], :, :3] @ q + M[hit[i], :, 3]
            assert G.member(nav.daughter_kinds[hit[i]], nav.daughter_params[hit[i]], *L)
        else:
            assert abs(first - step[i]) < 2.1e-3


def test_volume_safety_definition_and_sphere_tracing():
    nav = W.navigator_case()
    vol = build_volume(nav)
    x, y, z, dx, dy, dz = nav_tracks(nav, vol, 3000, seed=14)
    M = nav.xforms.reshape(64, 3, 4)
    P = np.stack([x, y, z])
    want = vol.mother.safety_to_out(x, y, z)
    for k in range(64):
        L = M[k, :, :3] @ P + M[k, :, 3:4]
        want = np.minimum(want, vol.daughters[k].safety_to_in(L[0], L[1], L[2]))
    assert np.max(np.abs(vol.safety(x, y, z) - want)) < 1e-12
    # sphere tracing on the volume safety reaches the navigation step (independent chain: sdf -> step)
    step, _ = vol.compute_step(x, y, z, dx, dy, dz)
    t = np.zeros_like(x)
    for _ in range(3000):
        d = vol.safety(x + t * dx, y + t * dy, z + t * dz)
        live = (d > 1e-12) & (t < 400)
        if not live.any():
            break
        t = np.where(live, t + d, t)
    ok = np.abs(t - step) < 1e-8
    assert ok.mean() > 0.995


def test_fp64_nav_agrees_with_80bit_build():
    nav = W.navigator_case()
    vol = build_volume(nav)
    t = nav_tracks(nav, vol, 50000, seed=15)
    m = O.Shape(nav.mother_kind, nav.mother_params, long_double=True)
    ds = [O.Shape(k, p, long_double=True) for k, p in zip(nav.daughter_kinds, nav.daughter_params)]
    vl = O.Volume(m, ds, nav.xforms)
    s0, h0 = vol.compute_step(*t)
    s1, h1 = vl.compute_step(*t)
    assert np.array_equal(h0, h1)
    assert np.max(np.abs(s0 - s1)) < 1e-11


# ------------------------------------------------------------------ workloads

def test_generators_are_deterministic_and_isotropic():
    a = W.draw_tracks(123, 100000, (1, 2, 3), (4, 5, 6))
    b = W.draw_tracks(123, 100000, (1, 2, 3), (4, 5, 6))
    c = W.draw_tracks(124, 100000, (1, 2, 3), (4, 5, 6))
    assert all(np.array_equal(u, v) for u, v in zip(a, b))
    assert not np.array_equal(a[0], c[0])
    x, y, z, dx, dy, dz = a
    assert x.min() >= -3 and x.max() <= 5 and z.min() >= -3 and z.max() <= 9
    assert np.max(np.abs(dx * dx + dy * dy + dz * dz - 1)) < 7e-16
    assert abs(dx.mean()) < 0.01 and abs(dy.mean()) < 0.01 and abs(dz.mean()) < 0.01
    assert abs((dz * dz).mean() - 1 / 3) < 0.01 and abs((dx * dy).mean()) < 0.01
    # a prefix of a longer draw is NOT required to equal a shorter draw; same (seed, n) is the contract
    assert all(u.dtype == np.float64 and u.flags.c_contiguous for u in a)


def test_rejection_redraws_only_flagged_points():
    band = lambda x, y, z: np.abs(x) < 0.5
    a = W.draw_tracks(7, 50000, (0, 0, 0), (2, 2, 2))
    b = W.draw_tracks(7, 50000, (0, 0, 0), (2, 2, 2), band)
    keep = np.abs(a[0]) >= 0.5
    assert np.all(np.abs(b[0]) >= 0.5)
    assert np.array_equal(a[0][keep], b[0][keep]) and np.array_equal(a[3], b[3])
    assert (~keep).mean() > 0.2


@pytest.mark.parametrize("k,idx,frac", [(0, 0, 0.125), (1, 0, 0.1164), (2, 0, 0.1207), (2, 1, 0.1517), (3, 1, 0.1551)])
def test_config_inside_fractions_match_analytic_volumes(k, idx, frac):
    """Volume of the solid / volume of the sampling box."""
    case = W.shape_cases(k)[idx]
    s = O.Shape(case.kind, case.params)
    x, y, z, *_ = case.tracks(200000, lambda x, y, z: np.abs(s.sdf(x, y, z)) < W.SURFACE_BAND)
    got = (s.inside(x, y, z) == O.INSIDE).mean()
    assert abs(got - frac) < 0.004, (got, frac)


def test_config_shapes_are_as_baseline_json_states():
    assert W.shape_cases(0)[0].params == [5.0, 5.0, 5.0] and W.shape_cases(0)[0].sizes == (65536,)
    t = W.shape_cases(1)[0]
    assert t.params == [5.0, 10.0, 15.0, 0.0, 4 * math.pi / 3] and t.half == (15.0, 15.0, 22.5) and t.sizes == (1048576,)
    c, d = W.shape_cases(2)
    assert c.half == (18.0, 18.0, 30.0) and d.half == (15.0, 10.5, 22.5) and c.sizes == d.sizes == (4194304,)
    p, o = W.shape_cases(3)
    assert p.sizes == (2 ** 10, 2 ** 14, 2 ** 18, 2 ** 22, 2 ** 24) and o.params == [20.0] and o.half == (30.0, 30.0, 30.0)
    par = p.params
    assert par[2] == 10 and len(par) == 33
    zs, rmin, rmax = par[3::3], par[4::3], par[5::3]
    assert all(b > a for a, b in zip(zs, zs[1:])) and -50 <= zs[0] and zs[-1] <= 50
    assert all(0 <= r <= 5 for r in rmin) and all(10 <= r <= 30 for r in rmax)
    assert p.queries == ("distance_to_in", "safety_to_in")


def test_ties_go_to_the_lowest_index_mother_first():
    """Reading R13: sequential strict '<' from the mother exit.  Exact ties are built from duplicates."""
    mother = O.Shape(O.BOX, [20, 20, 20])
    d = O.Shape(O.BOX, [5, 5, 5])
    ident = [1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]
    vol = O.Volume(mother, [d, d, d], np.array([ident, ident, ident], dtype=np.float64))
    x, y, z, dx, dy, dz = W.draw_tracks(4, 5000, (0, 0, 0), (20, 20, 20), lambda x, y, z: vol.safety(x, y, z) < 1e-6)
    step, hit = vol.compute_step(x, y, z, dx, dy, dz)
    assert set(np.unique(hit)) == {-1, 0}
    # a daughter that fills the mother exactly: its entry distance from inside is -1 (skipped) and from a
    # point on no side; instead tie the mother exit with a daughter placed flush outside the wall
    flush = O.Shape(O.BOX, [5, 20, 20])
    xf = np.array([[1, 0, 0, -25.0, 0, 1, 0, 0, 0, 0, 1, 0]], dtype=np.float64)   # centred at x = +25: touches x = 20
    vol2 = O.Volume(mother, [flush], xf)
    s2, h2 = vol2.compute_step([0.0], [0.0], [0.0], [1.0], [0.0], [0.0])
    assert s2[0] == 20.0 and h2[0] == -1
