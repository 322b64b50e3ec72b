"""GPU parity of the lanes-per-track form of the full-phi polycone queries (csrc/vg_pcon_coop.cuh; DESIGN.md sec. 6.2;
PAPER.md:122: small batches) against the oracle, all five queries, and of the form switch: the same batch through the
thread-per-track kernels (VG_OPT_COOP_MAX_N = 0) and through the lane groups (VG_OPT_COOP_MAX_N >= n), sizes on both
sides of the threshold, groups of 4 / 8 / 16 / 32 lanes (nz = 2..32), z steps, misaligned slices, surface-band starts."""
import math

import numpy as np
import pytest

import oracle as O
import workloads as W
from parity import assert_int_equal, assert_real_close
from test_gpu_parity import _random_params, check_all, dev, oracle_band, run_gpu, run_oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
TWO_PI = 2 * math.pi


@pytest.fixture(scope="module")
def vg():
    import paper_1512_06637_b200 as m
    assert torch.cuda.is_available(), "the CUDA path needs a GPU; there is no fallback"
    return m


@pytest.fixture(params=["lanes", "medium", "threads"])
def form(request, vg):
    """lanes: a group of lanes per track whatever n; medium: one track per thread, tables in device memory (what every batch
    above VG_OPT_COOP_MAX_N runs as; here every n > 1); threads: the persistent kernels with the tables staged per CTA."""
    old = vg.vg_get_option(vg.OPT_COOP_MAX_N)
    vg.vg_set_option(vg.OPT_COOP_MAX_N, {"lanes": 1 << 40, "medium": 1, "threads": 0}[request.param])
    yield request.param
    vg.vg_set_option(vg.OPT_COOP_MAX_N, old)


def polycone(seed, nz, rmin_hi=5.0, steps=0):
    rng = np.random.default_rng(seed)
    z = np.sort(rng.uniform(-50.0, 50.0, nz)) + np.arange(nz) * 1e-3
    rmin = rng.uniform(0.0, rmin_hi, nz) if rmin_hi > 0 else np.zeros(nz)
    rmax = rng.uniform(10.0, 30.0, nz)
    out = [0.0, TWO_PI, float(nz)]
    for i in range(nz):
        out += [float(z[i]), float(rmin[i]), float(rmax[i])]
    for i in sorted(rng.choice(np.arange(1, nz - 1), size=min(steps, max(nz - 2, 0)), replace=False), reverse=True) if nz >= 3 else []:
        zi, a, b = out[3 + 3 * i: 6 + 3 * i]  # a z step (R26): the plane is duplicated with radii that overlap the old range
        mid = 0.5 * (a + b)
        out[6 + 3 * i: 6 + 3 * i] = [zi, float(rng.uniform(0.0, mid)) if rng.random() < 0.5 else 0.0, mid + float(rng.uniform(0.2, 15.0))]
        out[2] += 1.0
    return out


@pytest.mark.parametrize("n", [1, 2, 3, 7, 33, 1000, 1024, 16384, 40001])
def test_config3_polycone_small_batches(vg, form, n):
    sc = W.shape_cases(3)[0]
    t = sc.tracks(n, band=oracle_band(O.Shape(sc.kind, sc.params)))
    check_all(vg, sc.kind, sc.params, t, W.QUERIES5, what="cfg3 polycone %s" % form)


@pytest.mark.parametrize("seed,nz,rmin_hi,steps", [(1, 2, 5.0, 0), (2, 3, 0.0, 1), (3, 5, 5.0, 0), (4, 6, 5.0, 2), (5, 9, 9.0, 0),
                                                   (6, 10, 5.0, 2), (7, 17, 5.0, 0), (8, 18, 0.0, 2), (9, 30, 5.0, 2), (10, 32, 5.0, 0)])
def test_every_group_width_and_z_steps(vg, form, seed, nz, rmin_hi, steps):
    """nsec = 1..31: groups of 4, 8, 16 and 32 lanes, a lane with one section or (nsec > 32: none here) several."""
    par = polycone(seed, nz, rmin_hi, steps)
    c, h = W.bounding_half(W.POLYCONE, par)
    t = W.draw_tracks(500 + seed, 20011, c, tuple(1.5 * v for v in h), oracle_band(O.Shape(W.POLYCONE, par)))
    check_all(vg, W.POLYCONE, par, t, W.QUERIES5, what="polycone nz=%d steps=%d %s" % (nz, steps, form))


def test_threshold_switches_the_form_and_both_sides_agree_with_the_oracle(vg):
    """n = threshold - 1, threshold, threshold + 1: the first two run as lane groups, the third as the one-track-per-thread
    walk (one launch each through the launch counter; every answer against the oracle)."""
    sc = W.shape_cases(3)[0]
    so, sg = O.Shape(sc.kind, sc.params), vg.Shape(sc.kind, sc.params)
    old = vg.vg_get_option(vg.OPT_COOP_MAX_N)
    try:
        vg.vg_set_option(vg.OPT_COOP_MAX_N, 5000)
        for n in (4999, 5000, 5001):
            t = sc.tracks(n, band=oracle_band(so))
            dt = dev(t)
            for q in W.QUERIES5:
                before = vg.vg_launch_count()
                g = run_gpu(sg, q, dt, W.STEP_MAX)
                assert vg.vg_launch_count() - before == 1
                o = run_oracle(so, q, t, W.STEP_MAX)
                if q == "inside":
                    assert_int_equal(g, o, "threshold n=%d %s" % (n, q))
                else:
                    assert_real_close(g, o, "threshold n=%d %s" % (n, q))
    finally:
        vg.vg_set_option(vg.OPT_COOP_MAX_N, old)


def test_misaligned_slices_and_step_max(vg, form):
    """Arrays that are only 8-byte aligned (a slice starting at element 1), and a finite physics step."""
    sc = W.shape_cases(3)[0]
    so, sg = O.Shape(sc.kind, sc.params), vg.Shape(sc.kind, sc.params)
    t = sc.tracks(3001, band=oracle_band(so))
    big = [torch.from_numpy(np.concatenate([[0.0], a])).cuda() for a in t]
    ds = [b[1:] for b in big]
    assert all(d.data_ptr() % 16 == 8 for d in ds)
    for step_max in (W.STEP_MAX, 12.5):
        for q in ("distance_to_in", "distance_to_out"):
            g = getattr(sg, q)(*ds, step_max).cpu().numpy()
            assert_real_close(g, getattr(so, q)(*t, step_max), "misaligned %s step_max=%g" % (q, step_max))
    assert_real_close(sg.safety_to_in(*ds[:3]).cpu().numpy(), so.safety_to_in(*t[:3]), "misaligned safety_to_in")
    assert_int_equal(sg.inside(*ds[:3]).cpu().numpy(), so.inside(*t[:3]), "misaligned inside")


def test_starts_on_the_surface(vg, form):
    """Reading R32: tracks moved onto their own crossing of the polycone (p + t d, then +-1e-12 along d) return the same
    classes and next distances as the oracle."""
    sc = W.shape_cases(3)[0]
    so, sg = O.Shape(sc.kind, sc.params), vg.Shape(sc.kind, sc.params)
    x, y, z, dx, dy, dz = sc.tracks(60001, band=oracle_band(so))
    tin = so.distance_to_in(x, y, z, dx, dy, dz)
    hit = np.isfinite(tin) & (tin > 0)
    for off in (0.0, 1e-12, -1e-12):
        s = (tin[hit] + off)
        t = tuple(np.ascontiguousarray(a) for a in (x[hit] + s * dx[hit], y[hit] + s * dy[hit], z[hit] + s * dz[hit], dx[hit], dy[hit], dz[hit]))
        dt = dev(t)
        assert_int_equal(sg.inside(*dt[:3]).cpu().numpy(), so.inside(*t[:3]), "surface inside off=%g" % off)
        for q in ("distance_to_in", "distance_to_out"):
            assert_real_close(getattr(sg, q)(*dt, W.STEP_MAX).cpu().numpy(), getattr(so, q)(*t, W.STEP_MAX), "surface %s off=%g" % (q, off))
