"""GPU parity: the CUDA path (through the C ABI of include/vg.h) against the oracle, element by element, on the
same seeded inputs (BASELINE.json configs[0..3]).  Inputs come from workloads/ with
the oracle's sdf deciding the 1e-6 surface-band rejection; nothing here comes from the CUDA path."""
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


@pytest.fixture(scope="module")
def vg():
    import paper_1512_06637_b200 as m
    assert torch.cuda.is_available(), "the CUDA path needs a GPU; there is no fallback"
    return m


@pytest.fixture(params=["pipelined", "plain", "streaming", "auto"])
def kernel_form(request, vg):
    """Force every 16-byte aligned batch through one kernel form (whatever its size), or take the library's choice."""
    old = vg.vg_get_option(vg.OPT_PIPE_MIN_N), vg.vg_get_option(vg.OPT_FORM)
    vg.vg_set_option(vg.OPT_PIPE_MIN_N, 0)
    vg.vg_set_option(vg.OPT_FORM, {"pipelined": vg.FORM_PIPELINED, "plain": vg.FORM_DIRECT, "streaming": vg.FORM_STREAMING,
                                  "auto": vg.FORM_AUTO}[request.param])
    yield request.param
    vg.vg_set_option(vg.OPT_PIPE_MIN_N, old[0])
    vg.vg_set_option(vg.OPT_FORM, old[1])


def dev(arrs):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs]


def oracle_band(s):
    return lambda x, y, z: np.abs(s.sdf(x, y, z)) < W.SURFACE_BAND


def run_oracle(s, q, t, step_max):
    if q in ("distance_to_in", "distance_to_out"):
        return getattr(s, q)(*t, step_max)
    return getattr(s, q)(*t[:3])


def run_gpu(g, q, dt, step_max):
    if q in ("distance_to_in", "distance_to_out"):
        r = getattr(g, q)(*dt, step_max)
    else:
        r = getattr(g, q)(*dt[:3])
    torch.cuda.synchronize()
    return r.cpu().numpy()


def oracle80(kind, params, q, t, step_max):
    """c.7: a mismatch is re-evaluated with the 80-bit build of the oracle (only called when a comparison fails)."""
    def ld(idx):
        s80 = O.Shape(kind, params, long_double=True)
        return run_oracle(s80, q, tuple(np.ascontiguousarray(a[idx]) for a in t), step_max)
    return ld


def check_all(vg, kind, params, t, queries=W.QUERIES5, step_max=W.STEP_MAX, what=""):
    so, sg = O.Shape(kind, params), vg.Shape(kind, params)
    dt = dev(t)
    worst = 0.0
    ref = {}
    for q in queries:
        o = ref[q] = run_oracle(so, q, t, step_max)
        g = run_gpu(sg, q, dt, step_max)
        tag = "%s %s n=%d" % (what, q, len(t[0]))
        if q == "inside":
            assert_int_equal(g, o, tag)
        else:
            worst = max(worst, assert_real_close(g, o, tag, ld=oracle80(kind, params, q, t, step_max)))
    if tuple(queries) == tuple(W.QUERIES5) and len(t[0]) > 0:  # the fused five-query entry point against the same oracle values
        fused = sg.query_all(*dt, step_max)
        torch.cuda.synchronize()
        for q, g in zip(W.QUERIES5, fused):
            tag = "%s fused %s n=%d" % (what, q, len(t[0]))
            if q == "inside":
                assert_int_equal(g.cpu().numpy(), ref[q], tag)
            else:
                worst = max(worst, assert_real_close(g.cpu().numpy(), ref[q], tag))
    return worst


# ------------------------------------------------------------- the configurations at full size, all elements

FULL = [(k, i) for k in (0, 1, 2) for i in range(len(W.shape_cases(k)))]


@pytest.mark.parametrize("k,i", FULL)
def test_config_full_size(vg, k, i):
    sc = W.shape_cases(k)[i]
    t = sc.tracks(band=oracle_band(O.Shape(sc.kind, sc.params)))
    check_all(vg, sc.kind, sc.params, t, sc.queries, what="cfg%d %s" % (k, sc.name))


@pytest.mark.parametrize("i", [0, 1])
@pytest.mark.parametrize("n", [2 ** 10, 2 ** 14, 2 ** 18, 2 ** 22, 2 ** 24])
def test_config3_sweep(vg, i, n):
    sc = W.shape_cases(3)[i]
    t = sc.tracks(n, band=oracle_band(O.Shape(sc.kind, sc.params)))
    check_all(vg, sc.kind, sc.params, t, sc.queries, what="cfg3 %s" % sc.name)


@pytest.mark.parametrize("i", [0, 1])
def test_config3_shapes_all_five_queries(vg, i):
    sc = W.shape_cases(3)[i]
    t = sc.tracks(2 ** 20 + 77, band=oracle_band(O.Shape(sc.kind, sc.params)))
    check_all(vg, sc.kind, sc.params, t, W.QUERIES5, what="cfg3 %s" % sc.name)


# ------------------------------------------------------------------- ragged sizes, misaligned slices, tiny n

ALL_CASES = [(k, i) for k in (0, 1, 2, 3) for i in range(len(W.shape_cases(k)))]


@pytest.mark.parametrize("k,i", ALL_CASES)
def test_ragged_tail_and_misaligned_slices(vg, kernel_form, k, i):
    """n spans many blocks and ends in a ragged tail; slices starting at element 1 are only 8-byte aligned and
    take the 64-bit path (include/vg.h: never an error, never a host fallback)."""
    sc = W.shape_cases(k)[i]
    so, sg = O.Shape(sc.kind, sc.params), vg.Shape(sc.kind, sc.params)
    n = 100003
    t = sc.tracks(n + 1, band=oracle_band(so))
    dt = dev(t)
    for off, m in ((0, n), (1, n), (1, n - 1), (0, 513), (1, 511), (0, 1), (0, 2), (2, 1025), (2, 1024)):
        ts = [a[off:off + m] for a in t]
        ds = [a[off:off + m] for a in dt]
        for q in W.QUERIES5:
            o = run_oracle(so, q, ts, W.STEP_MAX)
            if q == "inside":
                out = torch.empty(m + off, dtype=torch.int32, device="cuda")[off:off + m]
                sg.inside(*ds[:3], out=out)
                assert_int_equal(out.cpu().numpy(), o, "%s inside off=%d" % (sc.name, off))
            else:
                out = torch.empty(m + off, dtype=torch.float64, device="cuda")[off:off + m]
                sg.query(q, *ds, step_max=W.STEP_MAX, out=out)
                assert_real_close(out.cpu().numpy(), o, "%s %s off=%d" % (sc.name, q, off))


@pytest.mark.parametrize("n", [0, 1, 2, 3, 255, 256, 257, 511, 512, 513, 1023, 1025])
def test_tiny_sizes(vg, kernel_form, n):
    sc = W.shape_cases(1)[0]
    so = O.Shape(sc.kind, sc.params)
    t = sc.tracks(n, band=oracle_band(so))
    if n == 0:
        sg = vg.Shape(sc.kind, sc.params)
        e = [torch.empty(0, dtype=torch.float64, device="cuda") for _ in range(6)]
        assert sg.inside(*e[:3]).numel() == 0 and sg.distance_to_in(*e).numel() == 0
        return
    check_all(vg, sc.kind, sc.params, t, what="tiny")


def test_query_all_subsets_and_misaligned_outputs(vg):
    """vg_query_all: NULL outputs are skipped (one kernel per requested answer), all five run fused; outputs that are
    only 8-byte aligned take the 64-bit path; guard elements stay untouched."""
    import ctypes as C
    sc = W.shape_cases(1)[0]
    so, sg = O.Shape(sc.kind, sc.params), vg.Shape(sc.kind, sc.params)
    n = 4099
    t = sc.tracks(n, band=oracle_band(so))
    dt = dev(t)
    ref = {q: run_oracle(so, q, t, W.STEP_MAX) for q in W.QUERIES5}
    # misaligned outputs (offset 1) with guards
    bufs = [torch.full((n + 3,), -7, dtype=torch.int32, device="cuda")] + \
           [torch.full((n + 3,), -7.0, dtype=torch.float64, device="cuda") for _ in range(4)]
    before = vg.vg_launch_count()
    sg.query_all(*dt, W.STEP_MAX, out=[b[1:n + 1] for b in bufs])
    torch.cuda.synchronize()
    assert vg.vg_launch_count() - before == 1
    for q, b in zip(W.QUERIES5, bufs):
        assert b[0].item() == -7 and (b[n + 1:] == -7).all()
        g = b[1:n + 1].cpu().numpy()
        assert_int_equal(g, ref[q], "fused off=1 " + q) if q == "inside" else assert_real_close(g, ref[q], "fused off=1 " + q)
    # a subset through the raw C ABI: NULL pointers skip that answer
    din = torch.empty(n, dtype=torch.float64, device="cuda")
    sout = torch.empty(n, dtype=torch.float64, device="cuda")
    null = C.c_void_p(0)
    p = [C.c_void_p(a.data_ptr()) for a in dt]
    before = vg.vg_launch_count()
    rc = vg._lib.vg_query_all(sg._h, *p, float(W.STEP_MAX), n, null, C.c_void_p(din.data_ptr()), null, null,
                              C.c_void_p(sout.data_ptr()), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    torch.cuda.synchronize()
    assert rc == 0 and vg.vg_launch_count() - before == 2
    assert_real_close(din.cpu().numpy(), ref["distance_to_in"], "subset din")
    assert_real_close(sout.cpu().numpy(), ref["safety_to_out"], "subset sout")
    assert vg._lib.vg_query_all(sg._h, *p, float(W.STEP_MAX), n, null, null, null, null, null, null) == vg.ERR_ARG


def test_outputs_do_not_overrun(vg, kernel_form):
    """Guard elements after the output must stay untouched for odd n on the 128-bit path."""
    sc = W.shape_cases(0)[0]
    sg = vg.Shape(sc.kind, sc.params)
    for n in (1, 3, 255, 1001):
        t = dev(sc.tracks(n))
        buf = torch.full((n + 5,), -7.0, dtype=torch.float64, device="cuda")
        sg.distance_to_in(*t, out=buf[:n])
        ibuf = torch.full((n + 5,), -7, dtype=torch.int32, device="cuda")
        sg.inside(*t[:3], out=ibuf[:n])
        torch.cuda.synchronize()
        assert (buf[n:] == -7.0).all() and (ibuf[n:] == -7).all()


# ---------------------------------------------------------------------- shape variants and random parameters

VARIANTS = [
    ("tube_full", W.TUBE, [5.0, 10.0, 15.0, 0.0, TWO_PI]),
    ("tube_solid", W.TUBE, [0.0, 10.0, 15.0, 0.0, TWO_PI]),
    ("tube_narrow", W.TUBE, [3.0, 9.0, 12.0, 0.7, 1.1]),
    ("tube_half", W.TUBE, [3.0, 9.0, 12.0, -1.0, math.pi]),
    ("tube_solid_wedge", W.TUBE, [0.0, 9.0, 12.0, 2.0, 4.5]),
    ("cone_wedge", W.CONE, [2.0, 6.0, 4.0, 12.0, 20.0, 0.3, 4.0]),
    ("cone_narrow", W.CONE, [2.0, 6.0, 4.0, 12.0, 20.0, -2.0, 1.3]),
    ("cone_solid", W.CONE, [0.0, 6.0, 0.0, 12.0, 20.0, 0.0, TWO_PI]),
    ("cone_apex_in", W.CONE, [0.0, 6.0, 4.0, 12.0, 20.0, 0.0, TWO_PI]),
    ("cone_reversed", W.CONE, [4.0, 12.0, 2.0, 6.0, 20.0, 0.0, TWO_PI]),
    ("cone_solid_wedge", W.CONE, [0.0, 8.0, 0.0, 3.0, 10.0, 1.0, 2.0]),
    ("trd_box", W.TRD, [5.0, 5.0, 7.0, 7.0, 15.0]),
    ("trd_steep", W.TRD, [1.0, 20.0, 18.0, 2.0, 5.0]),
    ("box_flat", W.BOX, [50.0, 0.5, 7.0]),
    ("orb_small", W.ORB, [0.75]),
    ("polycone_wedge", W.POLYCONE, [0.5, 4.0, 4.0, -10.0, 1.0, 5.0, -2.0, 2.0, 9.0, 3.0, 0.0, 6.0, 12.0, 3.0, 4.0]),
    ("polycone_solid", W.POLYCONE, [0.0, TWO_PI, 3.0, -10.0, 0.0, 5.0, 0.0, 0.0, 9.0, 8.0, 0.0, 2.0]),
    ("polycone_narrow", W.POLYCONE, [-1.0, 1.2, 3.0, -10.0, 0.0, 5.0, 0.0, 0.0, 9.0, 8.0, 3.0, 4.0]),
    # z steps (reading R26): radii jump at z = -4 (outwards, the bore opens) and at z = 6 (inwards, the bore closes)
    ("polycone_step", W.POLYCONE, [0.0, TWO_PI, 7.0, -12.0, 0.0, 6.0, -4.0, 1.0, 8.0, -4.0, 3.0, 12.0, 2.0, 2.0, 10.0, 6.0, 2.0, 11.0,
                                   6.0, 0.0, 5.0, 14.0, 1.5, 4.0]),
    ("polycone_step_wedge", W.POLYCONE, [-0.7, 4.1, 7.0, -12.0, 0.0, 6.0, -4.0, 1.0, 8.0, -4.0, 3.0, 12.0, 2.0, 2.0, 10.0, 6.0, 2.0,
                                         11.0, 6.0, 0.0, 5.0, 14.0, 1.5, 4.0]),
    ("polycone_two_tubes", W.POLYCONE, [0.0, TWO_PI, 4.0, -10.0, 2.0, 5.0, 0.0, 2.0, 5.0, 0.0, 3.0, 9.0, 6.0, 3.0, 9.0]),
    ("polycone_step_outer_only", W.POLYCONE, [0.0, TWO_PI, 4.0, -10.0, 0.0, 9.0, 0.0, 0.0, 9.0, 0.0, 0.0, 4.0, 6.0, 0.0, 4.0]),
]


@pytest.mark.parametrize("name,kind,params", VARIANTS, ids=[v[0] for v in VARIANTS])
def test_shape_variants(vg, name, kind, params):
    c, h = W.bounding_half(kind, params)
    so = O.Shape(kind, params)
    t = W.draw_tracks(4242, 200001, c, tuple(1.5 * v for v in h), oracle_band(so))
    check_all(vg, kind, params, t, what=name)


def _random_params(kind, rng):
    if kind == W.BOX:
        return list(rng.uniform(0.5, 20.0, 3))
    if kind == W.ORB:
        return [float(rng.uniform(0.5, 30.0))]
    if kind == W.TUBE:
        rmin = float(rng.choice([0.0, rng.uniform(0.1, 8.0)]))
        return [rmin, rmin + float(rng.uniform(0.5, 10.0)), float(rng.uniform(0.5, 20.0)),
                float(rng.uniform(-math.pi, math.pi)), float(rng.choice([TWO_PI, rng.uniform(0.2, 6.0)]))]
    if kind == W.CONE:
        a = float(rng.choice([0.0, rng.uniform(0.1, 6.0)]))
        b = float(rng.choice([0.0, rng.uniform(0.1, 6.0)]))
        return [a, a + float(rng.uniform(0.5, 8.0)), b, b + float(rng.uniform(0.5, 8.0)), float(rng.uniform(0.5, 20.0)),
                float(rng.uniform(-math.pi, math.pi)), float(rng.choice([TWO_PI, rng.uniform(0.2, 6.0)]))]
    if kind == W.TRD:
        return list(rng.uniform(0.5, 15.0, 5))
    nz = int(rng.integers(2, 12))
    z = np.sort(rng.uniform(-30, 30, nz))
    z += np.arange(nz) * 0.05  # keep the planes strictly increasing and apart
    out = [float(rng.uniform(-math.pi, math.pi)), float(rng.choice([TWO_PI, rng.uniform(0.2, 6.0)])), float(nz)]
    for i in range(nz):
        a = float(rng.choice([0.0, rng.uniform(0.0, 5.0)]))
        out += [float(z[i]), a, a + float(rng.uniform(0.5, 20.0))]
    # every other polycone gets z steps (R26): an interior plane is duplicated with new radii that overlap the old range
    if nz >= 3 and rng.random() < 0.5:
        for i in sorted(rng.choice(np.arange(1, nz - 1), size=min(2, nz - 2), replace=False), reverse=True):
            zi, a, b = out[3 + 3 * i: 6 + 3 * i]
            mid = 0.5 * (a + b)
            a2 = float(rng.choice([0.0, rng.uniform(0.0, mid)]))
            b2 = mid + float(rng.uniform(0.2, 15.0))
            out[6 + 3 * i: 6 + 3 * i] = [zi, a2 if a2 < mid else 0.0, b2]
            out[2] += 1.0
    return out


@pytest.mark.parametrize("kind", range(6), ids=[W.KIND_NAME[k] for k in range(6)])
def test_random_parameters(vg, kind):
    rng = np.random.default_rng(9000 + kind)
    for rep in range(int(os.environ.get("VG_STRESS_REPS", "12"))):  # VG_STRESS_REPS=200 for a long soak
        params = _random_params(kind, rng)
        c, h = W.bounding_half(kind, params)
        so = O.Shape(kind, params)
        t = W.draw_tracks(77 + rep, 30011, c, tuple(1.5 * v for v in h), oracle_band(so))
        check_all(vg, kind, params, t, what="%s%r" % (W.KIND_NAME[kind], params))
