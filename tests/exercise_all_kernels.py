"""Launches every kernel of libvg once on small odd-sized inputs (all solids, all queries, every kernel form, 8-byte-only
alignment, the three polycone forms, the fused call, ComputeStep in both phase-2 forms, the world, a boolean of every
operand kind, the host entry points).  Not a test
by itself (`python tests/exercise_all_kernels.py` on a GPU box; tests/test_gpu_nav_and_edges.py runs it as one).  compute-sanitizer
is closed on this pool, so the script brings its own bounds check: every result array sits between guard words that must
come back untouched, sizes are odd, and every result is compared with the oracle."""
import math
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))
import oracle as O  # noqa: E402
import paper_1512_06637_b200 as vg  # noqa: E402
import workloads as W  # noqa: E402
from parity import assert_int_equal, assert_real_close  # noqa: E402

N = 5001


def dev(t, misalign=False):
    if not misalign:
        return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in t]
    out = []
    for a in t:  # 8-byte aligned only: the TPT = 1 kernels
        buf = torch.empty(len(a) + 1, dtype=torch.float64, device="cuda")
        buf[1:].copy_(torch.from_numpy(np.ascontiguousarray(a)))
        out.append(buf[1:])
    return out


GUARD = 4  # elements in front of and behind every guarded result array (keeps 16-byte alignment for FP64 and int32)


def guarded(n, dtype, shift=0):
    """A result array of n elements inside a buffer pre-filled with a pattern; `shift` = 1 makes it 8-byte aligned only."""
    buf = torch.full((n + 2 * GUARD + shift,), -12345, dtype=dtype, device="cuda")
    return buf, buf[GUARD + shift: GUARD + shift + n]


def guards_intact(buf, n, shift=0):
    head, tail = buf[: GUARD + shift], buf[GUARD + shift + n:]
    return bool((head == -12345).all()) and bool((tail == -12345).all())


def check_shape(kind, par, what):
    so, sg = O.Shape(kind, par), vg.Shape(kind, par)
    c, h = W.bounding_half(kind, par)
    t = W.draw_tracks(17, N, c, tuple(1.5 * v for v in h), lambda x, y, z: np.abs(so.sdf(x, y, z)) < W.SURFACE_BAND)
    for form in (vg.FORM_AUTO, vg.FORM_DIRECT, vg.FORM_PIPELINED, vg.FORM_STREAMING):
        vg.vg_set_option(vg.OPT_FORM, form)
        vg.vg_set_option(vg.OPT_PIPE_MIN_N, 0)
        for mis in (False, True):
            dt = dev(t, mis)
            bi, oi = guarded(N, torch.int32, 1 if mis else 0)
            bd, od = guarded(N, torch.float64, 1 if mis else 0)
            assert_int_equal(sg.inside(*dt[:3], out=oi).cpu().numpy(), so.inside(*t[:3]), what)
            assert_real_close(sg.distance_to_in(*dt, W.STEP_MAX, out=od).cpu().numpy(), so.distance_to_in(*t, W.STEP_MAX), what)
            assert guards_intact(bi, N, 1 if mis else 0) and guards_intact(bd, N, 1 if mis else 0), what + ": write outside the result array"
            for q in ("distance_to_out", "safety_to_in"):
                bd, od = guarded(N, torch.float64, 1 if mis else 0)
                sg.query(q, *dt, step_max=W.STEP_MAX, out=od) if q.startswith("distance") else sg.query(q, *dt[:3], out=od)
                assert guards_intact(bd, N, 1 if mis else 0), what + " " + q + ": write outside the result array"
            assert_real_close(sg.distance_to_out(*dt, W.STEP_MAX).cpu().numpy(), so.distance_to_out(*t, W.STEP_MAX), what)
            assert_real_close(sg.safety_to_in(*dt[:3]).cpu().numpy(), so.safety_to_in(*t[:3]), what)
            assert_real_close(sg.safety_to_out(*dt[:3]).cpu().numpy(), so.safety_to_out(*t[:3]), what)
    vg.vg_set_option(vg.OPT_FORM, vg.FORM_AUTO)
    if kind == W.POLYCONE:  # the three polycone forms: a group of lanes per track, one track per thread, persistent CTAs
        old = vg.vg_get_option(vg.OPT_COOP_MAX_N)
        for coop in (1 << 40, 1, 0):
            vg.vg_set_option(vg.OPT_COOP_MAX_N, coop)
            for mis in (False, True):
                dt = dev(t, mis)
                sh = 1 if mis else 0
                bi, oi = guarded(N, torch.int32, sh)
                assert_int_equal(sg.inside(*dt[:3], out=oi).cpu().numpy(), so.inside(*t[:3]), what + " form %d" % coop)
                assert guards_intact(bi, N, sh), what + " inside form %d: write outside the result array" % coop
                for q in ("distance_to_in", "distance_to_out", "safety_to_in", "safety_to_out"):
                    bd, od = guarded(N, torch.float64, sh)
                    g = sg.query(q, *dt, step_max=W.STEP_MAX, out=od) if q.startswith("distance") else sg.query(q, *dt[:3], out=od)
                    o = getattr(so, q)(*t, W.STEP_MAX) if q.startswith("distance") else getattr(so, q)(*t[:3])
                    assert_real_close(g.cpu().numpy(), o, what + " %s form %d" % (q, coop))
                    assert guards_intact(bd, N, sh), what + " %s form %d: write outside the result array" % (q, coop)
        vg.vg_set_option(vg.OPT_COOP_MAX_N, old)
    gb = [guarded(N, torch.int32)] + [guarded(N, torch.float64) for _ in range(4)]  # the fused call, every output guarded
    fused = sg.query_all(*dev(t), W.STEP_MAX, out=[g[1] for g in gb])
    assert all(guards_intact(g[0], N) for g in gb), what + " fused: write outside a result array"
    assert_real_close(fused[1].cpu().numpy(), so.distance_to_in(*t, W.STEP_MAX), what + " fused")
    ht = [torch.from_numpy(a).pin_memory() for a in t]
    assert_real_close(sg.query_host("distance_to_out", *ht, step_max=W.STEP_MAX).numpy(), so.distance_to_out(*t, W.STEP_MAX), what + " host")
    blk = torch.empty((6, N), dtype=torch.float64).pin_memory()
    for i in range(6):
        blk[i].copy_(ht[i])
    res = sg.query_all_host(*[blk[i] for i in range(6)], step_max=W.STEP_MAX)
    assert_real_close(res[3].numpy(), so.safety_to_in(*t[:3]), what + " host fused")


def main():
    torch.cuda.set_device(0)
    two_pi = 2 * math.pi
    shapes = [(W.BOX, [5, 5, 5]), (W.ORB, [20]), (W.TUBE, [5, 10, 15, 0, 4 * math.pi / 3]), (W.TUBE, [0, 8, 8, 0, two_pi]),
              (W.TUBE, [3, 9, 12, 0.7, 1.1]), (W.CONE, [2, 6, 4, 12, 20, 0, two_pi]), (W.CONE, [2, 6, 4, 12, 20, 0.3, 4.0]),
              (W.TRD, [5, 10, 7, 3, 15]), (W.POLYCONE, W.polycone_params(W.config_seed(3, 0))), (W.POLYCONE, W.STEPPED_POLYCONE),
              (W.POLYCONE, [-0.7, 4.1] + W.STEPPED_POLYCONE[2:])]
    for kind, par in shapes:
        check_shape(kind, [float(v) for v in par], "%s%r" % (W.KIND_NAME[kind], par[:3]))
    nav = W.navigator_case()
    vo = O.Volume(O.Shape(nav.mother_kind, nav.mother_params), [O.Shape(k, p) for k, p in zip(nav.daughter_kinds, nav.daughter_params)], nav.xforms)
    vgv = vg.Volume(vg.Shape(nav.mother_kind, nav.mother_params), [vg.Shape(k, p) for k, p in zip(nav.daughter_kinds, nav.daughter_params)], nav.xforms)
    t = nav.tracks(N, band=lambda x, y, z: vo.safety(x, y, z) < W.SURFACE_BAND)
    so, ho = vo.compute_step(*t, W.STEP_MAX)
    for form in (1, 2, 0):  # phase 2 per lane, pooled over the warp, the library's choice
        vg.vg_set_option(vg.OPT_NAV_FORM, form)
        bs, os_ = guarded(N, torch.float64)
        bh, oh = guarded(N, torch.int32)
        sg, hg = vgv.compute_step(*dev(t), W.STEP_MAX, step=os_, hit=oh)
        assert_int_equal(hg.cpu().numpy(), ho, "compute_step hit form %d" % form)
        assert_real_close(sg.cpu().numpy(), so, "compute_step form %d" % form)
        assert guards_intact(bs, N) and guards_intact(bh, N), "compute_step form %d: write outside a result array" % form
    vg.vg_set_option(vg.OPT_NAV_FORM, 0)
    assert_real_close(vgv.safety(*dev(t[:3])).cpu().numpy(), vo.safety(*t[:3]), "volume safety")
    wc = W.world_case()
    wo = O.World([O.Shape(k, p) for k, p in zip(wc.kinds, wc.params)], wc.parents, wc.xforms)
    wg = vg.World([vg.Shape(k, p) for k, p in zip(wc.kinds, wc.params)], wc.parents, wc.xforms)

    def wband(x, y, z):
        nd = wo.locate(x, y, z)
        return (nd < 0) | (wo.safety(nd, x, y, z) < W.SURFACE_BAND)
    t = wc.tracks(N, wband)
    dt = dev(t)
    node = wg.locate(*dt[:3])
    assert_int_equal(node.cpu().numpy(), wo.locate(*t[:3]), "world locate")
    s1, n1 = wg.step(node, *dt, W.STEP_MAX)
    s0, n0 = wo.step(node.cpu().numpy(), *t, W.STEP_MAX)
    assert_int_equal(n1.cpu().numpy(), n0, "world next")
    assert_real_close(s1.cpu().numpy(), s0, "world step")
    assert_real_close(wg.safety(node, *dt[:3]).cpu().numpy(), wo.safety(node.cpu().numpy(), *t[:3]), "world safety")
    for bc in W.boolean_cases():
        co = O.Boolean(bc.op, O.Shape(bc.kind_a, bc.par_a), O.Shape(bc.kind_b, bc.par_b), bc.xform)
        cg = vg.Boolean(bc.op, vg.Shape(bc.kind_a, bc.par_a), vg.Shape(bc.kind_b, bc.par_b), bc.xform)
        M = np.asarray(bc.xform).reshape(3, 4)

        def bband(x, y, z):
            L = M[:, :3] @ np.stack([x, y, z]) + M[:, 3:4]
            return (np.abs(co.a.sdf(x, y, z)) < W.SURFACE_BAND) | (np.abs(co.b.sdf(L[0], L[1], L[2])) < W.SURFACE_BAND)
        t = bc.tracks(N, bband)
        dt = dev(t)
        assert_int_equal(cg.inside(*dt[:3]).cpu().numpy(), co.inside(*t[:3]), bc.name)
        assert_real_close(cg.distance_to_in(*dt, W.STEP_MAX).cpu().numpy(), co.distance_to_in(*t, W.STEP_MAX), bc.name)
        assert_real_close(cg.distance_to_out(*dt, W.STEP_MAX).cpu().numpy(), co.distance_to_out(*t, W.STEP_MAX), bc.name)
        assert_real_close(cg.safety_to_in(*dt[:3]).cpu().numpy(), co.safety_to_in(*t[:3]), bc.name)
    # the two-tracks-per-thread point kernels of the booleans (aligned arrays, >= 2 x 148 x 256 tracks): odd size, guarded outputs
    bc = W.boolean_cases()[0]
    co = O.Boolean(bc.op, O.Shape(bc.kind_a, bc.par_a), O.Shape(bc.kind_b, bc.par_b), bc.xform)
    cg = vg.Boolean(bc.op, vg.Shape(bc.kind_a, bc.par_a), vg.Shape(bc.kind_b, bc.par_b), bc.xform)
    M = np.asarray(bc.xform).reshape(3, 4)

    def bband2(x, y, z):
        L = M[:, :3] @ np.stack([x, y, z]) + M[:, 3:4]
        return (np.abs(co.a.sdf(x, y, z)) < W.SURFACE_BAND) | (np.abs(co.b.sdf(L[0], L[1], L[2])) < W.SURFACE_BAND)
    nb = 2 * 148 * 256 + 5
    t = bc.tracks(nb, bband2)
    dt = dev(t)
    bi, oi = guarded(nb, torch.int32)
    cg.inside(*dt[:3], out=oi)
    assert guards_intact(bi, nb), "boolean inside (two tracks per thread) wrote outside its array"
    assert_int_equal(oi.cpu().numpy(), co.inside(*t[:3]), "boolean inside, two tracks per thread")
    for q in ("safety_to_in", "safety_to_out"):
        bd, od = guarded(nb, torch.float64)
        getattr(cg, q)(*dt[:3], out=od)
        assert guards_intact(bd, nb), "boolean %s (two tracks per thread) wrote outside its array" % q
        assert_real_close(od.cpu().numpy(), getattr(co, q)(*t[:3]), "boolean %s, two tracks per thread" % q)
    vg.vg_probe_fp64_fma_rate(1)
    vg.vg_probe_empty_launch(2)
    torch.cuda.synchronize()
    print("exercise_all_kernels: ok, %d libvg kernel launches" % vg.vg_launch_count())


if __name__ == "__main__":
    main()
