"""vg_query_host_static (include/vg.h, csrc/vg_static.cu): the host-buffer query that allocates nothing -- its device staging
area is a static array of the library's device image -- against the existing paths (vg_query_host, whose staging memory is
cudaMalloc'ed on first use, and the device entry points) and the oracle.  Two calls in a row share the array: the second,
shorter call must not see the first one's leftovers.  Collected last (the file name): a failure here hides no other test."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from parity import assert_int_equal, assert_real_close

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def vg():
    import paper_1512_06637_b200 as m
    assert torch.cuda.is_available(), "the CUDA path needs a GPU; there is no fallback"
    return m


def band(s):
    return lambda x, y, z: np.abs(s.sdf(x, y, z)) < W.SURFACE_BAND


def host(t, pinned):
    ts = [torch.from_numpy(np.ascontiguousarray(a)) for a in t]
    return [a.pin_memory() for a in ts] if pinned else ts


def check(vg, sg, so, t, pinned, what):
    ht = host(t, pinned)
    dt = [a.cuda() for a in ht]
    for q in W.QUERIES5:
        args = ht if q.startswith("distance") else ht[:3]
        got = sg.query_host_static(q, *args, step_max=W.STEP_MAX).numpy()
        old = sg.query_host(q, *args, step_max=W.STEP_MAX).numpy()
        if q.startswith("distance"):
            dev = getattr(sg, q)(*dt, W.STEP_MAX).cpu().numpy()
            ref = getattr(so, q)(*t, W.STEP_MAX)
        else:
            dev = getattr(sg, q)(*dt[:3]).cpu().numpy()
            ref = getattr(so, q)(*t[:3])
        close = assert_int_equal if q == "inside" else assert_real_close
        close(got, old, "%s %s: static staging vs vg_query_host" % (what, q))
        close(got, dev, "%s %s: static staging vs the device entry point" % (what, q))
        close(got, ref, "%s %s: static staging vs the oracle" % (what, q))


@pytest.mark.parametrize("cfg", [1, 3])
def test_two_calls_in_a_row_match_the_existing_paths(vg, cfg):
    """configs[1] tube / configs[3] polycone: a full-size call (VG_STATIC_MAX_TRACKS tracks), then a shorter one on other
    tracks in the same array, then a single track; pageable and pinned host memory."""
    sc = W.shape_cases(cfg)[0]
    so, sg = O.Shape(sc.kind, sc.params), vg.Shape(sc.kind, sc.params)
    c, h = W.bounding_half(sc.kind, sc.params)
    for k, (n, pinned) in enumerate(((vg.STATIC_MAX_TRACKS, False), (40001, True), (1, False))):
        t = W.draw_tracks(900 + 10 * cfg + k, n, c, tuple(1.5 * v for v in h), band(so))
        check(vg, sg, so, t, pinned, "cfg%d call %d (n=%d)" % (cfg, k, n))


def test_no_device_memory_is_allocated_and_a_side_stream_works(vg):
    sc = W.shape_cases(1)[0]
    so, sg = O.Shape(sc.kind, sc.params), vg.Shape(sc.kind, sc.params)
    c, h = W.bounding_half(sc.kind, sc.params)
    t = W.draw_tracks(77, 50000, c, tuple(1.5 * v for v in h), band(so))
    ht = host(t, True)
    out = torch.empty(len(t[0]), dtype=torch.float64).pin_memory()
    st = torch.cuda.Stream()
    for q in ("distance_to_out", "distance_to_in"):  # the driver loads a kernel's code on its first launch: not the call's doing
        sg.query_host_static(q, *ht, step_max=W.STEP_MAX, out=out, stream=st)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for q in ("distance_to_out", "distance_to_in"):
        sg.query_host_static(q, *ht, step_max=W.STEP_MAX, out=out, stream=st)
        assert_real_close(out.numpy(), getattr(so, q)(*t, W.STEP_MAX), "side stream %s" % q)
    assert torch.cuda.mem_get_info()[0] >= free0, "the call took device memory"


def test_sizes_beyond_the_static_array_are_rejected(vg):
    sg = vg.Shape(W.BOX, [5.0, 5.0, 5.0])
    n = vg.STATIC_MAX_TRACKS + 1
    a = torch.zeros(n, dtype=torch.float64)
    out = torch.full((n,), 7.0, dtype=torch.float64)
    with pytest.raises(vg.VgError, match="VG_STATIC_MAX_TRACKS"):
        sg.query_host_static("safety_to_in", a, a, a, out=out)
    assert bool((out == 7.0).all())  # nothing was enqueued
    assert sg.query_host_static("safety_to_in", a[:0], a[:0], a[:0]).numel() == 0  # n = 0: nothing to do


def test_two_host_threads_share_the_array_without_racing(vg):
    """All calls use ONE staging array; the entry point serialises them with a lock and waits for its own work, so two host
    threads on two streams, each with its own tracks, must both get their own answers (ctypes drops the GIL in the call)."""
    import threading
    sc = W.shape_cases(1)[0]
    so, sg = O.Shape(sc.kind, sc.params), vg.Shape(sc.kind, sc.params)
    c, h = W.bounding_half(sc.kind, sc.params)
    jobs = []
    for k in range(2):
        t = W.draw_tracks(300 + k, 30000 + 5000 * k, c, tuple(1.5 * v for v in h), band(so))
        jobs.append((t, host(t, True), so.distance_to_in(*t, W.STEP_MAX), torch.cuda.Stream()))
    errors = []

    def work(k):
        t, ht, want, st = jobs[k]
        try:
            torch.cuda.set_device(0)
            for _ in range(40):
                got = sg.query_host_static("distance_to_in", *ht, step_max=W.STEP_MAX, stream=st).numpy()
                assert_real_close(got, want, "thread %d" % k)
        except Exception as e:  # noqa: BLE001 (reported by the main thread)
            errors.append(e)
    threads = [threading.Thread(target=work, args=(k,)) for k in range(2)]
    for th in threads:
        th.start()
    for th in threads:
        th.join()
    assert not errors, errors[0]


def test_the_call_can_be_captured_into_a_cuda_graph(vg):
    """The caller the entry point exists for: under graph capture nothing may allocate or synchronise.  One direct call
    first (it looks up the array's address), then the call is captured on pinned arrays; every replay answers for the
    tracks that sit in those arrays at that moment."""
    sc = W.shape_cases(1)[0]
    so, sg = O.Shape(sc.kind, sc.params), vg.Shape(sc.kind, sc.params)
    c, h = W.bounding_half(sc.kind, sc.params)
    n = 20000
    sets = [W.draw_tracks(500 + k, n, c, tuple(1.5 * v for v in h), band(so)) for k in range(3)]
    ht = host(sets[0], True)
    out = torch.empty(n, dtype=torch.float64).pin_memory()
    sg.query_host_static("distance_to_in", *ht, step_max=W.STEP_MAX, out=out)
    assert_real_close(out.numpy(), so.distance_to_in(*sets[0], W.STEP_MAX), "direct call before the capture")
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        sg.query_host_static("distance_to_in", *ht, step_max=W.STEP_MAX, out=out)
    for k in (1, 2, 0):
        for a, src in zip(ht, sets[k]):
            a.copy_(torch.from_numpy(src))
        out.fill_(-7.0)
        g.replay()
        torch.cuda.synchronize()
        assert_real_close(out.numpy(), so.distance_to_in(*sets[k], W.STEP_MAX), "graph replay on track set %d" % k)
