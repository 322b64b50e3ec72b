"""CPU-side checks of the boundary (no GPU): libvg.so loads, exports every symbol include/vg.h declares, validates
parameters, treats n == 0 as a no-op and FAILS LOUDLY (VG_ERR_CUDA) when asked to compute without a CUDA device;
plus the world_size-2 gloo test of the track sharding."""
import ctypes as C
import math
import os
import re
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "vg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(vg_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    import paper_1512_06637_b200 as vg
    lib = C.CDLL(vg.LIB_PATH)
    names = declared_symbols()
    assert len(names) >= 18 and "vg_compute_step" in names and "vg_query_host" in names
    for name in names:
        assert hasattr(lib, name), "libvg.so does not export %s" % name


def test_oracle_and_cuda_path_share_no_code():
    """Neither side includes or imports the other (the independence the parity claim rests on)."""
    csrc = os.path.join(ROOT, "paper_1512_06637_b200", "csrc")
    for f in os.listdir(csrc):
        for inc in re.findall(r'#include\s*[<"]([^>"]+)[>"]', open(os.path.join(csrc, f)).read()):
            assert "oracle" not in inc.lower(), (f, inc)
            if "/" in inc:
                assert inc == "../../include/vg.h", (f, inc)
    for f in ("__init__.py", "build.py", "shard.py"):
        src = open(os.path.join(ROOT, "paper_1512_06637_b200", f)).read()
        assert "import oracle" not in src and "from oracle" not in src
    osrc = open(os.path.join(ROOT, "oracle", "vg_oracle.c")).read()
    assert "vg.h" not in osrc and "csrc" not in re.sub(r"/\*.*?\*/", "", osrc, flags=re.S)
    opy = open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "paper_1512_06637_b200" not in opy.split('"""', 2)[2]


def test_options_round_trip_without_a_gpu():
    import paper_1512_06637_b200 as vg
    old = vg.vg_get_option(vg.OPT_PIPE_MIN_N)
    assert old > 0
    vg.vg_set_option(vg.OPT_PIPE_MIN_N, 12345)
    assert vg.vg_get_option(vg.OPT_PIPE_MIN_N) == 12345
    vg.vg_set_option(vg.OPT_PIPE_MIN_N, old)
    with pytest.raises(vg.VgError):
        vg.vg_set_option(vg.OPT_PIPE_MIN_N, -1)
    assert vg.vg_get_option(vg.OPT_FORM) == vg.FORM_AUTO
    for form in (vg.FORM_DIRECT, vg.FORM_PIPELINED, vg.FORM_STREAMING, vg.FORM_AUTO):
        vg.vg_set_option(vg.OPT_FORM, form)
        assert vg.vg_get_option(vg.OPT_FORM) == form
    with pytest.raises(vg.VgError):
        vg.vg_set_option(vg.OPT_FORM, 4)
    with pytest.raises(vg.VgError):
        vg.vg_set_option(99, 1)


BAD = [
    (0, [5, 5]), (0, [5, -1, 5]), (0, [5, 0, 5]), (0, [5, math.nan, 5]), (0, [5, math.inf, 5]),
    (1, [0]), (1, [-2]), (1, [1, 2]),
    (2, [5, 4, 15, 0, 1]), (2, [-1, 4, 15, 0, 1]), (2, [1, 4, 0, 0, 1]), (2, [1, 4, 15, 0, 0]), (2, [1, 4, 15, 0]),
    (3, [2, 1, 4, 12, 20, 0, 1]), (3, [2, 6, 4, 3, 20, 0, 1]), (3, [2, 6, 4, 12, -20, 0, 1]), (3, [2, 6, 4, 12, 20, 0, -1]),
    (4, [5, 10, 7, 3, 0]), (4, [5, 10, 7, 3]), (4, [0, 10, 7, 3, 15]),
    (5, [0, 6.3, 1, 0, 0, 5]), (5, [0, 6.3, 2, 0, 0, 5, 0, 0, 5]), (5, [0, 6.3, 2, 1, 0, 5, 0, 0, 5]),
    (5, [0, 6.3, 2, 0, 6, 5, 1, 0, 5]), (5, [0, 6.3, 2.5, 0, 0, 5, 1, 0, 5]), (5, [0, 6.3, 3, 0, 0, 5, 1, 0, 5]),
    (5, [0, 6.3, 33] + [v for i in range(33) for v in (float(i), 0.0, 5.0)]), (9, [1, 2, 3]),
]


@pytest.mark.parametrize("kind,params", BAD)
def test_invalid_shape_parameters_are_rejected(kind, params):
    import paper_1512_06637_b200 as vg
    with pytest.raises(vg.VgError) as e:
        vg.Shape(kind, params)
    assert e.value.code in (vg.ERR_PARAM, vg.ERR_ARG)


GOOD = [(0, [5, 5, 5]), (1, [20]), (2, [5, 10, 15, 0, 4 * math.pi / 3]), (2, [0, 10, 15, 0, 7]),
        (3, [2, 6, 4, 12, 20, 0, 2 * math.pi]), (3, [0, 6, 0, 12, 20, 1, 2]), (4, [5, 10, 7, 3, 15]),
        (5, [0, 6.3, 2, -1, 0, 5, 1, 0, 5]),
        (5, [0, 6.3, 32] + [v for i in range(32) for v in (float(i), 0.0, 5.0)])]


@pytest.mark.parametrize("kind,params", GOOD)
def test_valid_shapes_create_without_a_gpu(kind, params):
    import paper_1512_06637_b200 as vg
    s = vg.Shape(kind, params)
    assert vg._lib.vg_shape_kind(s._h) == kind


def test_null_handles_and_zero_tracks():
    import paper_1512_06637_b200 as vg
    lib = vg._lib
    s = vg.Shape(vg.BOX, [5, 5, 5])
    null = C.c_void_p(0)
    assert lib.vg_inside(s._h, null, null, null, 0, null, null) == vg.OK         # n == 0: nothing inspected
    assert lib.vg_distance_to_in(s._h, null, null, null, null, null, null, 1e30, 0, null, null) == vg.OK
    assert lib.vg_inside(null, null, null, null, 0, null, null) == vg.ERR_ARG    # NULL shape
    assert lib.vg_inside(s._h, null, null, null, 4, null, null) == vg.ERR_ARG    # NULL arrays with n > 0
    assert lib.vg_inside(s._h, null, null, null, -1, null, null) == vg.ERR_ARG
    assert b"NULL" in lib.vg_last_error() or b"n < 0" in lib.vg_last_error()
    odd = C.c_void_p(0x1004)
    assert lib.vg_safety_to_in(s._h, odd, odd, odd, 4, odd, null) == vg.ERR_ARG  # not 8-byte aligned
    lib.vg_shape_destroy(null)
    lib.vg_volume_destroy(null)
    assert lib.vg_shape_kind(null) == vg.ERR_ARG


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the behaviour WITHOUT a CUDA device")
def test_compute_calls_fail_loudly_without_a_gpu():
    """No CPU fallback behind the interface (include/vg.h): a launch without a device is VG_ERR_CUDA."""
    import paper_1512_06637_b200 as vg
    lib = vg._lib
    s = vg.Shape(vg.BOX, [5, 5, 5])
    fake = C.c_void_p(0x10000)  # never dereferenced on the host
    assert lib.vg_inside(s._h, fake, fake, fake, 16, fake, C.c_void_p(0)) == vg.ERR_CUDA
    assert lib.vg_last_error() != b""
    x = torch.zeros(4, dtype=torch.float64)
    with pytest.raises(TypeError):
        s.inside(x, x, x)
    with pytest.raises(vg.VgError):
        s.query_host("inside", x, x, x, out=torch.zeros(4, dtype=torch.int32))
    m = vg.Shape(vg.BOX, [10, 10, 10])
    with pytest.raises(vg.VgError):
        vg.Volume(m, [s], [[1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]])  # needs device memory for the table
    with pytest.raises(vg.VgError) as e:
        vg.World([m, s], [-1, 0], [[1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]] * 2)  # the node table as well
    assert e.value.code == vg.ERR_CUDA
    with pytest.raises(vg.VgError) as e:
        vg.World([m, s], [0, 0], [[1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]] * 2)  # validation comes before the device
    assert e.value.code == vg.ERR_PARAM
    # a full-phi polycone is created without its candidate grid (no device to hold it) and stays a valid handle
    pc = vg.Shape(vg.POLYCONE, [0.0, 7.0, 3.0, -1.0, 0.0, 2.0, 0.0, 1.0, 3.0, 2.0, 0.0, 1.0])
    assert lib.vg_shape_kind(pc._h) == vg.POLYCONE


# ------------------------------------------------------------------------------------------ sharding (gloo)

def test_track_ranges_partition_the_tracks():
    from paper_1512_06637_b200.shard import track_range
    for n in (0, 1, 7, 65536, 4194304, 4194305):
        for world in (1, 2, 3, 8):
            r = [track_range(n, g, world) for g in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[g][1] == r[g + 1][0] for g in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        track_range(10, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, n, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import numpy as np
    import oracle as O
    import workloads as W
    from paper_1512_06637_b200.shard import barrier, max_over_ranks, sum_over_ranks, track_range
    sc = W.shape_cases(0)[0]
    t = sc.tracks(n)                       # every rank draws the same seeded tracks ...
    lo, hi = track_range(n, rank, world)   # ... and answers its own contiguous range, no exchange
    s = O.Shape(sc.kind, sc.params)        # (the oracle stands in for the kernels on this CPU-only test)
    part = s.distance_to_in(*[a[lo:hi] for a in t], 1e30)
    barrier()
    tmax = max_over_ranks(0.5 + rank)
    total = sum_over_ranks(hi - lo)
    q.put((rank, lo, hi, part, tmax, total))
    dist.destroy_process_group()


def test_two_ranks_shard_without_exchange_and_reduce_the_timing():
    import numpy as np
    import sys
    sys.path.insert(0, ROOT)
    import oracle as O
    import workloads as W
    n, world = 10001, 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted([q.get(timeout=120) for _ in range(world)], key=lambda r: r[0])
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    sc = W.shape_cases(0)[0]
    t = sc.tracks(n)
    whole = O.Shape(sc.kind, sc.params).distance_to_in(*t, 1e30)
    assert got[0][1] == 0 and got[0][2] == got[1][1] and got[1][2] == n
    assert np.array_equal(np.concatenate([got[0][3], got[1][3]]), whole)
    assert all(r[4] == 1.5 for r in got) and all(r[5] == n for r in got)


# ------------------------------------------------------- host logic: the candidate grids of the polycone safeties

def _polycone_segments(par, face):
    """(r0, z0, r1, z1, bit) of every edge of the (r, z) outline with the bit it has in the masks (vg_params.h): caps 0 / 1,
    outer / inner edge of section k at 2 + 2k / 3 + 2k, the faces of the j-th z step after the sections.  `face`: the
    phi-face grid holds every edge; the surface grid leaves out edges on the axis (both radii 0)."""
    nz = int(par[2])
    pl = [(par[3 + 3 * i], par[4 + 3 * i], par[5 + 3 * i]) for i in range(nz)]
    secs, steps = [], []
    for a, b in zip(pl, pl[1:]):
        if b[0] == a[0]:
            steps.append((len(secs) - 1, a, b))
        else:
            secs.append((a, b))
    segs = []
    for k, (a, b) in enumerate(secs):
        segs.append((a[2], a[0], b[2], b[0], 2 + 2 * k))
        if face or a[1] > 0 or b[1] > 0:
            segs.append((a[1], a[0], b[1], b[0], 3 + 2 * k))
    for j, (_, a, b) in enumerate(steps):
        base = 2 + 2 * len(secs) + 2 * j
        if a[2] != b[2]:
            segs.append((min(a[2], b[2]), a[0], max(a[2], b[2]), a[0], base))
        if a[1] != b[1]:
            segs.append((min(a[1], b[1]), a[0], max(a[1], b[1]), a[0], base + 1))
    segs.append((pl[0][1], pl[0][0], pl[0][2], pl[0][0], 0))
    segs.append((pl[-1][1], pl[-1][0], pl[-1][2], pl[-1][0], 1))
    return segs, secs


@pytest.mark.parametrize("seed", [1, 2, 3, 4])
def test_polycone_candidate_grid_holds_the_nearest_edge_of_every_point(seed):
    """vg_pcon_grid.h builds, per cell of a (rho, z) grid, the set of outline edges that can be nearest to a point of the
    cell.  Checked here on the host (no device): for random points the edge that IS nearest (distances written out in
    numpy) has its bit in the mask of the point's cell, for the surface grid and for the phi-face grid; the per-row section
    index never exceeds the section of any point of the row."""
    import paper_1512_06637_b200 as vg
    rng = np.random.default_rng(seed)
    nz = int(rng.integers(3, 20))
    z = np.sort(rng.uniform(-50, 50, nz)) + np.arange(nz) * 1e-3
    par = [0.3, float(rng.choice([7.0, 4.0])), float(nz)]
    for i in range(nz):
        a = float(rng.choice([0.0, rng.uniform(0, 5)]))
        par += [float(z[i]), a, a + float(rng.uniform(5, 25))]
    if seed % 2 == 0:  # add a z step
        i = nz // 2
        zi, a, b = par[3 + 3 * i: 6 + 3 * i]
        par[6 + 3 * i: 6 + 3 * i] = [zi, 0.0, 0.5 * (a + b) + 6.0]
        par[2] += 1.0
    s = vg.Shape(vg.POLYCONE, par)
    dims = (C.c_int * 2)()
    geom = (C.c_double * 3)()
    vg._lib.vg_debug_polycone_grid.argtypes = [C.c_void_p] * 6
    assert vg._lib.vg_debug_polycone_grid(s._h, None, None, None, geom, dims) == vg.OK
    rows, cols = dims[0], dims[1]
    masks = np.zeros(rows * cols, dtype=np.uint64)
    fmasks = np.zeros(rows * 2 * cols, dtype=np.uint64)
    rowsec = np.zeros(rows, dtype=np.uint8)
    assert vg._lib.vg_debug_polycone_grid(s._h, masks.ctypes.data, fmasks.ctypes.data, rowsec.ctypes.data, geom, dims) == vg.OK
    inv_cr, inv_cz, zg0 = geom[0], geom[1], geom[2]
    R = cols / inv_cr
    for face, m, ncol, ulo in ((False, masks, cols, 0.0), (True, fmasks, 2 * cols, -R)):
        segs, secs = _polycone_segments(par, face)
        n = 200000
        u = rng.uniform(ulo, R, n)
        v = rng.uniform(zg0, zg0 + rows / inv_cz, n)
        d2 = np.full((len(segs), n), np.inf)
        for j, (r0, z0, r1, z1, _) in enumerate(segs):
            eu, ev = r1 - r0, z1 - z0
            t = np.clip(((u - r0) * eu + (v - z0) * ev) / (eu * eu + ev * ev), 0, 1)
            d2[j] = (u - r0 - t * eu) ** 2 + (v - z0 - t * ev) ** 2
        nearest = np.argmin(d2, axis=0)
        bits = np.array([sg[4] for sg in segs], dtype=np.uint64)[nearest]
        cell = np.minimum((v - zg0) * inv_cz, rows - 1).astype(int) * ncol + np.minimum((u - ulo) * inv_cr, ncol - 1).astype(int)
        assert np.all((m[cell] >> bits) & np.uint64(1) == 1), "a nearest edge is missing from its cell's mask (face=%s)" % face
        pop = np.array([bin(int(w)).count("1") for w in m])
        assert pop.min() >= 1 and pop.mean() < 0.5 * len(segs)  # every cell has a candidate; the masks do prune
    planes = np.array([sc[0][0] for sc in secs[1:]])
    zrow = zg0 + np.arange(rows) / inv_cz
    assert np.all(rowsec <= np.array([(planes <= zz).sum() for zz in zrow]))
    assert np.all(rowsec >= np.array([(planes <= zz - 1e-3).sum() for zz in zrow]))


# ------------------------------------------------------------------- host logic: flattening of a CSG tree

def test_boolean_trees_are_flattened_in_tree_order_with_composed_transforms():
    """vg_boolean_create turns a tree into primitives + transforms + a postfix program (no device needed).  Checked
    against the same tree walked in Python: primitive kinds in tree order, every transform == the product of the
    placements on the way down (4x4 matrices in numpy), and the program evaluates to the tree's set expression on all
    2^n assignments of its primitives."""
    import paper_1512_06637_b200 as vg
    import workloads as W
    vg._lib.vg_debug_boolean_program.argtypes = [C.c_void_p] * 5
    for cc in W.csg_cases() + [W.CsgCase("two", ("op", W.SUBTRACTION, ("leaf", W.BOX, [1.0, 2.0, 3.0]), ("leaf", W.ORB, [1.5]),
                                                 W.placement(W.quaternion_to_matrix((0.5, 0.5, 0.5, 0.5)), (0.1, 0.2, 0.3))), (0, 0, 0), (1, 1, 1), 1)]:
        shape = cc.build(vg)
        kinds = (C.c_int * 8)()
        xf = (C.c_double * 96)()
        prog = (C.c_ubyte * 16)()
        nprog = C.c_int(0)
        nleaf = vg._lib.vg_debug_boolean_program(shape._h, kinds, xf, prog, C.byref(nprog))
        want = []  # (kind, 4x4 frame of the tree -> frame of the primitive), tree order

        def walk(t, pre):
            if t[0] == "leaf":
                want.append((t[1], pre))
                return ("leaf", len(want) - 1)
            a = walk(t[2], pre)
            b = walk(t[3], np.vstack([np.asarray(t[4]).reshape(3, 4), [0, 0, 0, 1]]) @ pre)
            return ("op", t[1], a, b)
        expr = walk(cc.tree, np.eye(4))
        assert nleaf == len(want) and [kinds[i] for i in range(nleaf)] == [k for k, _ in want]
        X = np.array(xf[:12 * nleaf]).reshape(nleaf, 3, 4)
        for i, (_, M) in enumerate(want):
            assert np.max(np.abs(X[i] - M[:3])) < 1e-14, (cc.name, i)

        def ev(e, bits):
            if e[0] == "leaf":
                return bool((bits >> e[1]) & 1)
            a, b = ev(e[2], bits), ev(e[3], bits)
            return {W.UNION: a or b, W.INTERSECTION: a and b, W.SUBTRACTION: a and not b}[e[1]]
        for bits in range(1 << nleaf):
            st = []
            for tok in prog[:nprog.value]:
                if tok < 0x80:
                    st.append(bool((bits >> tok) & 1))
                else:
                    b, a = st.pop(), st.pop()
                    st.append({W.UNION: a or b, W.INTERSECTION: a and b, W.SUBTRACTION: a and not b}[tok & 0x7f])
            assert len(st) == 1 and st[0] == ev(expr, bits), (cc.name, bits)
    assert vg._lib.vg_debug_boolean_program(vg.Shape(vg.BOX, [1, 1, 1])._h, None, None, None, None) == vg.ERR_ARG
