#!/usr/bin/env python
"""bench.py -- tracks/s per query on one B200 (BASELINE.json `metric`) for the geometry hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-detail]

A "step" is one pass of the hot path over one batch of synthetic tracks of BASELINE.json configs[1] (tube segment
rmin 5, rmax 10, dz 15, phi 0..4pi/3, N = 1,048,576 tracks): Inside, DistanceToIn, DistanceToOut, SafetyToIn and
SafetyToOut, five kernel launches through the C ABI.  `value` = tracks x queries / second with the tracks resident
in HBM; every launch reads a different copy of the batch (rotating buffer sets whose total size is several times
the 126 MB L2), so no launch finds its inputs in L2.  The K timed steps are replays of CUDA graphs captured from
the same C-ABI calls (the launches are microseconds long; eager launches would time the Python interpreter).
`e2e` is the same step through the host-buffer entry points (pinned host arrays in, host arrays out, copies
inside the timed region).  `detail` adds every (config, shape, query) of BASELINE.json with its roofline fraction.
`--impl reference` times the oracle (oracle/, plain scalar CPU code) on the host cores for the same step.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402  (seeded input generators; no arithmetic of the method)

METRIC = "tracks/sec per query per shape (1 B200) and fraction of HBM / FP64 roofline"
UNIT = "track-queries/s"
# algorithmic bytes per track: SoA inputs read once + one result written once
BYTES = {"inside": 24 + 4, "safety_to_in": 24 + 8, "safety_to_out": 24 + 8, "distance_to_in": 48 + 8,
         "distance_to_out": 48 + 8, "compute_step": 48 + 12, "all": 48 + 4 + 4 * 8}
BYTES.update({"world_locate": 24 + 4, "world_step": 48 + 4 + 8 + 4, "world_safety": 24 + 4 + 8})
L2_BYTES = 126e6
HBM_FALLBACK_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(solid, query, n):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of that kernel at that N, from the committed summary of
    the last `ncu --set full` capture (profiles/traffic.csv); None when the capture has no such row."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for line in f:
                c = line.strip().split(",")
                if len(c) >= 7 and c[1] == solid and c[2] == query and c[3] == str(n):
                    return {"bytes": int(c[4]) + int(c[5]), "dram_read": int(c[4]), "dram_write": int(c[5]),
                            "capture": "profiles/%s_full_capture.md" % c[6],
                            "note": "results still sit in the 126 MB L2 when the kernel ends, so DRAM writes read low"}
    except OSError:
        pass
    return None


# ------------------------------------------------------------------------------------------- clock sampler

class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the GPU is under the bench load."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thread = index, [], None, None
        self.marks = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()

    def summary(self, t0, t1, load0, load1):
        def pick(a, b):
            return [r for ts, r in self.rows if a <= ts <= b and len(r) >= 7]
        rows, window = pick(t0, t1), "timed region"
        if len(rows) < 3:
            rows, window = pick(load0, load1), "bench load phase (timed region shorter than the sampling period)"
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "window": "nvidia-smi unavailable"}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "reasons": reasons,
                "power_w_max": max(float(r[2]) for r in rows), "samples": len(rows), "window": window}


# ------------------------------------------------------------------------------------ device-resident cases

class Case:
    """One solid (or the navigation volume) with its seeded tracks resident in HBM as `nsets` rotating copies."""

    def __init__(self, vg, torch, name, n, queries, seed_shift=0, shape=None, nav=None, world=None, boolean=None, csg=None):
        self.vg, self.torch, self.name, self.n, self.queries = vg, torch, name, int(n), tuple(queries)
        dev = torch.device("cuda", torch.cuda.current_device())
        self.nodes = None
        if world is not None:
            self.kind = "world"
            shapes = [vg.Shape(k, p) for k, p in zip(world.kinds, world.params)]
            self.handle = vg.World(shapes, world.parents, world.xforms)

            def band(x, y, z):  # outside the world, or in the surface band of any node (library's own queries)
                d = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (x, y, z)]
                nd = self.handle.locate(*d)
                s = self.handle.safety(torch.clamp(nd, min=0), *d)
                return ((nd < 0) | (s < W.SURFACE_BAND)).cpu().numpy()
        elif csg is not None:  # a nested boolean (reading R31)
            self.kind = "boolean"
            self.handle = csg.build(vg)
            seed, center, half = csg.seed + seed_shift, csg.center, csg.half
            leaves = []  # (primitive handle, 4x4 frame of the tree -> frame of the primitive), composed here for the band only

            def walk(t, pre):
                if t[0] == "leaf":
                    leaves.append((vg.Shape(t[1], t[2]), pre))
                    return
                walk(t[2], pre)
                walk(t[3], np.vstack([np.asarray(t[4]).reshape(3, 4), [0, 0, 0, 1]]) @ pre)
            walk(csg.tree, np.eye(4))

            def band(x, y, z):  # clear of the surface of every primitive of the tree (library's own safeties)
                bad = np.zeros(len(x), dtype=bool)
                for h, M in leaves:
                    L = M[:3, :3] @ np.stack([x, y, z]) + M[:3, 3:4]
                    bad |= np.abs(self._gpu3(h.safety_to_in, L[0], L[1], L[2])) < W.SURFACE_BAND
                return bad
        elif boolean is not None:
            self.kind = "boolean"
            a, b = vg.Shape(boolean.kind_a, boolean.par_a), vg.Shape(boolean.kind_b, boolean.par_b)
            self.handle = vg.Boolean(boolean.op, a, b, boolean.xform)
            seed, center, half = boolean.seed + seed_shift, boolean.center, boolean.half
            M = np.asarray(boolean.xform).reshape(3, 4)

            def band(x, y, z):  # clear of both operands' surfaces (library's own safeties)
                L = M[:, :3] @ np.stack([x, y, z]) + M[:, 3:4]
                return (np.abs(self._gpu3(a.safety_to_in, x, y, z)) < W.SURFACE_BAND) | \
                       (np.abs(self._gpu3(b.safety_to_in, L[0], L[1], L[2])) < W.SURFACE_BAND)
        elif nav is not None:
            self.kind = "navigator"
            mother = vg.Shape(nav.mother_kind, nav.mother_params)
            daughters = [vg.Shape(k, p) for k, p in zip(nav.daughter_kinds, nav.daughter_params)]
            self.handle = vg.Volume(mother, daughters, nav.xforms)
            seed, center, half = nav.seed + seed_shift, nav.center, nav.half
            # surface-band rejection with the library's own safety (the product path never touches oracle/)
            band = lambda x, y, z: self._gpu3(self.handle.safety, x, y, z) < W.SURFACE_BAND
        else:
            self.kind = W.KIND_NAME[shape.kind]
            self.handle = vg.Shape(shape.kind, shape.params)
            seed, center, half = shape.seed + seed_shift, shape.center, shape.half
            band = lambda x, y, z: np.abs(self._gpu3(self.handle.safety_to_in, x, y, z)) < W.SURFACE_BAND
        self.host = world.tracks(self.n, band) if world is not None else W.draw_tracks(seed, self.n, center, half, band)
        per_set = 48 * self.n
        self.nsets = int(min(16, max(2, -(-int(4 * L2_BYTES) // per_set))))
        self.cold = self.nsets * per_set >= 2 * L2_BYTES
        base = [torch.from_numpy(a).to(dev) for a in self.host]
        self.sets = [base] + [[a.clone() for a in base] for _ in range(self.nsets - 1)]
        self.outd = [torch.empty(self.n, dtype=torch.float64, device=dev) for _ in range(self.nsets)]
        self.outi = [torch.empty(self.n, dtype=torch.int32, device=dev) for _ in range(self.nsets)]
        self.out4 = None  # four more result arrays per set, allocated on the first fused launch
        self.cursor = 0
        if world is not None:  # the node of every track, as vg_world_locate returns it
            self.nodes = [self.handle.locate(*st[:3]) for st in self.sets]

    def _gpu3(self, fn, x, y, z):
        t = self.torch
        d = [t.from_numpy(np.ascontiguousarray(a)).cuda() for a in (x, y, z)]
        return fn(*d).cpu().numpy()

    def launch(self, q):
        """One C-ABI call of query `q` on the next buffer set (enqueue only)."""
        k = self.cursor
        self.cursor = (k + 1) % self.nsets
        s = self.sets[k]
        if q == "all":  # the fused five-query call (vg_query_all)
            if self.out4 is None:
                self.out4 = [[self.torch.empty_like(self.outd[0]) for _ in range(3)] for _ in range(self.nsets)]
            self.handle.query_all(*s, W.STEP_MAX, out=[self.outi[k], self.outd[k]] + self.out4[k])
        elif q == "world_locate":
            self.handle.locate(*s[:3], out=self.outi[k])
        elif q == "world_step":
            if self.out4 is None:
                self.out4 = [self.torch.empty_like(self.outi[0]) for _ in range(self.nsets)]
            self.handle.step(self.nodes[k], *s, step_max=W.STEP_MAX, step=self.outd[k], next=self.out4[k])
        elif q == "world_safety":
            self.handle.safety(self.nodes[k], *s[:3], out=self.outd[k])
        elif q == "compute_step":
            self.handle.compute_step(*s, step_max=W.STEP_MAX, step=self.outd[k], hit=self.outi[k])
        elif q == "inside":
            self.handle.inside(*s[:3], out=self.outi[k])
        elif q in ("distance_to_in", "distance_to_out"):
            self.handle.query(q, *s, step_max=W.STEP_MAX, out=self.outd[k])
        else:
            self.handle.query(q, *s[:3], out=self.outd[k])

    def step(self):
        for q in self.queries:
            self.launch(q)


def capture_steps(torch, case, with_events):
    """CUDA graphs of one step each, as many as it takes for the buffer-set rotation to come round; every kernel
    node is bracketed by external timing events when the torch build supports them."""
    nq = len(case.queries)
    ngraphs = case.nsets  # after nsets steps every launch position has used every set
    graphs, events = [], []
    case.cursor = 0
    case.step()  # eager warm-up before capture (lazy attribute / occupancy queries happen here)
    torch.cuda.synchronize()
    case.cursor = 0
    for _ in range(ngraphs):
        g = torch.cuda.CUDAGraph()
        ev = [torch.cuda.Event(enable_timing=True, external=True) for _ in range(nq + 1)] if with_events else []
        with torch.cuda.graph(g):
            for j, q in enumerate(case.queries):
                if with_events:
                    ev[j].record()
                case.launch(q)
            if with_events:
                ev[nq].record()
        graphs.append(g)
        events.append(ev)
    return graphs, events


def time_query_alone(torch, case, q, min_ms=30.0, hot=False):
    """Average duration of one launch of `q` (cold inputs): a graph of nsets launches over the rotating sets,
    replayed between two CUDA events on the launching stream until >= min_ms have been timed.  hot = True: every
    launch reads the SAME buffer set (what the paper's 5000 repetitions on fixed particles did): the
    batch stays in the 126 MB L2 if it fits."""
    case.cursor = 0
    case.launch(q)
    torch.cuda.synchronize()
    case.cursor = 0
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        for _ in range(case.nsets):
            if hot:
                case.cursor = 0
            case.launch(q)
    for _ in range(3):
        g.replay()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps, ms = 4, 0.0
    while True:
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            g.replay()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        if ms >= min_ms or reps >= 4096:
            break
        reps *= 4
    return ms * 1e-3 / (reps * case.nsets)


# ------------------------------------------------------------------------------------------ the oracle legs

def oracle_step(O, shape, tracks, queries):
    for q in queries:
        if q in ("distance_to_in", "distance_to_out"):
            getattr(shape, q)(*tracks, W.STEP_MAX)
        else:
            getattr(shape, q)(*tracks[:3])


def cpu_baseline(seconds=10.0):
    """The oracle as it stands, timed on this box's host cores on the tracks of configs[1] (all five queries)."""
    import oracle as O
    sc = W.shape_cases(1)[0]
    s = O.Shape(sc.kind, sc.params)
    t = sc.tracks(sc.sizes[-1], band=lambda x, y, z: np.abs(s.sdf(x, y, z)) < W.SURFACE_BAND)
    oracle_step(O, s, t, sc.queries)  # warm-up (thread pool, page faults)
    reps, t0 = 0, time.perf_counter()
    while True:
        oracle_step(O, s, t, sc.queries)
        reps += 1
        el = time.perf_counter() - t0
        if el >= seconds:
            break
    return {"value": len(sc.queries) * len(t[0]) * reps / el, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
            "sample": "%d repetitions of the five queries over all %d tracks of configs[1] (%.1f s of wall time, "
                      "gcc -O2 -ffp-contract=off, OpenMP static)" % (reps, len(t[0]), el)}


# ---- the paper's own measurement (Fig. 4): DistanceToOut on a Box and a Tube, particles placed at
# random INSIDE the body "escaping" from it, N = 10^3, 10^4, 10^5 on the x axis, every point repeated many times, speed
# relative to a serial CPU code.  The figure's values did not survive the text extraction, so this is the
# same protocol measured here, not a comparison with the paper's curve.

FIG4_N = (1000, 10000, 100000)


def fig4_cases():
    box, tube = W.shape_cases(0)[0], W.shape_cases(1)[0]
    return [("box", box.kind, box.params, (0, 0, 0), tuple(box.params)),
            ("tube", tube.kind, tube.params, (0, 0, 0), (tube.params[1], tube.params[1], tube.params[2]))]


def fig4_cpu(seconds_per_point=0.25):
    """Serial-CPU leg of the Fig. 4 protocol: the oracle on ONE thread (part of the cpu_baseline object)."""
    import oracle as O
    nthreads = O.num_threads()
    O.set_num_threads(1)
    rows = []
    try:
        for name, kind, par, c, h in fig4_cases():
            s = O.Shape(kind, par)
            for n in FIG4_N:
                t = W.draw_tracks(W.config_seed(9) + n, n, c, h, lambda x, y, z: s.sdf(x, y, z) > -W.SURFACE_BAND)
                s.distance_to_out(*t, W.STEP_MAX)
                reps, t0 = 0, time.perf_counter()
                while True:
                    s.distance_to_out(*t, W.STEP_MAX)
                    reps += 1
                    el = time.perf_counter() - t0
                    if el >= seconds_per_point:
                        break
                rows.append({"shape": name, "n": n, "us_per_call": el * 1e6 / reps, "threads": 1})
    finally:
        O.set_num_threads(nthreads)
    return rows


def fig4_gpu(vg, torch, reps=5000):
    """GPU legs: device-resident tracks, `reps` back-to-back launches as one CUDA graph (the paper repeated every point
    5000 times on the same particles: a hot-cache number by construction); and the host-fed call (pinned host arrays in,
    pinned result out) that includes both transfers, which is what the paper's GPU curve paid at small N."""
    rows = []
    for name, kind, par, c, h in fig4_cases():
        sg = vg.Shape(kind, par)

        def outside(x, y, z):
            d = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (x, y, z)]
            return (sg.safety_to_in(*d) > -W.SURFACE_BAND).cpu().numpy()

        for n in FIG4_N:
            host = W.draw_tracks(W.config_seed(9) + n, n, c, h, outside)
            dev = [torch.from_numpy(a).cuda() for a in host]
            out = torch.empty(n, dtype=torch.float64, device="cuda")
            sg.distance_to_out(*dev, W.STEP_MAX, out=out)
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            per_graph = 100
            with torch.cuda.graph(g):
                for _ in range(per_graph):
                    sg.distance_to_out(*dev, W.STEP_MAX, out=out)
            g.replay()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(reps // per_graph):
                g.replay()
            e1.record()
            torch.cuda.synchronize()
            us_dev = e0.elapsed_time(e1) * 1e3 / (reps // per_graph * per_graph)
            assert bool((out > 0).all()), "Fig. 4 protocol: every particle starts inside and escapes"
            hblock = torch.empty((6, n), dtype=torch.float64).pin_memory()  # one [6][n] host basket
            for i, a in enumerate(host):
                hblock[i].copy_(torch.from_numpy(a))
            hp = [hblock[i] for i in range(6)]
            hout = torch.empty(n, dtype=torch.float64).pin_memory()
            for _ in range(5):
                sg.query_host("distance_to_out", *hp, step_max=W.STEP_MAX, out=hout)
            k, w0 = 200, time.perf_counter()
            for _ in range(k):
                sg.query_host("distance_to_out", *hp, step_max=W.STEP_MAX, out=hout)
            us_host = (time.perf_counter() - w0) * 1e6 / k
            rows.append({"shape": name, "query": "distance_to_out", "n": n, "repetitions": reps // per_graph * per_graph,
                         "device_resident_us_per_launch": us_dev, "device_resident_tracks_per_s": n / us_dev * 1e6,
                         "host_fed_us_per_call": us_host, "host_fed_tracks_per_s": n / us_host * 1e6})
    return rows


def run_reference(args, rank):
    """--impl reference: the oracle on the host cores, same config / metric / unit (rank 0 only)."""
    if rank != 0:
        return
    import oracle as O
    sc = W.shape_cases(1)[0]
    s = O.Shape(sc.kind, sc.params)
    full = sc.tracks(sc.sizes[-1], band=lambda x, y, z: np.abs(s.sdf(x, y, z)) < W.SURFACE_BAND)
    probe = [a[:65536] for a in full]
    oracle_step(O, s, probe, sc.queries)
    t0 = time.perf_counter()
    oracle_step(O, s, probe, sc.queries)
    per_track = (time.perf_counter() - t0) / 65536
    budget = 120.0  # seconds for the whole --steps + --warmup run
    n = int(min(len(full[0]), max(4096, budget / ((args.steps + args.warmup) * per_track))))
    t = [np.ascontiguousarray(a[:n]) for a in full]
    for _ in range(args.warmup):
        oracle_step(O, s, t, sc.queries)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_step(O, s, t, sc.queries)
    el = time.perf_counter() - t0
    value = len(sc.queries) * n * args.steps / el
    sample = "each step = the five queries over the first %d of the %d tracks of configs[1]" % (n, len(full[0]))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": el * 1e3 / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[1]: tube segment rmin=5 rmax=10 dz=15 phi 0..4pi/3, five queries", "n_tracks": n,
                       "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------- our arm

# Algorithmic FP64 operations per track of the ALU-bound rows (DESIGN.md sec. 6 derives them from the formulas:
# +, -, x, compare/min/max/select = 1, FMA = 2, divide / sqrt = 1), used for `bound: "alu"` entries of `detail`.
ALGO_FLOP = {("polycone", "distance_to_in"): 677, ("polycone", "safety_to_in"): 394, ("navigator", "compute_step"): 5518}


def roofline_entry(shape_kind, q, n, seconds, hbm_peak, fp64_fma_per_s):
    gbs = BYTES[q] * n / seconds / 1e9
    e = {"tracks_per_s": n / seconds, "us_per_launch": seconds * 1e6, "hbm_gbs": gbs, "hbm_frac": gbs / hbm_peak}
    flop = ALGO_FLOP.get((shape_kind, q))
    if flop:
        e["bound"] = "alu"
        e["fp64_tflops"] = flop * n / seconds / 1e12
        e["fp64_frac"] = e["fp64_tflops"] * 1e12 / (2.0 * fp64_fma_per_s)
    else:
        e["bound"] = "hbm"
    return e


def launch_floor(vg, torch, per_graph=64, reps=50):
    """Duration of one EMPTY kernel launch in a graph of back-to-back launches (vg_probe_empty_launch): the floor under
    any single launch, whatever it computes (the latency-adjusted bound of the small-N rows)."""
    vg.vg_probe_empty_launch(4)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        vg.vg_probe_empty_launch(per_graph)
    g.replay()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        g.replay()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e-3 / (reps * per_graph)


def detail_sweep(vg, torch, hbm_peak, fma_rate, main_case):
    """Every (config, shape, query) of BASELINE.json configs[0..4], each launch timed alone on cold inputs."""
    rows = []
    floor_s = launch_floor(vg, torch)
    plan = []
    for k in (0, 1, 2, 3):
        for i, sc in enumerate(W.shape_cases(k)):
            for n in sc.sizes:
                plan.append((k, sc, n))
    for k, sc, n in plan:
        case = main_case if (k == 1) else Case(vg, torch, sc.name, n, sc.queries, shape=sc)
        for q in sc.queries:
            sec = time_query_alone(torch, case, q)
            e = roofline_entry(case.kind, q, n, sec, hbm_peak, fma_rate)
            e.update({"config": k, "shape": sc.name, "query": q, "n": n, "cold_inputs": case.cold})
            if n <= 262144:  # launch-bound sizes: the bound a single launch can reach is max(bytes / BW, empty launch)
                ideal = max(BYTES[q] * n / (hbm_peak * 1e9), floor_s)
                e.update({"empty_launch_us": floor_s * 1e6, "latency_adjusted_bound_us": ideal * 1e6,
                          "latency_adjusted_frac": ideal / sec})
            rows.append(e)
        if len(sc.queries) == 5 and sc.kind != W.POLYCONE:  # the fused five-query kernel on the same tracks
            sec = time_query_alone(torch, case, "all")
            e = roofline_entry(case.kind, "all", n, sec, hbm_peak, fma_rate)
            e.update({"config": k, "shape": sc.name, "query": "all five (vg_query_all, one kernel)", "n": n, "cold_inputs": case.cold,
                      "track_queries_per_s": 5 * n / sec})
            rows.append(e)
        if case is not main_case:
            del case
            torch.cuda.empty_cache()
    nav = W.navigator_case()
    case = Case(vg, torch, "navigator", nav.sizes[-1], ("compute_step",), nav=nav)
    sec = time_query_alone(torch, case, "compute_step")
    e = roofline_entry("navigator", "compute_step", case.n, sec, hbm_peak, fma_rate)
    e.update({"config": 4, "shape": "box(100)+64 daughters", "query": "compute_step", "n": case.n, "cold_inputs": case.cold})
    rows.append(e)
    del case
    torch.cuda.empty_cache()
    # polycone variants -- the configs[3] polycone cut to phi in [0, 4 pi / 3], and one with two z steps
    pc = W.polycone_params(W.config_seed(3, 0))
    variants = [("polycone_phi_segment", [0.0, 4.0 * np.pi / 3.0] + pc[2:]), ("polycone_z_steps", W.STEPPED_POLYCONE)]
    for vname, vpar in variants:
        sc = W.ShapeCase(3, vname, W.POLYCONE, vpar, *W._scaled(W.POLYCONE, vpar), W.config_seed(3, 3), [4194304],
                         ("distance_to_in", "safety_to_in"))
        case = Case(vg, torch, sc.name, 4194304, sc.queries, shape=sc)
        for q in sc.queries:
            sec = time_query_alone(torch, case, q)
            e = roofline_entry("polycone_variant", q, case.n, sec, hbm_peak, fma_rate)
            e.update({"config": "8(f) f2", "shape": vname, "query": q, "n": case.n, "cold_inputs": case.cold, "bound": "alu"})
            rows.append(e)
        del case
        torch.cuda.empty_cache()
    # boolean solids of two primitives (one of each operation)
    for bc in [b for b in W.boolean_cases() if b.name in ("tube_union_box", "cone_intersection_orb", "box_minus_tube")]:
        case = Case(vg, torch, bc.name, 4194304, W.QUERIES5, boolean=bc)
        for q in case.queries:
            sec = time_query_alone(torch, case, q)
            e = roofline_entry("boolean", q, case.n, sec, hbm_peak, fma_rate)
            e.update({"config": "8(f) f2", "shape": bc.name, "query": q, "n": case.n, "cold_inputs": case.cold})
            if q.startswith("distance"):
                e["bound"] = "alu"
            rows.append(e)
        del case
        torch.cuda.empty_cache()
    cc = [c for c in W.csg_cases() if c.name == "twice_drilled_block_in_a_sphere"][0]  # a tree of four primitives (R31)
    case = Case(vg, torch, cc.name, 4194304, W.QUERIES5, csg=cc)
    for q in case.queries:
        sec = time_query_alone(torch, case, q)
        e = roofline_entry("boolean", q, case.n, sec, hbm_peak, fma_rate)
        e.update({"config": "8(f) f2", "shape": "csg tree: " + cc.name, "query": q, "n": case.n, "cold_inputs": case.cold, "bound": "alu"})
        rows.append(e)
    del case
    torch.cuda.empty_cache()
    # the three-level tree of placed solids (193 nodes), every track in its own node
    wc = W.world_case()
    case = Case(vg, torch, "world", wc.sizes[-1], ("world_locate", "world_step", "world_safety"), world=wc)
    for q in case.queries:
        sec = time_query_alone(torch, case, q)
        e = roofline_entry("world", q, case.n, sec, hbm_peak, fma_rate)
        e.update({"config": "8(f) f3", "shape": "box(100) > 64 daughters > 128 grand-daughters", "query": q, "n": case.n,
                  "cold_inputs": case.cold, "bound": "alu", "track_order": "as drawn (nodes mixed within a warp)"})
        rows.append(e)
    # the same tracks in basket order (sorted by node, what the paper's scheduler hands to the geometry)
    for k in range(case.nsets):
        order = torch.argsort(case.nodes[k].to(torch.int64), stable=True)
        case.sets[k] = [a[order].contiguous() for a in case.sets[k]]
        case.nodes[k] = case.nodes[k][order].contiguous()
    for q in case.queries:
        sec = time_query_alone(torch, case, q)
        e = roofline_entry("world", q, case.n, sec, hbm_peak, fma_rate)
        e.update({"config": "8(f) f3", "shape": "box(100) > 64 daughters > 128 grand-daughters", "query": q, "n": case.n,
                  "cold_inputs": case.cold, "bound": "alu", "track_order": "sorted by node (baskets)"})
        rows.append(e)
    return rows


def run_profile(args):
    """--profile: launch every kernel of configs[1..4] (largest N) `--steps` times eagerly and exit: the command
    ncu wraps for the per-kernel captures under profiles/ (no timing is reported from this mode)."""
    import torch
    torch.cuda.set_device(0)
    import paper_1512_06637_b200 as vg
    if args.pipe_min_n is not None:
        vg.vg_set_option(vg.OPT_PIPE_MIN_N, args.pipe_min_n)
    if args.form is not None:
        vg.vg_set_option(vg.OPT_FORM, {"auto": vg.FORM_AUTO, "direct": vg.FORM_DIRECT, "pipelined": vg.FORM_PIPELINED, "streaming": vg.FORM_STREAMING}[args.form])
    if args.no_pdl:
        vg.vg_set_option(vg.OPT_PDL, 0)
    cases = []
    for k in (1, 2, 3):
        for sc in W.shape_cases(k):
            cases.append(Case(vg, torch, sc.name, min(sc.sizes[-1], 4194304), sc.queries, shape=sc))
    nav = W.navigator_case()
    cases.append(Case(vg, torch, "navigator", nav.sizes[-1], ("compute_step",), nav=nav))
    wc = W.world_case()
    cases.append(Case(vg, torch, "world", wc.sizes[-1], ("world_locate", "world_step", "world_safety"), world=wc))
    bc = [b for b in W.boolean_cases() if b.name == "box_minus_tube"][0]
    cases.append(Case(vg, torch, bc.name, 4194304, W.QUERIES5, boolean=bc))
    stepped = W.ShapeCase(3, "polycone_step", W.POLYCONE, W.STEPPED_POLYCONE, *W._scaled(W.POLYCONE, W.STEPPED_POLYCONE),
                          W.config_seed(3, 2), [4194304], ("distance_to_in", "safety_to_in"))
    cases.append(Case(vg, torch, stepped.name, 4194304, stepped.queries, shape=stepped))
    torch.cuda.synchronize()
    torch.cuda.profiler.start()  # ncu --profile-from-start off: the set-up launches (surface-band rejection) are skipped
    for _ in range(args.steps):
        for c in cases:
            c.step()
            if len(c.queries) == 5 and c.kind not in ("polycone", "boolean"):
                c.launch("all")  # the fused five-query kernel
    torch.cuda.synchronize()
    torch.cuda.profiler.stop()
    print(json.dumps({"profile_mode": True, "launches": vg.vg_launch_count()}))


def run_ours(args, rank, world, local_rank):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback "
                         "(use --impl reference for the oracle on the host cores)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    import paper_1512_06637_b200 as vg
    from paper_1512_06637_b200.shard import barrier, max_over_ranks, sum_over_ranks
    if args.pipe_min_n is not None:
        vg.vg_set_option(vg.OPT_PIPE_MIN_N, args.pipe_min_n)
    if args.form is not None:
        vg.vg_set_option(vg.OPT_FORM, {"auto": vg.FORM_AUTO, "direct": vg.FORM_DIRECT, "pipelined": vg.FORM_PIPELINED, "streaming": vg.FORM_STREAMING}[args.form])
    if args.no_pdl:
        vg.vg_set_option(vg.OPT_PDL, 0)

    hbm_peak, hbm_src = measured_peaks()
    sampler = ClockSampler(local_rank)
    sampler.start()
    load0 = time.time()
    fma_rate = 1.0  # measured below, AFTER the timed region and the per-query timings: the probe drives the FP64 pipe at full
                    # power for ~70 ms and would leave the board power-capped for the measurements that matter

    # weak scaling: every rank owns one full configs[1] batch (its own seed); no data-path collective
    sc = W.shape_cases(1)[0]
    case = Case(vg, torch, sc.name, sc.sizes[-1], sc.queries, seed_shift=1000 * rank, shape=sc)
    graphs, _ = capture_steps(torch, case, False)
    for i in range(max(args.warmup, 3)):
        graphs[i % len(graphs)].replay()
    torch.cuda.synchronize()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    e0.record()
    for i in range(args.steps):
        graphs[i % len(graphs)].replay()
    e1.record()
    torch.cuda.synchronize()
    t1 = time.time()
    barrier()
    ms = max_over_ranks(e0.elapsed_time(e1), "cuda")
    tracks_all = sum_over_ranks(case.n, "cuda")
    nq = len(case.queries)
    value = tracks_all * nq * args.steps / (ms * 1e-3)

    # per-kernel durations, same process, right after the timed region: event-record nodes between the kernel nodes
    # of the timed graphs cost ~5 us each (measured) and would distort `value`, so every query is timed alone as a
    # graph of nsets back-to-back launches (cold inputs) between two CUDA events on the launching stream
    kernel_timing = "each query alone: graph of %d back-to-back launches over the rotating buffer sets between two CUDA events" % case.nsets
    per_q = {q: time_query_alone(torch, case, q) for q in case.queries}

    per_query = {q: roofline_entry(case.kind, q, case.n, per_q[q], hbm_peak, fma_rate) for q in case.queries}
    for q in case.queries:  # the hot variant: same buffers every launch, the 48 MB batch stays in L2
        hot_s = time_query_alone(torch, case, q, hot=True)
        per_query[q]["hot_us_per_launch"] = hot_s * 1e6
        per_query[q]["hot_tracks_per_s"] = case.n / hot_s
    dom = max(case.queries, key=lambda q: per_q[q])
    kname = ("query_stream_kernel<TubeT<hollow, wide phi>, %s>" if dom == "distance_to_in" else "query_kernel<TubeT<hollow, wide phi>, %s>") % dom
    roof = {"bound": "hbm", "kernel": kname, "achieved": per_query[dom]["hbm_gbs"],
            "peak": hbm_peak, "unit": "GB/s", "frac": per_query[dom]["hbm_gbs"] / hbm_peak, "peak_source": hbm_src,
            "traffic": (ncu_traffic("Tube", dom, case.n) or {}).get("bytes"), "traffic_detail": ncu_traffic("Tube", dom, case.n),
            "algorithmic_bytes_per_launch": BYTES[dom] * case.n,
            "us_per_launch": per_q[dom] * 1e6, "share_of_step": per_q[dom] / sum(per_q.values()),
            "sum_of_kernels_us": sum(per_q.values()) * 1e6,
            "kernel_timing": kernel_timing,
            "step_hbm_frac": sum(BYTES[q] for q in case.queries) * case.n / (ms * 1e-3 / args.steps) / 1e9 / hbm_peak}

    # the same step as ONE fused kernel (vg_query_all): 48 B read + 36 B written per track instead of 168 + 36
    fused_s = time_query_alone(torch, case, "all")
    fused = {"us_per_step": fused_s * 1e6, "value": nq * case.n / fused_s, "unit": UNIT, "api": "vg_query_all (one kernel, five results)",
             "hbm_gbs": BYTES["all"] * case.n / fused_s / 1e9, "hbm_frac": BYTES["all"] * case.n / fused_s / 1e9 / hbm_peak,
             "algorithmic_bytes_per_track": BYTES["all"], "speedup_vs_five_launches": sum(per_q.values()) / fused_s,
             "note": "reported beside `value`, which stays the five per-query launches BASELINE.json's metric names"}

    # end to end: pinned host arrays -> C-ABI host entry point -> pinned host results, copies inside the timed region.
    # The call a user makes for one step over host tracks is vg_query_all_host (the tracks cross the host link once);
    # the five single-query host calls are timed beside it.
    # the host basket is ONE pinned [6][n] allocation (and the four FP64 results one [4][n]): equally spaced arrays cross
    # the link as one strided copy per chunk (vg_host.cu); separately allocated arrays work too, with six copies per chunk
    hblock = torch.empty((6, case.n), dtype=torch.float64).pin_memory()
    for i, a in enumerate(case.host):
        hblock[i].copy_(torch.from_numpy(a))
    host = [hblock[i] for i in range(6)]
    oblock = torch.empty((4, case.n), dtype=torch.float64).pin_memory()
    hout_d = [oblock[i] for i in range(4)]
    hout_i = torch.empty(case.n, dtype=torch.int32).pin_memory()

    def e2e_step():
        case.handle.query_all_host(*host, step_max=W.STEP_MAX, out=[hout_i] + hout_d)

    def e2e_step5():
        for q in case.queries:
            case.handle.query_host(q, *host, step_max=W.STEP_MAX, out=hout_i if q == "inside" else hout_d[0])

    def time_e2e(fn):
        for _ in range(3):
            fn()
        barrier()
        w0 = time.perf_counter()
        for _ in range(ke):
            fn()
        w1 = time.perf_counter()
        barrier()
        return max_over_ranks(w1 - w0, "cuda")

    ke = max(3, min(args.steps, 20))
    e2e_s = time_e2e(e2e_step)
    e2e5_s = time_e2e(e2e_step5)
    h2d5 = sum((48 if q.startswith("distance") else 24) for q in case.queries) * case.n
    d2h = sum((4 if q == "inside" else 8) for q in case.queries) * case.n
    e2e = {"value": tracks_all * nq * ke / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 48 * case.n, "d2h_bytes_per_step": d2h,
           "steps": ke, "ms_per_step": e2e_s * 1e3 / ke,
           "api": "vg_query_all_host (one pinned [6][n] host basket in, pinned results out, chunked copy/compute overlap)",
           "host_link_gbs": (48 * case.n + d2h) / (e2e_s / ke) / 1e9,
           "five_single_query_calls": {"value": tracks_all * nq * ke / e2e5_s, "ms_per_step": e2e5_s * 1e3 / ke,
                                       "h2d_bytes_per_step": h2d5, "d2h_bytes_per_step": d2h, "api": "vg_query_host x5"}}

    fma_rate = vg.vg_probe_fp64_fma_rate(30)  # the ALU-bound rows of `detail` are the only users (configs[1] is HBM-bound)
    launches_per_step = nq
    detail, fig4 = None, None
    if world == 1 and not args.no_detail:
        detail = detail_sweep(vg, torch, hbm_peak, fma_rate, case)
        fig4 = fig4_gpu(vg, torch)
    load1 = time.time()
    sampler.stop()
    clocks = sampler.summary(t0, t1, load0, load1)

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": "configs[1]: tube segment rmin=5 rmax=10 dz=15 phi 0..4pi/3, N=%d tracks per GPU, "
                                       "Inside + DistanceToIn + DistanceToOut + SafetyToIn + SafetyToOut per step" % case.n,
                           "n_tracks_per_gpu": case.n, "queries_per_step": nq, "step_max": W.STEP_MAX,
                           "l2_policy": "inputs larger than L2: every launch reads the next of %d copies of the batch "
                                        "(%d MB of inputs in rotation, L2 = 126 MB)" % (case.nsets, case.nsets * 48 * case.n // 10 ** 6),
                           "launch": "CUDA graphs captured from the C-ABI calls, one graph per step",
                           "pipe_min_n": vg.vg_get_option(vg.OPT_PIPE_MIN_N), "form": vg.vg_get_option(vg.OPT_FORM), "pdl": vg.vg_get_option(vg.OPT_PDL),
                           "parallelism": "tracks sharded over ranks, no collective" if world > 1 else "1 GPU"},
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * args.steps,
                "roofline": roof, "per_query": per_query, "fused": fused,
                "fp64_peak": {"fma_per_s": fma_rate, "tflops": 2 * fma_rate / 1e12,
                              "how": "register-resident DFMA chains, vg_probe_fp64_fma_rate, same run"}}
        if world == 1:
            line["cpu_baseline"] = cpu_baseline()
            if fig4 is not None:  # the serial-CPU leg of the Fig. 4 protocol and the speed relative to it
                cpu4 = fig4_cpu()
                line["cpu_baseline"]["fig4_serial"] = cpu4
                ref = {(r["shape"], r["n"]): r["us_per_call"] for r in cpu4}
                for r in fig4:
                    r["serial_oracle_us_per_call"] = ref[(r["shape"], r["n"])]
                    r["speedup_device_resident"] = r["serial_oracle_us_per_call"] / r["device_resident_us_per_launch"]
                    r["speedup_host_fed"] = r["serial_oracle_us_per_call"] / r["host_fed_us_per_call"]
                line["fig4_protocol"] = {"what": "PAPER.md:120-136 (Fig. 4): DistanceToOut, Box and Tube, particles inside the body, "
                                                 "speed relative to a serial CPU code (here: the oracle on one thread; the paper's "
                                                 "own curve is not in the text, BASELINE.md)", "rows": fig4}
        if detail is not None:
            line["detail"] = detail
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-detail", action="store_true", help="skip the per-config sweep (configs[0..4])")
    ap.add_argument("--pipe-min-n", type=int, default=None,
                    help="vg_set_option(VG_OPT_PIPE_MIN_N): batch size from which the TMA-pipelined kernel runs "
                         "(default: the library's); for A/B runs of the two kernel forms")
    ap.add_argument("--form", choices=["auto", "direct", "pipelined", "streaming"], default=None,
                    help="vg_set_option(VG_OPT_FORM): kernel form for A/B runs (default: the library's per-kernel choice)")
    ap.add_argument("--no-pdl", action="store_true", help="vg_set_option(VG_OPT_PDL, 0): launch without programmatic dependent launch")
    ap.add_argument("--profile", action="store_true", help="eager launches of every kernel, for ncu; no timing")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.profile:
        run_profile(args)
        return
    if world != args.gpus and world == 1 and args.gpus > 1:
        raise SystemExit("bench.py: --gpus %d needs torchrun (one rank per GPU); see the module docstring" % args.gpus)
    run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
