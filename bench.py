#!/usr/bin/env python
"""bench.py -- tracks/s per query on one B200 (BASELINE.json `metric`) for the geometry hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-detail] [--min-ms M]

Workload of the headline: BASELINE.json configs[2], the largest single-GPU configuration -- a cone segment
(rmin1 2, rmax1 6, rmin2 4, rmax2 12, dz 20, full phi) AND a trd (5, 10, 7, 3, 15), N = 4,194,304 tracks each, all five
queries (Inside, DistanceToIn, DistanceToOut, SafetyToIn, SafetyToOut) on both: one *pass* = ten kernel launches through
the C ABI.  A *step* is `config.passes_per_step` passes, chosen so that the timed region (exactly --steps steps) lasts at
least --min-ms (200 ms); the region is timed five times and the median is reported.  `value` =
tracks x queries / second with the tracks resident in HBM; every launch reads a different copy of the batch (rotating
buffer sets, each 201 MB > the 126 MB L2), so no launch finds its inputs in L2.  The steps are replays of a CUDA graph
captured from the same C-ABI calls.  `e2e` is the same pass through the host-buffer entry points (pinned host arrays in,
host arrays out, copies inside the timed region).

Output: the LAST stdout line is one compact JSON object (< 2 KB: the driver keeps only the tail of stdout).  Everything
else -- one row per (config, shape, query) of BASELINE.json configs[0..4] with its roofline fractions, the hot / cold
variants, the 8(f) rows, the Fig. 4 protocol, the oracle timed on every config -- is printed on EARLIER lines (one JSON
object per line) and written to `bench_detail.json` beside this file.

Extra keys of the compact line: `per_config` (<= 10 rows, one per (config, shape, N): the query furthest below its bound
with us per launch and f / f8 / fp64 / lat fractions, `cl` = size-matched memory ceiling / measured, `pipe` = ncu's FP64-pipe
utilisation of that kernel from the committed capture), `value_fused_calls` (the same ten answers per track pair from the
two fused vg_query_all calls instead of ten launches), `cpu_Mtq_s_1thr_allcores` (the oracle per config).

`--gpus N` without torchrun starts N ranks itself (torch.distributed.run, one rank per GPU, NCCL only for the timing
reductions); under torchrun (WORLD_SIZE set) it runs as the rank it is.
`--impl reference` times the oracle (oracle/, plain scalar CPU code) on the host cores on the same workload.
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
BYTES.update({"world_locate": 24 + 4, "world_step": 48 + 4 + 8 + 4, "world_safety": 24 + 4 + 8, "volume_safety": 24 + 8})
L2_BYTES = 126e6
COLD_ROTATION_BYTES = 4 * 126e6  # bytes of track arrays in rotation (>= 256 MB): even Inside, which reads half
                                 # of a set, comes back to a set only after >= 2 x L2 of other reads
MAX_SETS = 192
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
                            "fp64_pipe_pct": float(c[7]) if len(c) > 7 and c[7] else None,
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
        # rotation >= 256 MB and >= 2 x L2 (SURVEY 8(d) cold variant), at most MAX_SETS copies (N <= 2^14 stays L2-resident:
        # there a launch is two orders of magnitude longer than its bytes take, cold or not)
        self.nsets = int(min(MAX_SETS, max(2, -(-int(COLD_ROTATION_BYTES) // per_set))))
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
        elif q == "volume_safety":
            self.handle.safety(*s[:3], out=self.outd[k])
        elif q.startswith("probe:"):  # the arithmetic-free kernel of the same loads, store, grid and form (vg_probe_stream)
            pq = q[6:]
            out = self.outi[k] if pq == "inside" else self.outd[k]
            if pq in ("distance_to_in", "distance_to_out"):
                self.vg.vg_probe_stream(pq, *s, out=out)
            else:
                self.vg.vg_probe_stream(pq, *s[:3], out=out)
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


def time_query_alone(torch, case, q, min_ms=100.0, hot=False, trials=5, want_trials=False):
    """Duration of one launch of `q` (cold inputs): a graph of nsets launches over the rotating sets, replayed between
    two CUDA events on the launching stream until >= min_ms have been timed; median of `trials` such regions (SURVEY
    8(d) protocol).  hot = True: every launch reads the SAME buffer set (what the paper's 5000 repetitions on fixed
    particles did): the batch stays in the 126 MB L2 if it fits."""
    case.cursor = 0
    case.launch(q)
    torch.cuda.synchronize()
    case.cursor = 0
    per_graph = case.nsets if not hot else max(case.nsets, 8)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        for _ in range(per_graph):
            if hot:
                case.cursor = 0
            case.launch(q)
    for _ in range(3):
        g.replay()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def region(reps):
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            g.replay()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    reps = 2
    ms = region(reps)
    while ms < min_ms and reps < (1 << 20):  # grow the region to >= min_ms
        reps = int(max(reps * 2, reps * 1.15 * min_ms / max(ms, 1e-3))) if ms < 0.5 * min_ms else reps * 2
        ms = region(reps)
    vals = sorted([ms] + [region(reps) for _ in range(trials - 1)])
    sec = [v * 1e-3 / (reps * per_graph) for v in vals]
    med = sec[len(sec) // 2]
    return (med, sec) if want_trials else med


# ------------------------------------------------------------------------------------------ the oracle legs

def oracle_step(O, shape, tracks, queries):
    for q in queries:
        if q in ("distance_to_in", "distance_to_out"):
            getattr(shape, q)(*tracks, W.STEP_MAX)
        else:
            getattr(shape, q)(*tracks[:3])


HEADLINE_CFG = 2  # BASELINE.json configs[2]: the largest single-GPU configuration (cone + trd, 4,194,304 tracks each)
HEADLINE_WORKLOAD = "configs[2]: cone(2,6,4,12,20,full phi) + trd(5,10,7,3,15), N=4194304 tracks each, all 5 queries on both"


def oracle_headline_inputs(O, n=None):
    """[(oracle shape, tracks, queries)] of the headline workload, the first n tracks of each shape (None: all)."""
    out = []
    for sc in W.shape_cases(HEADLINE_CFG):
        s = O.Shape(sc.kind, sc.params)
        m = sc.sizes[-1] if n is None else int(n)
        out.append((s, sc.tracks(m, band=lambda x, y, z, s=s: np.abs(s.sdf(x, y, z)) < W.SURFACE_BAND), sc.queries))
    return out


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


ORACLE_BUILD = "gcc -O2 -ffp-contract=off -fopenmp, schedule(static)"


def cpu_baseline(seconds=10.0, n=1048576):
    """The oracle as it stands, timed on this box's host cores on a bounded sample of the headline workload: the first
    `n` tracks of each of the two configs[2] solids, all five queries, repeated for ~`seconds`."""
    import oracle as O
    inp = oracle_headline_inputs(O, n)
    for s, t, qs in inp:
        oracle_step(O, s, t, qs)  # warm-up (thread pool, page faults)
    reps, t0 = 0, time.perf_counter()
    while True:
        for s, t, qs in inp:
            oracle_step(O, s, t, qs)
        reps += 1
        el = time.perf_counter() - t0
        if el >= seconds:
            break
    units = sum(len(qs) * len(t[0]) for _, t, qs in inp)
    return {"value": units * reps / el, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
            "sample": "%d x (5 queries on the first %d tracks of each configs[2] solid), %.1f s wall" % (reps, n, el),
            "cpu": cpu_model(), "build": ORACLE_BUILD}


def cpu_per_config(budget_s=6.0):
    """The oracle on every config of BASELINE.json: one thread and all cores, full N
    unless one pass at full N would exceed `budget_s` seconds (then a prefix whose size is stated; the oracle's cost
    per track does not depend on N).  Rows go to the side file; the compact line carries the two rates per config."""
    import oracle as O
    all_threads = O.num_threads()
    plan = []
    for k in (0, 1, 2, 3):
        for sc in W.shape_cases(k):
            s = O.Shape(sc.kind, sc.params)
            plan.append((k, sc.name, sc.sizes[-1], sc.queries, s,
                         lambda m, sc=sc, s=s: sc.tracks(m, band=lambda x, y, z: np.abs(s.sdf(x, y, z)) < W.SURFACE_BAND)))
    nav = W.navigator_case()
    vo = O.Volume(O.Shape(nav.mother_kind, nav.mother_params),
                  [O.Shape(kk, pp) for kk, pp in zip(nav.daughter_kinds, nav.daughter_params)], nav.xforms)
    plan.append((4, "navigator", nav.sizes[-1], ("compute_step",), vo,
                 lambda m: nav.tracks(m, band=lambda x, y, z: vo.safety(x, y, z) < W.SURFACE_BAND)))

    def one_pass(obj, t, qs):
        if qs == ("compute_step",):
            obj.compute_step(*t, W.STEP_MAX)
        else:
            oracle_step(O, obj, t, qs)

    rows = []
    try:
        for k, name, nfull, qs, obj, draw in plan:
            probe = draw(16384)
            O.set_num_threads(1)
            one_pass(obj, probe, qs)
            t0 = time.perf_counter()
            one_pass(obj, probe, qs)
            per_track_1 = (time.perf_counter() - t0) / 16384
            for threads in (1, all_threads):
                O.set_num_threads(threads)
                n = int(min(nfull, max(16384, budget_s / (per_track_1 / threads * (1.0 if threads == 1 else 1.5)))))
                t = draw(n)
                one_pass(obj, t, qs)  # warm-up: page faults of the result arrays, thread pool
                t0 = time.perf_counter()
                one_pass(obj, t, qs)
                el = time.perf_counter() - t0
                rows.append({"row": "cpu_oracle", "config": k, "shape": name, "queries": list(qs), "n": n, "n_full": nfull,
                             "threads": threads, "seconds_per_pass": el, "ns_per_track_query": el * 1e9 / (n * len(qs)),
                             "track_queries_per_s": n * len(qs) / el, "cpu": cpu_model(), "build": ORACLE_BUILD})
    finally:
        O.set_num_threads(all_threads)
    return rows


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
    """--impl reference: the oracle on the host cores, same workload / metric / unit (rank 0 only).  Each step is one
    pass (five queries, both configs[2] solids) over a prefix of the tracks sized so that the run ends within ~2 min."""
    if rank != 0:
        return
    import oracle as O
    probe = oracle_headline_inputs(O, 65536)
    for s, t, qs in probe:
        oracle_step(O, s, t, qs)
    t0 = time.perf_counter()
    for s, t, qs in probe:
        oracle_step(O, s, t, qs)
    per_track = (time.perf_counter() - t0) / 65536  # seconds per track of BOTH solids, five queries each
    budget = 100.0  # seconds for the whole --steps + --warmup run
    nfull = W.shape_cases(HEADLINE_CFG)[0].sizes[-1]
    n = int(min(nfull, max(4096, budget / ((args.steps + args.warmup) * per_track))))
    inp = oracle_headline_inputs(O, n)
    for _ in range(args.warmup):
        for s, t, qs in inp:
            oracle_step(O, s, t, qs)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        for s, t, qs in inp:
            oracle_step(O, s, t, qs)
    el = time.perf_counter() - t0
    units = sum(len(qs) * len(t[0]) for _, t, qs in inp)
    value = units * args.steps / el
    sample = "each step = 5 queries on the first %d of the %d tracks of each configs[2] solid" % (n, nfull)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": el * 1e3 / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": HEADLINE_WORKLOAD, "n_tracks_per_solid_per_step": n, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample,
                             "cpu": cpu_model(), "build": ORACLE_BUILD},
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


def detail_sweep(vg, torch, hbm_peak, fma_rate, have, headline_rows, min_ms, emit):
    """Every (config, shape, query) of BASELINE.json configs[0..4], each launch timed alone on cold inputs (and hot, where
    a batch fits L2), then the SURVEY 8(f) rows.  `have` = the headline's cases by shape name (reused, not re-drawn),
    `headline_rows` = their rows already timed with the full protocol."""
    rows = []

    def add(e):
        rows.append(e)
        emit(e)

    tq = lambda case, q, **kw: time_query_alone(torch, case, q, min_ms=min_ms, **kw)
    tq3 = lambda case, q: time_query_alone(torch, case, q, min_ms=min_ms / 2, trials=3)  # 8(f) rows
    floor_s = launch_floor(vg, torch)
    plan = []
    for k in (0, 1, 2, 3):
        for i, sc in enumerate(W.shape_cases(k)):
            for n in sc.sizes:
                plan.append((k, sc, n))
    for k, sc, n in plan:
        mine = sc.name not in have
        case = Case(vg, torch, sc.name, n, sc.queries, shape=sc) if mine else have[sc.name]
        for q in sc.queries:
            if not mine:
                e = dict(headline_rows[(sc.name, q)])
            else:
                sec = tq(case, q)
                e = roofline_entry(case.kind, q, n, sec, hbm_peak, fma_rate)
            e.update({"config": k, "shape": sc.name, "query": q, "n": n, "cold_inputs": case.cold, "sets_in_rotation": case.nsets})
            if 48 * n <= 0.5 * L2_BYTES:  # the hot variant: same buffers every launch, the batch stays in L2
                hot_s = tq(case, q, hot=True)
                e.update({"hot_us_per_launch": hot_s * 1e6, "hot_tracks_per_s": n / hot_s})
            if k in (0, 1) or n <= 262144:  # the size-matched memory ceiling: the same loads and store without the arithmetic
                ceil_s = tq3(case, "probe:" + q)
                e.update({"mem_ceiling_us": ceil_s * 1e6, "frac_of_mem_ceiling": ceil_s / (e["us_per_launch"] * 1e-6)})
            if n <= 262144:  # launch-bound sizes: the bound a single launch can reach is max(bytes / BW, empty launch)
                ideal = max(BYTES[q] * n / (hbm_peak * 1e9), floor_s)
                e.update({"empty_launch_us": floor_s * 1e6, "latency_adjusted_bound_us": ideal * 1e6,
                          "latency_adjusted_frac": ideal / (e["us_per_launch"] * 1e-6)})
            add(e)
        if len(sc.queries) == 5 and sc.kind != W.POLYCONE:  # the fused five-query kernel on the same tracks
            sec = tq(case, "all")
            e = roofline_entry(case.kind, "all", n, sec, hbm_peak, fma_rate)
            e.update({"config": k, "shape": sc.name, "query": "all five (vg_query_all, one kernel)", "n": n, "cold_inputs": case.cold,
                      "track_queries_per_s": 5 * n / sec})
            add(e)
        if mine:
            del case
            torch.cuda.empty_cache()
    nav = W.navigator_case()
    case = Case(vg, torch, "navigator", nav.sizes[-1], ("compute_step",), nav=nav)
    sec = tq(case, "compute_step")
    e = roofline_entry("navigator", "compute_step", case.n, sec, hbm_peak, fma_rate)
    e.update({"config": 4, "shape": "box(100)+64 daughters", "query": "compute_step", "n": case.n, "cold_inputs": case.cold})
    add(e)
    sec = tq(case, "volume_safety")  # vg_volume_safety (an addition of this build): not part of any step
    e = roofline_entry("navigator", "volume_safety", case.n, sec, hbm_peak, fma_rate)
    e.update({"config": "4 (+)", "shape": "box(100)+64 daughters", "query": "volume_safety", "n": case.n, "cold_inputs": case.cold})
    add(e)
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
            sec = tq3(case, q)
            e = roofline_entry("polycone_variant", q, case.n, sec, hbm_peak, fma_rate)
            e.update({"config": "8(f) f2", "shape": vname, "query": q, "n": case.n, "cold_inputs": case.cold, "bound": "alu"})
            add(e)
        del case
        torch.cuda.empty_cache()
    # boolean solids of two primitives (one of each operation)
    for bc in [b for b in W.boolean_cases() if b.name in ("tube_union_box", "cone_intersection_orb", "box_minus_tube")]:
        case = Case(vg, torch, bc.name, 4194304, W.QUERIES5, boolean=bc)
        for q in case.queries:
            sec = tq3(case, q)
            e = roofline_entry("boolean", q, case.n, sec, hbm_peak, fma_rate)
            e.update({"config": "8(f) f2", "shape": bc.name, "query": q, "n": case.n, "cold_inputs": case.cold})
            if q.startswith("distance"):
                e["bound"] = "alu"
            add(e)
        del case
        torch.cuda.empty_cache()
    cc = [c for c in W.csg_cases() if c.name == "twice_drilled_block_in_a_sphere"][0]  # a tree of four primitives (R31)
    case = Case(vg, torch, cc.name, 4194304, W.QUERIES5, csg=cc)
    for q in case.queries:
        sec = tq3(case, q)
        e = roofline_entry("boolean", q, case.n, sec, hbm_peak, fma_rate)
        e.update({"config": "8(f) f2", "shape": "csg tree: " + cc.name, "query": q, "n": case.n, "cold_inputs": case.cold, "bound": "alu"})
        add(e)
    del case
    torch.cuda.empty_cache()
    # the three-level tree of placed solids (193 nodes), every track in its own node
    wc = W.world_case()
    case = Case(vg, torch, "world", wc.sizes[-1], ("world_locate", "world_step", "world_safety"), world=wc)
    for q in case.queries:
        sec = tq3(case, q)
        e = roofline_entry("world", q, case.n, sec, hbm_peak, fma_rate)
        e.update({"config": "8(f) f3", "shape": "box(100) > 64 daughters > 128 grand-daughters", "query": q, "n": case.n,
                  "cold_inputs": case.cold, "bound": "alu", "track_order": "as drawn (nodes mixed within a warp)"})
        add(e)
    # the same tracks in basket order (sorted by node, what the paper's scheduler hands to the geometry)
    for k in range(case.nsets):
        order = torch.argsort(case.nodes[k].to(torch.int64), stable=True)
        case.sets[k] = [a[order].contiguous() for a in case.sets[k]]
        case.nodes[k] = case.nodes[k][order].contiguous()
    for q in case.queries:
        sec = tq3(case, q)
        e = roofline_entry("world", q, case.n, sec, hbm_peak, fma_rate)
        e.update({"config": "8(f) f3", "shape": "box(100) > 64 daughters > 128 grand-daughters", "query": q, "n": case.n,
                  "cold_inputs": case.cold, "bound": "alu", "track_order": "sorted by node (baskets)"})
        add(e)
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
    pc = W.shape_cases(3)[0]  # the small batches of configs[3]: the lanes-per-track kernels (vg_pcon_coop.cuh)
    for n_small in (1024, 16384):
        cases.append(Case(vg, torch, pc.name, n_small, pc.queries, shape=pc))
    nav = W.navigator_case()
    cases.append(Case(vg, torch, "navigator", nav.sizes[-1], ("compute_step", "volume_safety"), nav=nav))
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


def _sig(v, digits=4):
    """Floats of the compact line rounded to `digits` significant digits (the line must stay under 2 KB)."""
    if isinstance(v, float):
        return float("%.*g" % (digits, v)) if v == v and abs(v) != float("inf") else None
    if isinstance(v, dict):
        return {k: _sig(x, digits) for k, x in v.items()}
    if isinstance(v, (list, tuple)):
        return [_sig(x, digits) for x in v]
    return v


KERNEL_NAME = {  # launch form of AUTO for the headline kernels (csrc/vg_kernels.cuh Tune<S, Q>); ncu names in profiles/
    "cone": "query_kernel<ConeT<1>,%s>", "trd": "query_kernel<Trd,%s>"}
NCU_SOLID = {"cone": "Cone", "trd": "Trd", "tube": "Tube", "box": "Box", "orb": "Orb", "polycone": "Polycone"}
SHORT_Q = {"inside": "in", "distance_to_in": "dti", "distance_to_out": "dto", "safety_to_in": "sti", "safety_to_out": "sto",
           "compute_step": "step"}
HBM_NOMINAL_GBS = 8000.0  # BASELINE.json north_star: "~8 TB/s peak"; the 70 % target is read against this


def per_config_rows(detail, fma_rate):
    """<= 10 short rows for the compact line: per (config, shape) the query FURTHEST below its bound.  us = one launch
    (cold inputs), f = fraction of the measured HBM copy rate, f8 = fraction of the nominal 8 TB/s, fp64 = SURVEY 8(d)'s
    algorithmic FP64 operations / s over the FP64 rate measured in this run (ALU-bound rows), lat = latency-adjusted
    fraction max(bytes / BW, empty launch) / measured (launch-bound sizes), cl = duration of the arithmetic-free kernel
    with the same loads, store, grid and form on the same buffers (vg_probe_stream) / measured, pipe = ncu's
    sm__inst_executed_pipe_fp64 (fraction of peak while active) of that kernel in the committed capture."""
    groups = {}
    for e in detail:
        if e.get("row") or not isinstance(e.get("config"), int) or str(e["query"]).startswith("all five"):
            continue
        groups.setdefault((e["config"], e["shape"], e["n"]), []).append(e)
    keep = []
    for (k, shape, n), es in sorted(groups.items(), key=lambda kv: (kv[0][0], kv[0][1], kv[0][2])):
        if k == 3 and n not in (1024, 16777216):
            continue
        score = lambda e: e["latency_adjusted_frac"] if n <= 262144 else (e.get("fp64_frac") if e["bound"] == "alu" else e["hbm_frac"])
        w = min(es, key=score)
        r = {"c": "%d %s 2^%d" % (k, shape.split("(")[0][:8], n.bit_length() - 1), "q": SHORT_Q.get(w["query"], w["query"]), "us": w["us_per_launch"]}
        if n <= 262144:
            r["lat"] = w["latency_adjusted_frac"]
        elif w["bound"] == "alu":
            r["fp64"] = w["fp64_frac"]  # SURVEY 8(d)'s numerator (every segment / every daughter) over the measured FP64 rate
            tr = ncu_traffic("navigator" if k == 4 else NCU_SOLID.get(shape, shape), w["query"], min(n, 4194304))
            if tr and tr.get("fp64_pipe_pct") is not None:  # what the hardware counted in the committed capture (n = 2^22)
                r["pipe"] = tr["fp64_pipe_pct"] / 100.0
        else:
            r["f"], r["f8"] = w["hbm_frac"], w["hbm_gbs"] / HBM_NOMINAL_GBS
        if "frac_of_mem_ceiling" in w:  # cl = the size-matched memory ceiling (same loads / store / grid, no arithmetic) / measured
            r["cl"] = w["frac_of_mem_ceiling"]
        keep.append(_sig(r, 3))
    return keep


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

    side = []  # every row of the side file, in the order it is produced

    def emit(row):
        side.append(row)
        if rank == 0:
            print(json.dumps(_sig(row, 6)), flush=True)

    hbm_peak, hbm_src = measured_peaks()
    sampler = ClockSampler(local_rank)
    sampler.start()
    load0 = time.time()
    warmup = max(args.warmup, 3)

    # weak scaling: every rank owns one full configs[2] batch (its own seeds); no data-path collective
    cases = [Case(vg, torch, sc.name, sc.sizes[-1], sc.queries, seed_shift=1000 * rank, shape=sc)
             for sc in W.shape_cases(HEADLINE_CFG)]
    launches = [(c, q) for c in cases for q in c.queries]  # one pass = ten launches
    nsets = max(c.nsets for c in cases)
    for c, q in launches:  # eager warm-up before capture (lazy attribute / occupancy queries happen here)
        c.launch(q)
    torch.cuda.synchronize()
    for c in cases:
        c.cursor = 0
    graph = torch.cuda.CUDAGraph()  # nsets passes: after them every launch position has used every buffer set
    with torch.cuda.graph(graph):
        for _ in range(nsets):
            for c, q in launches:
                c.launch(q)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    graph.replay()
    torch.cuda.synchronize()
    e0.record()
    graph.replay()
    e1.record()
    torch.cuda.synchronize()
    replay_ms = max_over_ranks(e0.elapsed_time(e1), "cuda")
    replays_per_step = max(1, int(-(-args.min_ms // (args.steps * replay_ms)))) if args.min_ms > 0 else 1
    passes_per_step = replays_per_step * nsets
    for _ in range(warmup):
        for _ in range(replays_per_step):
            graph.replay()
    torch.cuda.synchronize()
    trial_ms, t0 = [], time.time()
    for _ in range(args.trials):  # the timed region (exactly --steps steps), `trials` times; the median is reported
        barrier()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(args.steps * replays_per_step):
            graph.replay()
        e1.record()
        torch.cuda.synchronize()
        barrier()
        trial_ms.append(max_over_ranks(e0.elapsed_time(e1), "cuda"))
    t1 = time.time()
    ms = sorted(trial_ms)[len(trial_ms) // 2]
    units_per_pass = sum_over_ranks(sum(c.n * len(c.queries) for c in cases), "cuda")  # track-queries, all ranks
    value = units_per_pass * passes_per_step * args.steps / (ms * 1e-3)
    pass_us = ms * 1e3 / (args.steps * passes_per_step)
    algo_bytes_per_pass = sum(BYTES[q] * c.n for c, q in launches)

    # per-kernel durations, same process, right after the timed region: event-record nodes between the kernel nodes of
    # the timed graph cost ~5 us each (measured) and would distort `value`, so every query is timed alone as a graph of
    # back-to-back launches over the rotating sets (cold inputs) between two CUDA events on the launching stream
    head_rows, per_q = {}, {}
    for c, q in launches:
        sec, tr = time_query_alone(torch, c, q, min_ms=args.min_ms, trials=args.trials, want_trials=True)
        per_q[(c.name, q)] = sec
        e = roofline_entry(c.kind, q, c.n, sec, hbm_peak, 1.0)
        e.update({"hbm_frac_of_8TBs": e["hbm_gbs"] / HBM_NOMINAL_GBS, "trials_us": [x * 1e6 for x in tr]})
        head_rows[(c.name, q)] = e
    dom = max(per_q, key=per_q.get)
    dcase = [c for c in cases if c.name == dom[0]][0]
    tr = ncu_traffic(NCU_SOLID.get(dcase.kind, dcase.kind), dom[1], dcase.n)
    sum_k = sum(per_q.values())
    roof = {"bound": "hbm", "kernel": KERNEL_NAME.get(dcase.kind, "%s") % dom[1], "achieved": head_rows[dom]["hbm_gbs"],
            "peak": hbm_peak, "unit": "GB/s", "frac": head_rows[dom]["hbm_gbs"] / hbm_peak,
            "peak_source": hbm_src, "frac_of_8TBs": head_rows[dom]["hbm_gbs"] / HBM_NOMINAL_GBS,
            "traffic": (tr or {}).get("bytes"), "traffic_capture": (tr or {}).get("capture"),
            "algorithmic_bytes_per_launch": BYTES[dom[1]] * dcase.n, "us_per_launch": per_q[dom] * 1e6,
            "share_of_pass": per_q[dom] / sum_k, "sum_of_kernels_us": sum_k * 1e6, "pass_us": pass_us,
            "pass_hbm_frac": algo_bytes_per_pass / (pass_us * 1e-6) / 1e9 / hbm_peak}

    # end to end: pinned host arrays -> C-ABI host entry point -> pinned host results, copies inside the timed region.
    # The call a user makes for one pass over host tracks is vg_query_all_host per solid (the tracks cross the host link
    # once for all five answers).  Each host basket is ONE pinned [6][n] allocation (and the four FP64 results one
    # [4][n]): equally spaced arrays cross the link as one strided copy per chunk (vg_host.cu).
    hostbuf = []
    for c in cases:
        hb = torch.empty((6, c.n), dtype=torch.float64).pin_memory()
        for i, a in enumerate(c.host):
            hb[i].copy_(torch.from_numpy(a))
        ob = torch.empty((4, c.n), dtype=torch.float64).pin_memory()
        hostbuf.append((c, [hb[i] for i in range(6)], [torch.empty(c.n, dtype=torch.int32).pin_memory()] + [ob[i] for i in range(4)]))

    def e2e_pass():
        for c, hin, hout in hostbuf:
            c.handle.query_all_host(*hin, step_max=W.STEP_MAX, out=hout)

    for _ in range(2):
        e2e_pass()
    w0 = time.perf_counter()
    e2e_pass()
    one = time.perf_counter() - w0
    ke = max(3, int(-(-args.min_ms * 1e-3 // one))) if args.min_ms > 0 else 3
    e2e_trials = []
    for _ in range(3):
        barrier()
        w0 = time.perf_counter()
        for _ in range(ke):
            e2e_pass()
        w1 = time.perf_counter()
        barrier()
        e2e_trials.append(max_over_ranks(w1 - w0, "cuda"))
    e2e_s = sorted(e2e_trials)[1]
    h2d = sum(48 * c.n for c in cases)
    d2h = sum(36 * c.n for c in cases)
    e2e = {"value": units_per_pass * ke / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
           "steps": ke, "ms_per_step": e2e_s * 1e3 / ke, "passes_per_step": 1,
           "host_link_gbs": (h2d + d2h) / (e2e_s / ke) / 1e9, "api": "vg_query_all_host per solid, pinned [6][n] baskets"}
    del hostbuf

    # FP64 rate probe AFTER the timed regions above: it drives the FP64 pipe at full power for ~70 ms and would leave the
    # board power-capped for the measurements that matter; the ALU-bound rows of the sweep are its only users
    fma_rate = vg.vg_probe_fp64_fma_rate(30)
    detail, fig4 = None, None
    have = {c.name: c for c in cases}
    if world == 1 and not args.no_detail:
        emit({"row": "header", "note": "one JSON object per line; the LAST line is the compact bench record", "hbm_peak_gbs": hbm_peak,
              "hbm_peak_source": hbm_src, "fp64_fma_per_s": fma_rate, "fp64_tflops": 2 * fma_rate / 1e12,
              "fp64_how": "register-resident DFMA chains, vg_probe_fp64_fma_rate, same run",
              "timing": "each launch alone: graph of back-to-back launches over rotating buffer sets, >= %g ms per region, median of %d" % (args.min_ms, args.trials)})
        detail = detail_sweep(vg, torch, hbm_peak, fma_rate, have, head_rows, args.min_ms * args.detail_scale, emit)
        fig4 = fig4_gpu(vg, torch)
    else:
        for (name, q), e in head_rows.items():
            e.update({"config": HEADLINE_CFG, "shape": name, "query": q, "n": have[name].n, "cold_inputs": have[name].cold})
            emit(e)
        detail = list(head_rows.values())
    load1 = time.time()
    sampler.stop()
    clocks = sampler.summary(t0, t1, load0, load1)

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warmup,
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": HEADLINE_WORKLOAD, "n_tracks": cases[0].n, "launches_per_pass": len(launches),
                           "passes_per_step": passes_per_step, "trials": "median of %d" % args.trials, "timed_ms": ms,
                           "l2": "inputs > L2: %d rotating copies of 201 MB per solid" % nsets,
                           "parallelism": "tracks sharded, no collective" if world > 1 else "1 GPU"},
                "clocks": {k: clocks.get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons")},
                "gpu_launches": len(launches) * passes_per_step * args.steps,
                "roofline": {k: roof[k] for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "frac_of_8TBs", "traffic",
                                                  "algorithmic_bytes_per_launch", "us_per_launch", "share_of_pass", "pass_hbm_frac")},
                "e2e": {k: e2e[k] for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "ms_per_step")},
                "fp64_tflops_measured": 2 * fma_rate / 1e12}
        emit({"row": "headline", "trial_ms": trial_ms, "roofline": roof, "e2e": e2e, "clocks": clocks,
              "options": {"pipe_min_n": vg.vg_get_option(vg.OPT_PIPE_MIN_N), "form": vg.vg_get_option(vg.OPT_FORM), "pdl": vg.vg_get_option(vg.OPT_PDL)}})
        if world == 1:
            cb = cpu_baseline(seconds=args.cpu_seconds)
            line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")}
            emit(dict(cb, row="cpu_baseline"))
            if fig4 is not None:  # the serial-CPU leg of the Fig. 4 protocol and the speed relative to it
                ref = {(r["shape"], r["n"]): r["us_per_call"] for r in fig4_cpu()}
                for r in fig4:
                    r["serial_oracle_us_per_call"] = ref[(r["shape"], r["n"])]
                    r["speedup_device_resident"] = r["serial_oracle_us_per_call"] / r["device_resident_us_per_launch"]
                    r["speedup_host_fed"] = r["serial_oracle_us_per_call"] / r["host_fed_us_per_call"]
                    emit(dict(r, row="fig4_protocol", what="PAPER.md:120-136 (Fig. 4): DistanceToOut, particles inside the body, speed "
                              "relative to a serial CPU code (here the oracle on one thread; the paper's curve is not in the text)"))
            if not args.no_detail:
                cpu_rows = cpu_per_config()
                for r in cpu_rows:
                    emit(r)
                # per config: [one thread, all cores] in 1e6 track-queries/s, all shapes of the config pooled
                pool = {}
                for r in cpu_rows:
                    a = pool.setdefault((r["config"], r["threads"]), [0.0, 0.0])
                    a[0] += r["n"] * len(r["queries"])
                    a[1] += r["seconds_per_pass"]
                line["cpu_Mtq_s_1thr_allcores"] = {str(k): [pool[(k, t)][0] / pool[(k, t)][1] / 1e6 for t in sorted({t for kk, t in pool if kk == k})]
                                                   for k in sorted({kk for kk, _ in pool})}
                line["per_config"] = per_config_rows(detail, fma_rate)
                # the same ten answers per track pair from the two fused calls (vg_query_all) instead of ten launches
                fused = [e for e in detail if e.get("config") == HEADLINE_CFG and str(e.get("query", "")).startswith("all five")]
                if len(fused) == 2:
                    line["value_fused_calls"] = sum(5 * e["n"] for e in fused) / sum(e["us_per_launch"] * 1e-6 for e in fused)
        line["detail"] = "bench_detail.json"
        try:
            with open(os.path.join(ROOT, "bench_detail.json"), "w") as f:
                json.dump({"line": line, "rows": side}, f, indent=1)
        except OSError:
            line["detail"] = "earlier stdout lines"
        out = json.dumps(_sig(line), separators=(",", ":"))
        for drop in ("cpu_Mtq_s_1thr_allcores", "fp64_tflops_measured"):  # never let the record outgrow the driver's tail
            if len(out) > 2000 and drop in line:
                del line[drop]
                out = json.dumps(_sig(line), separators=(",", ":"))
        while len(out) > 2000 and line.get("per_config"):
            line["per_config"].pop()
            out = json.dumps(_sig(line), separators=(",", ":"))
        print(out, flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def spawn_ranks(args):
    """`python bench.py --gpus N` as a plain command: start one rank per GPU under torch.distributed.run (what the driver
    does itself for N > 1) and pass this process's arguments through."""
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")  # the driver counts ranks from NCCL's own log
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--min-ms", type=float, default=200.0,
                    help="minimum length of every timed region in ms (SURVEY 8(d): >= 200 ms; 0 = one graph replay per step, for ncu)")
    ap.add_argument("--trials", type=int, default=5, help="timed regions per number; the median is reported")
    ap.add_argument("--detail-scale", type=float, default=0.5,
                    help="timed-region length of the per-config sweep as a fraction of --min-ms (1.0 = the full SURVEY protocol)")
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="wall time of the cpu_baseline leg")
    ap.add_argument("--no-detail", action="store_true", help="skip the per-config sweep (configs[0..4]) and the 8(f) rows")
    ap.add_argument("--pipe-min-n", type=int, default=None,
                    help="vg_set_option(VG_OPT_PIPE_MIN_N): batch size from which the TMA-pipelined kernel runs "
                         "(default: the library's); for A/B runs of the two kernel forms")
    ap.add_argument("--form", choices=["auto", "direct", "pipelined", "streaming"], default=None,
                    help="vg_set_option(VG_OPT_FORM): kernel form for A/B runs (default: the library's per-kernel choice)")
    ap.add_argument("--no-pdl", action="store_true", help="vg_set_option(VG_OPT_PDL, 0): launch without programmatic dependent launch")
    ap.add_argument("--profile", action="store_true", help="eager launches of every kernel, for ncu; no timing")
    args = ap.parse_args()
    if args.impl == "ours" and not args.profile and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        raise SystemExit(spawn_ranks(args))
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.profile:
        run_profile(args)
        return
    run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
