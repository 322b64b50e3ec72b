"""Parity policy GPU vs oracle (BASELINE.json north_star):
Inside classes and hit indices bit-exact; +inf and -1 sentinels bit-exact; finite distances / safeties pass iff
|g - o| <= max(1e-9, 1e-12 |o|).  No whitelist."""
import numpy as np

ABS_TOL = 1e-9   # BASELINE.json: "within 1e-12 relative or 1e-9 absolute"
REL_TOL = 1e-12


def assert_int_equal(g, o, what):
    g, o = np.asarray(g), np.asarray(o)
    assert g.shape == o.shape, what
    bad = np.flatnonzero(g != o)
    assert bad.size == 0, "%s: %d of %d differ, first at %d: gpu %r oracle %r" % (
        what, bad.size, g.size, bad[0] if bad.size else -1, g[bad[:5]], o[bad[:5]])


def _recheck(ld, idx, g, o):
    """c.7: the failing tracks again with the 80-bit build of the oracle (x87 long double): which side is off?"""
    if ld is None or len(idx) == 0:
        return ""
    idx = np.asarray(idx[:5])
    try:
        ref = np.asarray(ld(idx), dtype=np.float64)
    except Exception as exc:  # the report must not mask the mismatch itself
        return "; 80-bit re-evaluation failed: %r" % (exc,)
    rows = ["track %d: gpu %.17g oracle %.17g oracle80 %.17g (|gpu - o80| %.2e, |oracle - o80| %.2e)" % (
        i, g[i], o[i], r, abs(g[i] - r), abs(o[i] - r)) for i, r in zip(idx, ref)]
    return "; 80-bit oracle on the first failing tracks: " + " | ".join(rows)


def assert_real_close(g, o, what, ld=None):
    """`ld`: optional callable(track indices) -> the same quantity from the 80-bit oracle, used only to report a mismatch."""
    g, o = np.asarray(g, dtype=np.float64), np.asarray(o, dtype=np.float64)
    assert g.shape == o.shape, what
    assert not np.isnan(g).any(), "%s: NaN in the GPU result" % what
    for name, sentinel in (("+inf", np.inf), ("-1", -1.0)):
        mg, mo = g == sentinel, o == sentinel
        bad = np.flatnonzero(mg != mo)
        assert bad.size == 0, "%s: %s masks differ at %d of %d tracks, first %d: gpu %r oracle %r%s" % (
            what, name, bad.size, g.size, bad[0] if bad.size else -1, g[bad[:5]], o[bad[:5]], _recheck(ld, bad, g, o))
    fin = np.isfinite(o)
    err = np.abs(g[fin] - o[fin])
    tol = np.maximum(ABS_TOL, REL_TOL * np.abs(o[fin]))
    bad = np.flatnonzero(err > tol)
    assert bad.size == 0, "%s: %d of %d finite values out of tolerance, worst |err| %.3e (gpu %r oracle %r)%s" % (
        what, bad.size, int(fin.sum()), err.max() if err.size else 0.0, g[fin][bad[:3]], o[fin][bad[:3]],
        _recheck(ld, np.flatnonzero(fin)[bad], g, o))
    return float(err.max()) if err.size else 0.0
