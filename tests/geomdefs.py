"""Independent numpy statements of the solids, used ONLY to pin the oracle (tests, -m "not gpu").

Nothing here is shared with oracle/ or with the CUDA path: membership is the closed point set of
SURVEY.md sec. 8(c) c.1 typed directly, and the boundary is given as explicit parametrised patches
(s, t) in [0,1]^2 -> R^3 for brute-force sampling.  The oracle instead works on an (r, z) polygon.
"""
import math

import numpy as np

BOX, ORB, TUBE, CONE, TRD, POLYCONE = range(6)
TWO_PI = 2 * math.pi


def in_wedge(x, y, sphi, dphi):
    if dphi >= TWO_PI:
        return np.ones(np.shape(x), dtype=bool)
    return np.mod(np.arctan2(y, x) - sphi, TWO_PI) <= dphi


def _lin(a1, a2, z, z1, z2):
    return a1 + (a2 - a1) * (z - z1) / (z2 - z1)


def sections(kind, par):
    """(z_lo, z_hi, rmin_lo, rmax_lo, rmin_hi, rmax_hi) list + (sphi, dphi) for solids of revolution."""
    if kind == TUBE:
        rmin, rmax, dz, sphi, dphi = par
        return [(-dz, dz, rmin, rmax, rmin, rmax)], sphi, dphi
    if kind == CONE:
        rmin1, rmax1, rmin2, rmax2, dz, sphi, dphi = par
        return [(-dz, dz, rmin1, rmax1, rmin2, rmax2)], sphi, dphi
    if kind == POLYCONE:
        sphi, dphi, nz = par[0], par[1], int(par[2])
        pl = [(par[3 + 3 * i], par[4 + 3 * i], par[5 + 3 * i]) for i in range(nz)]
        return [(pl[i][0], pl[i + 1][0], pl[i][1], pl[i][2], pl[i + 1][1], pl[i + 1][2]) for i in range(nz - 1)], sphi, dphi
    raise ValueError(kind)


def member(kind, par, x, y, z):
    """p in S, S closed (c.1)."""
    x, y, z = (np.asarray(v, dtype=np.float64) for v in (x, y, z))
    if kind == BOX:
        return (np.abs(x) <= par[0]) & (np.abs(y) <= par[1]) & (np.abs(z) <= par[2])
    if kind == ORB:
        return x * x + y * y + z * z <= par[0] ** 2
    if kind == TRD:
        dx1, dx2, dy1, dy2, dz = par
        X = _lin(dx1, dx2, z, -dz, dz)
        Y = _lin(dy1, dy2, z, -dz, dz)
        return (np.abs(z) <= dz) & (np.abs(x) <= X) & (np.abs(y) <= Y)
    secs, sphi, dphi = sections(kind, par)
    rho = np.sqrt(x * x + y * y)
    ok = np.zeros(x.shape, dtype=bool)
    for (z0, z1, a0, b0, a1, b1) in secs:
        if z1 == z0:  # a z step of a polycone (R26): no volume of its own
            continue
        rlo = _lin(a0, a1, z, z0, z1)
        rhi = _lin(b0, b1, z, z0, z1)
        ok |= (z >= z0) & (z <= z1) & (rho >= rlo) & (rho <= rhi)
    return ok & in_wedge(x, y, sphi, dphi)


def patches(kind, par):
    """List of callables f(s, t) -> (x, y, z) covering the boundary of the solid, s, t in [0, 1]."""
    out = []
    if kind == BOX:
        hx, hy, hz = par
        for sg in (-1.0, 1.0):
            out.append(lambda s, t, sg=sg: (sg * hx + 0 * s, (2 * s - 1) * hy, (2 * t - 1) * hz))
            out.append(lambda s, t, sg=sg: ((2 * s - 1) * hx, sg * hy + 0 * s, (2 * t - 1) * hz))
            out.append(lambda s, t, sg=sg: ((2 * s - 1) * hx, (2 * t - 1) * hy, sg * hz + 0 * s))
        return out
    if kind == ORB:
        r = par[0]
        out.append(lambda s, t: (r * np.sqrt(1 - (2 * t - 1) ** 2) * np.cos(TWO_PI * s),
                                 r * np.sqrt(1 - (2 * t - 1) ** 2) * np.sin(TWO_PI * s), r * (2 * t - 1)))
        return out
    if kind == TRD:
        dx1, dx2, dy1, dy2, dz = par

        def side(axis, sg):
            def f(s, t):
                z = (2 * t - 1) * dz
                X = _lin(dx1, dx2, z, -dz, dz)
                Y = _lin(dy1, dy2, z, -dz, dz)
                if axis == 0:
                    return sg * X, (2 * s - 1) * Y, z
                return (2 * s - 1) * X, sg * Y, z
            return f
        for sg in (-1.0, 1.0):
            out.append(side(0, sg))
            out.append(side(1, sg))
        out.append(lambda s, t: ((2 * s - 1) * dx1, (2 * t - 1) * dy1, -dz + 0 * s))
        out.append(lambda s, t: ((2 * s - 1) * dx2, (2 * t - 1) * dy2, dz + 0 * s))
        return out
    secs, sphi, dphi = sections(kind, par)
    dphi_eff = min(dphi, TWO_PI)

    def frustum(z0, z1, r0, r1):
        def f(s, t):
            z = z0 + t * (z1 - z0)
            r = r0 + t * (r1 - r0)
            ph = sphi + s * dphi_eff
            return r * np.cos(ph), r * np.sin(ph), z
        return f

    def cap(zc, rlo, rhi):
        def f(s, t):
            r = rlo + t * (rhi - rlo)
            ph = sphi + s * dphi_eff
            return r * np.cos(ph), r * np.sin(ph), zc + 0 * s
        return f

    def face(ph, z0, z1, a0, b0, a1, b1):
        def f(s, t):
            z = z0 + t * (z1 - z0)
            rlo = a0 + t * (a1 - a0)
            rhi = b0 + t * (b1 - b0)
            r = rlo + s * (rhi - rlo)
            return r * math.cos(ph), r * math.sin(ph), z
        return f

    for (z0, z1, a0, b0, a1, b1) in secs:
        out.append(frustum(z0, z1, b0, b1))  # for a z step (z0 == z1) this is the annular face between the two radii
        if a0 > 0 or a1 > 0:
            out.append(frustum(z0, z1, a0, a1))
        if dphi < TWO_PI and z1 > z0:
            out.append(face(sphi, z0, z1, a0, b0, a1, b1))
            out.append(face(sphi + dphi, z0, z1, a0, b0, a1, b1))
    z0, _, a0, b0, _, _ = secs[0]
    _, z1, _, _, a1, b1 = secs[-1]
    out.append(cap(z0, a0, b0))
    out.append(cap(z1, a1, b1))
    return out


def brute_distance(kind, par, p, coarse=160, zoom_rounds=4, zoom_grid=21):
    """min over the boundary patches of |p - s|, by dense sampling with local zoom (error << 1e-4)."""
    p = np.asarray(p, dtype=np.float64)
    best = np.inf
    g = (np.arange(coarse) + 0.5) / coarse
    S, T = np.meshgrid(g, g, indexing="ij")
    # include the patch borders explicitly
    edge = np.linspace(0, 1, coarse)
    for f in patches(kind, par):
        ss = np.concatenate([S.ravel(), edge, edge, 0 * edge, 0 * edge + 1])
        tt = np.concatenate([T.ravel(), 0 * edge, 0 * edge + 1, edge, edge])
        x, y, z = f(ss, tt)
        d2 = (x - p[0]) ** 2 + (y - p[1]) ** 2 + (z - p[2]) ** 2
        for k in np.argsort(d2)[:3]:
            s0, t0, w = ss[k], tt[k], 1.5 / coarse
            dk = d2[k]
            for _ in range(zoom_rounds):
                gs = np.clip(s0 + np.linspace(-w, w, zoom_grid), 0, 1)
                gt = np.clip(t0 + np.linspace(-w, w, zoom_grid), 0, 1)
                A, B = np.meshgrid(gs, gt, indexing="ij")
                xx, yy, zz = f(A.ravel(), B.ravel())
                dd = (xx - p[0]) ** 2 + (yy - p[1]) ** 2 + (zz - p[2]) ** 2
                j = int(np.argmin(dd))
                if dd[j] < dk:
                    dk, s0, t0 = dd[j], A.ravel()[j], B.ravel()[j]
                w *= 2.5 / zoom_grid * 2
            best = min(best, dk)
    return math.sqrt(best)


def march_first_flip(kind, par, p, d, tmax, step=1e-3):
    """Brute-force ray marching on the membership function: first parameter where membership flips,
    refined by bisection; np.inf if none up to tmax."""
    p = np.asarray(p, dtype=np.float64)
    d = np.asarray(d, dtype=np.float64)
    t = np.arange(0.0, tmax + step, step)
    m = member(kind, par, p[0] + t * d[0], p[1] + t * d[1], p[2] + t * d[2])
    flips = np.flatnonzero(m[1:] != m[:-1])
    if flips.size == 0:
        return np.inf
    lo, hi = t[flips[0]], t[flips[0] + 1]
    m_lo = m[flips[0]]
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        if bool(member(kind, par, *(p + mid * d))) == bool(m_lo):
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)


def random_rotation(rng):
    q = rng.normal(size=4)
    q /= np.linalg.norm(q)
    x, y, z, w = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])
