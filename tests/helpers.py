"""Test-side helpers: tiny mesh builders and closed forms written from the formulas in
BASELINE.json / DESIGN.md "Pins" (independent of both the oracle's and the CUDA path's code)."""
import numpy as np

P0 = 4.56e-6


def quad(p0, eu, ev):
    """Two triangles (p0,p0+eu,p0+eu+ev), (p0,p0+eu+ev,p0+ev) as float32[2,3,3]."""
    p0, eu, ev = (np.asarray(a, float) for a in (p0, eu, ev))
    return np.array([[p0, p0 + eu, p0 + eu + ev], [p0, p0 + eu + ev, p0 + ev]], dtype=np.float32)


def const_mats(T, alpha, rho_s, rho_d):
    return np.tile(np.array([alpha, rho_s, rho_d], dtype=np.float32), (T, 1))


def unit(v):
    v = np.asarray(v, float)
    return v / np.linalg.norm(v)


def flat_plate_force(omega, normal, area, alpha, rho_s, rho_d, P=P0):
    """BASELINE.json: F = P A cos(th) [(alpha+rho_d) s + (2 rho_s cos(th) + 2/3 rho_d) n_in],
    s = sun->body direction, n_in = plate normal pointing away from the sun."""
    w = unit(omega)
    s = -w
    n = unit(normal)
    n_in = -n if np.dot(n, w) > 0 else n
    c = abs(np.dot(n, w))
    return P * area * c * ((alpha + rho_d) * s + (2.0 * rho_s * c + (2.0 / 3.0) * rho_d) * n_in)


def convex_polyhedron_force(verts, mats, omega, P=P0):
    """Sum of lit flat plates (the field's box-wing model): valid for any closed
    convex mesh at any bounce cap because reflected photons leave for good."""
    verts = np.asarray(verts, float)
    mats = np.asarray(mats, float)
    w = unit(omega)
    s = -w
    e1 = verts[:, 1] - verts[:, 0]
    e2 = verts[:, 2] - verts[:, 0]
    nA = 0.5 * np.cross(e1, e2)                     # area-weighted normal
    area = np.linalg.norm(nA, axis=1)
    n = nA / area[:, None]
    cen = verts.mean(axis=1) - verts.reshape(-1, 3).mean(axis=0)
    n = np.where((np.sum(n * cen, axis=1) < 0)[:, None], -n, n)      # outward
    c = n @ w
    lit = c > 0
    a, rs, rd = mats[:, 0], mats[:, 1], mats[:, 2]
    tot = a + rs + rd            # = 1 up to fp32 rounding of the stored materials
    # per facet: P A c [ tot*s - rs*r - 2/3 rd n ],  r = s + 2 c n  (mirror of s about outward n)
    F = (P * area * c)[:, None] * ((tot - rs)[:, None] * s[None, :]
                                    - (2.0 * rs * c + (2.0 / 3.0) * rd)[:, None] * n)
    return F[lit].sum(axis=0)


def rel_l2(a, b):
    a = np.asarray(a, float)
    b = np.asarray(b, float)
    return np.linalg.norm(a - b, axis=-1) / np.linalg.norm(b, axis=-1)


def oracle_pairs(oracle, meshes, pairs, sun, N, B, seed=0, workers=None, **kw):
    """Oracle forces for a list of (design k, direction j) pairs, one oracle call per pair, spread
    over host threads (the oracle itself is single-threaded; ctypes releases the GIL).
    meshes: dict k -> (verts, mats).  Returns (F f64[n,3], sigma f64[n], summed stats dict)."""
    import os
    from concurrent.futures import ThreadPoolExecutor

    def one(kj):
        k, j = int(kj[0]), int(kj[1])
        v, m = meshes[k]
        return oracle.forces(v, m, sun[j:j + 1], N, B, seed=seed, k=k, j0=j, **kw)

    with ThreadPoolExecutor(workers or min(32, os.cpu_count() or 1)) as ex:
        res = list(ex.map(one, pairs))
    F = np.stack([r["F"][0] for r in res])
    sig = np.array([r["sigma"][0] for r in res])
    tot = None
    for r in res:
        s = r["stats"]
        if tot is None:
            tot = {a: (list(b) if isinstance(b, list) else b) for a, b in s.items()}
        else:
            for a, b in s.items():
                tot[a] = [x + y for x, y in zip(tot[a], b)] if isinstance(b, list) else tot[a] + b
    if kw.get("want_path_sig"):
        return F, sig, tot, np.stack([r["path_sig"][0] for r in res])
    return F, sig, tot


def assert_parity(F_gpu, F_orc, sigma, tol_vec=1e-4, tol_agg=1e-3, diverged=None):
    """BASELINE.json acceptance: per-vector relative L2 <= 1e-4 where no ray diverged; vectors above
    that (a ray took another path at a grazing edge) must lie within 4 sigma, and the aggregate
    relative L2 over all vectors must be <= 1e-3.  `diverged` (bool per vector, from the path
    signatures) makes the first clause exact: a vector with no divergent ray MUST be within 1e-4.
    Returns the number of vectors above 1e-4."""
    F_gpu = np.asarray(F_gpu, float).reshape(-1, 3)
    F_orc = np.asarray(F_orc, float).reshape(-1, 3)
    sigma = np.asarray(sigma, float).reshape(-1)
    err = np.linalg.norm(F_gpu - F_orc, axis=1)
    nrm = np.linalg.norm(F_orc, axis=1)
    ok = err <= tol_vec * nrm + 1e-30
    bad = ~ok
    if diverged is not None:
        assert not np.any(bad & ~np.asarray(diverged, bool)), "vector off by > 1e-4 although no ray diverged"
    assert np.all(err[bad] <= 4.0 * sigma[bad] + 1e-30), "vector beyond 1e-4 AND beyond 4 sigma: %s" % err[bad]
    agg = np.linalg.norm(F_gpu - F_orc) / np.linalg.norm(F_orc)
    assert agg <= tol_agg, agg
    return int(bad.sum())


def direct_force_by_surface_quadrature(verts, mats, omega, sub=96, P=P0, shadows=True):
    """Direct-light force (no bounce followed, the paper's "NB" variant) by integrating Eq. 1-3 over
    the SURFACE instead of shooting photons: every triangle is cut into sub^2 small triangles; a piece whose centroid
    sees the sun (shadow ray toward omega against all other triangles, numpy Moller-Trumbore) adds
    P dA cos(th) [(a + rs + rd) s - rs r - 2/3 rd n_f].  Independent of the oracle: surface sampling + shadow rays
    (the visibility query of the paper's next-event estimation) instead of an emitter plane + closest hit.
    shadows=False lights every sun-facing piece (to show how much the shadowing matters)."""
    verts = np.asarray(verts, float)
    mats = np.asarray(mats, float)
    w = unit(omega)
    s = -w
    T = len(verts)
    v0, e1, e2 = verts[:, 0], verts[:, 1] - verts[:, 0], verts[:, 2] - verts[:, 0]
    # centroids of the sub^2 pieces in barycentric coordinates (upright and inverted pieces)
    i, j = np.meshgrid(np.arange(sub), np.arange(sub), indexing="ij")
    up = (i + j) <= sub - 1
    dn = (i + j) <= sub - 2
    bu = np.concatenate([(i[up] + 1 / 3) / sub, (i[dn] + 2 / 3) / sub])
    bv = np.concatenate([(j[up] + 1 / 3) / sub, (j[dn] + 2 / 3) / sub])
    F = np.zeros(3)
    for f in range(T):
        nA = 0.5 * np.cross(e1[f], e2[f])
        area = np.linalg.norm(nA)
        if area == 0:
            continue
        n = nA / area
        nf = n if np.dot(n, w) > 0 else -n                      # side facing the sun (two-sided facets)
        c = np.dot(nf, w)
        if c <= 0:
            continue
        x = v0[f] + bu[:, None] * e1[f] + bv[:, None] * e2[f]   # piece centroids
        lit = np.ones(len(x), bool)
        for g in range(T if shadows else 0):                    # shadow rays x + t w, t > 0
            if g == f:
                continue
            pv = np.cross(w, e2[g])
            det = np.dot(e1[g], pv)
            if det == 0:
                continue
            tv = x - v0[g]
            u = tv @ pv / det
            qv = np.cross(tv, e1[g])
            v = qv @ w / det
            t = qv @ e2[g] / det
            lit &= ~((u >= 0) & (v >= 0) & (u + v <= 1) & (t > 0))
        a, rs, rd = mats[f]
        r = s + 2.0 * c * nf                                    # mirror of s about nf (nf faces the sun: -s . nf = c)
        dA = area / (sub * sub)
        F += lit.sum() * P * dA * c * ((a + rs + rd) * s - rs * r - (2.0 / 3.0) * rd * nf)
    return F
