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
