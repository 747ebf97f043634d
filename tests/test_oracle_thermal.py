"""CPU pins of the oracle's thermal (local Lambertian) emitters, PAPER.md:606-612 (Sec. 5.9; R22).
Closed forms and invariants only -- nothing here compares the oracle with itself.  No GPU."""
import numpy as np
import pytest

from paper_2602_10712_b200 import workloads as W
from helpers import quad, const_mats, unit

C = 299792458.0


def box(lo, hi, inward=False):
    """Closed axis-aligned box as 12 triangles, normals outward (or inward)."""
    lo, hi = np.asarray(lo, float), np.asarray(hi, float)
    d = hi - lo
    ex, ey, ez = np.array([d[0], 0, 0]), np.array([0, d[1], 0]), np.array([0, 0, d[2]])
    faces = [quad(lo, ez, ey), quad(lo + ex, ey, ez), quad(lo, ex, ez), quad(lo + ey, ez, ex),
             quad(lo, ey, ex), quad(lo + ez, ex, ey)]
    v = np.concatenate(faces)
    if inward:
        v = v[:, [0, 2, 1], :]
    return v.astype(np.float32)


@pytest.mark.parametrize("deposit", [0, 1])
def test_h1_isolated_emitter_recoil_is_two_thirds(oracle, deposit):
    """a Lambertian emitter's momentum flux is 2/3 of a collimated beam's: F = -(2/3) (W/c) n.  The
    paper's own example: 70 kW -> 1.55e-4 N.  Sign of W picks the side."""
    verts = quad([0, 0, 0], [1, 0, 0], [0, 0.5, 0.5])
    n = unit(np.cross([1, 0, 0], [0, 0.5, 0.5]))
    mats = const_mats(2, 0.2, 0.5, 0.3)
    r = oracle.thermal(verts, mats, [35000.0, 35000.0], 1 << 15, 3, deposit=deposit)
    Fc = -(2.0 / 3.0) * 70000.0 / C * n
    assert abs(np.linalg.norm(Fc) - 1.55e-4) < 0.01e-4                     # the paper's figure
    if deposit == 0:
        np.testing.assert_allclose(r["F"], Fc, rtol=1e-12, atol=1e-20)     # expected-value recoil is deterministic
    else:
        assert np.linalg.norm(r["F"] - Fc) <= 4 * r["sigma"]
    assert r["stats"]["launched"] == 2 << 15 == r["stats"]["primary_miss"]  # nothing to hit
    r2 = oracle.thermal(verts, mats, [-35000.0, -35000.0], 1 << 10, 3)
    np.testing.assert_allclose(r2["F"], -Fc, rtol=1e-12, atol=1e-20)


def test_h2_closed_black_cavity_has_no_net_force(oracle):
    """An emitter inside a closed, perfectly absorbing box: every photon's recoil is cancelled by its absorption
    (momentum conservation) -- exactly per photon with the analog deposit, within 4 sigma with the expected one."""
    room = box([-1, -1, -1], [1, 1, 1], inward=True)
    emitter = quad([-0.2, -0.2, -0.3], [0.4, 0, 0], [0, 0.4, 0.1])
    verts = np.concatenate([room, emitter])
    mats = const_mats(len(verts), 1.0, 0.0, 0.0)
    power = np.zeros(len(verts), np.float32); power[-2:] = 500.0
    r = oracle.thermal(verts, mats, power, 1 << 14, 4, deposit=1)
    assert r["stats"]["primary_miss"] == 0 and r["stats"]["absorbed"] == r["stats"]["launched"]
    assert np.linalg.norm(r["F"]) < 1e-12 * 1000.0 / C
    r = oracle.thermal(verts, mats, power, 1 << 14, 4, deposit=0)
    assert np.linalg.norm(r["F"]) <= 4 * r["sigma"]


def test_h3_perpendicular_squares_form_factor(oracle):
    """Unit square emitter in z = 0 radiating upwards, absorbing unit square in x = 0 sharing an edge: the fraction
    of photons absorbed is the form factor of two perpendicular unit squares with a common edge, 0.200044 (P7)."""
    a = quad([0, 0, 0], [1, 0, 0], [0, 1, 0])                  # normal +z
    b = quad([0, 0, 0], [0, 0, 1], [0, 1, 0])
    verts = np.concatenate([a, b])
    mats = const_mats(4, 1.0, 0.0, 0.0)
    N = 1 << 17
    r = oracle.thermal(verts, mats, [100.0, 100.0, 0.0, 0.0], N, 2)
    frac = r["stats"]["absorbed"] / r["stats"]["launched"]
    assert abs(frac - 0.200044) < 4 * np.sqrt(0.2 * 0.8 / (2 * N))
    # force: emitter recoil -(2/3) w z plus the momentum the absorber takes (it points towards -x and +z)
    w = 200.0 / C
    assert r["F"][0] < 0 and abs(r["F"][1]) < 4 * r["sigma"] + 1e-3 * w and -(2.0 / 3.0) * w < r["F"][2] < 0


def test_h4_linear_in_power_and_additive_over_facets(oracle):
    """F is linear in W (same photons) and the sum over emitting facets; zero power emits nothing."""
    verts, mats = oracle.build_mesh(W.FAMILY_BOXWING, W.draw_params(W.FAMILY_BOXWING, 1)[0])
    pw = np.zeros(16, np.float32); pw[3] = 700.0; pw[12] = -300.0
    r = oracle.thermal(verts, mats, pw, 1 << 12, 4, seed=2)
    r2 = oracle.thermal(verts, mats, 2 * pw, 1 << 12, 4, seed=2)
    np.testing.assert_allclose(r2["F"], 2 * r["F"], rtol=1e-12)
    pa, pb = pw.copy(), pw.copy(); pa[12] = 0; pb[3] = 0
    ra = oracle.thermal(verts, mats, pa, 1 << 12, 4, seed=2)
    rb = oracle.thermal(verts, mats, pb, 1 << 12, 4, seed=2)
    np.testing.assert_allclose(ra["F"] + rb["F"], r["F"], rtol=1e-10, atol=1e-22)
    assert ra["stats"]["launched"] == 1 << 12
    z = oracle.thermal(verts, mats, np.zeros(16, np.float32), 1 << 12, 4)
    assert np.all(z["F"] == 0) and z["stats"]["launched"] == 0


def test_h5_emitter_under_a_mirror_roof(oracle):
    """Emitter at z = 0 under a large mirror at z = 1 (normal facing down): what the mirror reflects comes back down
    and leaves (or hits the small emitter, a black body).  With the analog deposit each reflection off the mirror
    pushes it by 2 w d_z upwards, so F_z of the pair exceeds the free emitter's recoil by the reflected part; with a
    mirror covering almost the whole hemisphere, F_z -> -(2/3) w + 2 (2/3) w = +(2/3) w."""
    emitter = quad([-0.05, -0.05, 0], [0.1, 0, 0], [0, 0.1, 0])
    roof = quad([-200, -200, 1], [0, 400, 0], [400, 0, 0])                 # normal -z
    verts = np.concatenate([emitter, roof])
    mats = np.concatenate([const_mats(2, 1, 0, 0), const_mats(2, 0, 1, 0)])
    w = 100.0 / C
    for deposit in (0, 1):
        r = oracle.thermal(verts, mats, [50.0, 50.0, 0, 0], 1 << 15, 1, deposit=deposit)
        assert abs(r["F"][2] - (2.0 / 3.0) * w) <= 4 * r["sigma"] + 0.01 * w
        assert abs(r["F"][0]) <= 4 * r["sigma"] + 0.01 * w
