"""CPU pins of the oracle's glossy specular lobe ("per-face Phong material parameters"; SURVEY 8(f)
NEXT-2; R23): closed forms and invariants only -- nothing here compares the oracle with itself.  No GPU."""
import numpy as np
import pytest

from helpers import P0, quad, const_mats, unit, flat_plate_force


def plate(size=1.0):
    return quad([-size / 2, -size / 2, 0], [size, 0, 0], [0, size, 0])       # normal +z, area size^2


@pytest.mark.parametrize("deposit", [0, 1])
@pytest.mark.parametrize("ns", [0.0, 1.0, 10.0, 100.0])
def test_g1_normal_incidence_mean_cosine(oracle, ns, deposit):
    """Lobe cos^n about the mirror direction, which at normal incidence is the normal itself: nothing is truncated,
    E[cos] = int cos^(n+1) sin / int cos^n sin = (n+1)/(n+2), transverse mean 0.  A purely specular unit plate under
    pressure P therefore feels F = -P A (1 + (n+1)/(n+2)) z."""
    r = oracle.forces(plate(), const_mats(2, 0.0, 1.0, 0.0), [[0, 0, 1]], 1 << 16, 1, deposit=deposit,
                      shininess=[ns, ns])
    Fc = np.array([0, 0, -P0 * (1.0 + (ns + 1.0) / (ns + 2.0))])
    assert np.linalg.norm(r["F"][0] - Fc) <= 4 * r["sigma"][0]
    assert r["sigma"][0] < 0.01 * P0                        # the bound above is a real constraint
    assert r["stats"]["escaped"] == r["stats"]["launched"] == 1 << 16


def test_g2_mirror_limit_and_mixed_material(oracle):
    """n -> infinity is the ideal mirror of R5: oblique incidence on a plate with all three lobes, closed form of
    the flat plate (P1)."""
    om = unit([0.3, -0.2, 0.8])
    mats = const_mats(2, 0.25, 0.45, 0.30)
    r = oracle.forces(plate(), mats, [om], 1 << 14, 1, shininess=[1e7, 1e7])
    Fc = flat_plate_force(om, [0, 0, 1], 1.0, 0.25, 0.45, 0.30)
    assert np.linalg.norm(r["F"][0] - Fc) <= 4 * r["sigma"][0] + 1e-5 * np.linalg.norm(Fc)
    # negative shininess IS the mirror: bit-identical to the call without shininess
    a = oracle.forces(plate(), mats, [om], 1 << 10, 2, shininess=[-1.0, -1.0])
    b = oracle.forces(plate(), mats, [om], 1 << 10, 2)
    assert np.array_equal(a["F"], b["F"]) and a["stats"] == b["stats"]


@pytest.mark.parametrize("deposit", [0, 1])
def test_g3_lobe_axis_at_oblique_incidence(oracle, deposit):
    """A narrow lobe (n = 400, ~3 degrees wide) at 50 degrees incidence stays clear of the horizon, so its mean
    direction is ((n+1)/(n+2)) r with r the mirror direction: F = P A cos(theta_i) (d - (n+1)/(n+2) r).  A lobe laid
    about the normal, about -r, or rotated the wrong way round fails this by tens of sigma."""
    th = np.radians(50.0)
    om = np.array([np.sin(th) * np.cos(0.7), np.sin(th) * np.sin(0.7), np.cos(th)])
    d = -om
    refl = d + 2 * np.cos(th) * np.array([0, 0, 1.0])
    ns = 400.0
    r = oracle.forces(plate(), const_mats(2, 0.0, 1.0, 0.0), [om], 1 << 16, 1, deposit=deposit, shininess=[ns, ns])
    Fc = P0 * np.cos(th) * (d - (ns + 1.0) / (ns + 2.0) * refl)
    assert np.linalg.norm(r["F"][0] - Fc) <= 4 * r["sigma"][0] + 2e-4 * np.linalg.norm(Fc)
    assert r["sigma"][0] < 0.005 * np.linalg.norm(Fc)


def test_g4_horizon_rejection(oracle):
    """At 85 degrees incidence half of a wide lobe (n = 2) points below the facet.  Rejected directions are redrawn:
    no photon may pass through the plate into the absorber lying 1 mm behind it."""
    th = np.radians(85.0)
    om = np.array([np.sin(th), 0.0, np.cos(th)])
    front = plate()
    back = quad([-1.5, -1.5, -1e-3], [0, 3, 0], [3, 0, 0])                   # normal -z, absorbing, larger
    verts = np.concatenate([front, back])
    mats = np.concatenate([const_mats(2, 0.0, 1.0, 0.0), const_mats(2, 1.0, 0.0, 0.0)])
    sh = np.array([2.0, 2.0, -1.0, -1.0], np.float32)
    r = oracle.forces(verts, mats, [om], 1 << 15, 3, shininess=sh, want_first_hit=True)
    st = r["stats"]
    n_front = int((r["first_hit"][0] < 2).sum())
    assert n_front > 1000
    assert sum(st["hits_at_depth"][1:]) == 0                                 # nothing is hit after the plate
    assert st["absorbed"] == int((r["first_hit"][0] >= 2).sum())             # only primaries that hit the absorber
    # and the truncated lobe leans towards the normal: F_z is more negative than the untruncated lobe's
    r1 = oracle.forces(front, const_mats(2, 0.0, 1.0, 0.0), [om], 1 << 16, 1, shininess=[2.0, 2.0])
    d = -om
    refl = d + 2 * np.cos(th) * np.array([0, 0, 1.0])
    F_untruncated = P0 * np.cos(th) * (d - 0.75 * refl)
    assert r1["F"][0][2] < F_untruncated[2] - 4 * r1["sigma"][0]


@pytest.mark.parametrize("deposit", [0, 1])
def test_g5_bookkeeping_and_estimator_agreement(oracle, deposit):
    """Photon bookkeeping (P8) holds with glossy facets, and the two deposit rules estimate the same force (the
    expected-value rule deposits the specular part per drawn direction, R23)."""
    from paper_2602_10712_b200 import workloads as W
    verts, mats = oracle.build_mesh(W.FAMILY_BOXWING, W.draw_params(W.FAMILY_BOXWING, 1)[0])
    rng = np.random.default_rng(5)
    sh = rng.choice([-1.0, 0.0, 3.0, 40.0, 800.0], len(verts)).astype(np.float32)
    om = unit([0.4, 0.5, 0.6])
    r = oracle.forces(verts, mats, [om], 1 << 14, 6, deposit=deposit, shininess=sh)
    st = r["stats"]
    assert st["launched"] == st["primary_miss"] + st["absorbed"] + st["escaped"] + st["capped"]
    assert st["segments"] == sum(st["hits_at_depth"]) + st["primary_miss"] + st["escaped"]
    other = oracle.forces(verts, mats, [om], 1 << 14, 6, deposit=1 - deposit, shininess=sh)
    assert np.linalg.norm(r["F"][0] - other["F"][0]) <= 4 * np.hypot(r["sigma"][0], other["sigma"][0])


def test_g6_black_cavity_conserves_momentum_with_glossy_walls(oracle):
    """Thermal emitter in a closed box whose walls are glossy reflectors with some absorption: with the analog deposit
    every photon's momentum ends up in the walls, so the net force vanishes photon by photon (up to capped paths,
    which are excluded by making the cap deep and the walls dark enough)."""
    from test_oracle_thermal import box
    room = box([-1, -1, -1], [1, 1, 1], inward=True)
    emitter = quad([-0.2, -0.2, -0.3], [0.4, 0, 0], [0, 0.4, 0.1])
    verts = np.concatenate([room, emitter])
    mats = np.concatenate([const_mats(len(room), 0.6, 0.4, 0.0), const_mats(2, 1.0, 0.0, 0.0)])
    sh = np.concatenate([np.full(len(room), 6.0), [-1.0, -1.0]]).astype(np.float32)
    power = np.zeros(len(verts), np.float32); power[-2:] = 500.0
    r = oracle.thermal(verts, mats, power, 1 << 12, 15, deposit=1, shininess=sh)
    st = r["stats"]
    assert st["escaped"] == 0 and st["primary_miss"] == 0
    w = 1000.0 / 299792458.0
    # a capped photon (prob 0.4^16 ~ 4e-7 each) keeps its momentum: none expected among 8192
    assert st["capped"] == 0
    assert np.linalg.norm(r["F"]) < 1e-12 * w
