"""CPU pins of the oracle's torque (Eq. 4: tau = int (x - x_COM) x f(x) dx).
Each check compares the oracle with a closed form or an identity, never with itself.  No GPU."""
import numpy as np
import pytest

from paper_2602_10712_b200 import workloads as W
from helpers import P0, quad, const_mats, flat_plate_force, rel_l2


def test_t1_off_centre_plate_closed_form(oracle):
    """A uniformly lit flat plate: force density is uniform, so tau = (centroid - x_COM) x F with F the
    flat-plate closed form (P2).  Plate centred at (2, -1, 0.5), tilted normal, COM elsewhere."""
    p0 = np.array([1.5, -1.75, 0.5]); eu = np.array([1.0, 0, 0]); ev = np.array([0, 1.5, 0.3])
    verts = quad(p0, eu, ev)
    mats = const_mats(2, 0.3, 0.5, 0.2)
    centroid = p0 + 0.5 * eu + 0.5 * ev
    normal = np.cross(eu, ev); normal /= np.linalg.norm(normal)
    area = np.linalg.norm(np.cross(eu, ev))
    x_com = np.array([0.2, 0.1, -0.4])
    sun = np.array([[0.3, 0.2, 0.8], [-0.5, 0.1, 0.6], [0.1, -0.7, -0.5]], np.float32)
    for sampler in (0, 1):
        r = oracle.forces(verts, mats, sun, 1 << 16, 1, seed=3, sampler=sampler, x_com=x_com)
        for j in range(len(sun)):
            Fc = flat_plate_force(sun[j], normal, area, 0.3, 0.5, 0.2)
            Tc = np.cross(centroid - x_com, Fc)
            assert np.linalg.norm(r["T"][j] - Tc) <= 4.0 * r["sigma_T"][j] + 1e-6 * np.linalg.norm(Tc)
            if sampler == 0:
                assert np.linalg.norm(r["T"][j] - Tc) < 5e-3 * np.linalg.norm(Tc)


def test_t2_windmill_of_two_plates(oracle):
    """Two coplanar unit plates at x = +-2 facing the sun, one black, one a mirror: the forces differ by a
    factor 2, so the pair turns about y: tau = sum_i r_i x F_i.  A transposed cross product flips the sign."""
    black = quad([1.5, -0.5, 0.0], [1, 0, 0], [0, 1, 0])
    mirror = quad([-2.5, -0.5, 0.0], [1, 0, 0], [0, 1, 0])
    verts = np.concatenate([black, mirror])
    mats = np.concatenate([const_mats(2, 1, 0, 0), const_mats(2, 0, 1, 0)])
    om = np.array([[0, 0, 1]], np.float32)
    r = oracle.forces(verts, mats, om, 1 << 16, 2, seed=1, x_com=[0, 0, 0])
    Fb = np.array([0, 0, -P0]); Fm = np.array([0, 0, -2 * P0])
    Tc = np.cross([2.0, 0, 0], Fb) + np.cross([-2.0, 0, 0], Fm)       # = (0, 2P, 0) + (0, -4P, 0)
    np.testing.assert_allclose(Tc, [0, -2 * P0, 0], atol=1e-18)
    assert np.linalg.norm(r["T"][0] - Tc) <= 4.0 * r["sigma_T"][0]
    assert np.linalg.norm(r["T"][0] - Tc) < 5e-3 * np.linalg.norm(Tc)
    assert r["T"][0][1] < 0


def test_t3_centre_of_mass_shift_identity(oracle):
    """tau(x_COM + a) = tau(x_COM) - a x F for the same photons, to rounding -- with bounces (box-wing)."""
    verts, mats = oracle.build_mesh(W.FAMILY_BOXWING, W.draw_params(W.FAMILY_BOXWING, 1)[0])
    sun = W.fibonacci_sphere(5)
    a = np.array([0.7, -1.3, 2.1])
    r0 = oracle.forces(verts, mats, sun, 1 << 12, 4, seed=2, x_com=[0, 0, 0])
    r1 = oracle.forces(verts, mats, sun, 1 << 12, 4, seed=2, x_com=a)
    np.testing.assert_array_equal(r0["F"], r1["F"])
    np.testing.assert_allclose(r1["T"], r0["T"] - np.cross(a, r0["F"]), rtol=0, atol=1e-12 * np.abs(r0["T"]).max())
    assert sum(r0["stats"]["hits_at_depth"][1:]) > 0
    # and the forces are exactly those of the force-only entry point
    np.testing.assert_array_equal(oracle.forces(verts, mats, sun, 1 << 12, 4, seed=2)["F"], r0["F"])


def test_t4_centred_sphere_has_no_torque(oracle):
    """A sphere about its own centre: by symmetry the expected torque vanishes for any material mix
    (the force does not: cannonball, P4)."""
    verts = W.icosphere(2, 1.0)
    mats = const_mats(len(verts), 0.3, 0.3, 0.4)
    sun = W.fibonacci_sphere(4)
    r = oracle.forces(verts, mats, sun, 1 << 14, 2, seed=5, sampler=1, x_com=[0, 0, 0])
    for j in range(len(sun)):
        assert np.linalg.norm(r["T"][j]) <= 4.0 * r["sigma_T"][j]
        assert np.linalg.norm(r["T"][j]) < 0.05 * np.linalg.norm(r["F"][j]) * 1.0      # << |F| x radius


@pytest.mark.parametrize("deposit", [0, 1])
def test_t5_estimators_agree_on_torque(oracle, deposit):
    """Expected-value and analog deposits estimate the same torque (within 4 sigma of the analog one)."""
    verts, mats = oracle.build_mesh(W.FAMILY_BOXWING, W.draw_params(W.FAMILY_BOXWING, 1)[0])
    sun = W.fibonacci_sphere(3)
    xc = [0.1, 0.2, -0.3]
    ref = oracle.forces(verts, mats, sun, 1 << 16, 4, seed=7, deposit=0, x_com=xc)
    r = oracle.forces(verts, mats, sun, 1 << 14, 4, seed=8, deposit=deposit, sampler=1, x_com=xc)
    for j in range(len(sun)):
        assert np.linalg.norm(r["T"][j] - ref["T"][j]) <= 4.0 * np.hypot(r["sigma_T"][j], ref["sigma_T"][j])
