"""CPU pins of the oracle's direct / indirect split (Fig. 5 rows 3-4: "direct" and "indirect" force
maps; the no-bounce variant "NB").  F_direct = momentum deposited where sun light first meets the
surface; F_indirect = F - F_direct.  No GPU."""
import numpy as np
import pytest

from paper_2602_10712_b200 import workloads as W
from helpers import P0, quad, const_mats, convex_polyhedron_force, direct_force_by_surface_quadrature


def test_convex_body_has_no_indirect_force(oracle):
    # S1: reflected photons of a convex body leave for good, so everything is direct -- for any B and both deposits
    verts = W.icosphere(2, 1.0)
    mats = W.dirichlet_materials(len(verts), 5)
    sun = W.fibonacci_sphere(6)
    for deposit in (0, 1):
        r = oracle.forces_split(verts, mats, sun, 1 << 12, 6, deposit=deposit)
        assert np.array_equal(r["F"], r["F_direct"])
        assert np.all(r["F_indirect"] == 0.0)
    Fc = np.array([convex_polyhedron_force(verts, mats, w) for w in sun])
    assert np.all(np.linalg.norm(r["F_direct"] - Fc, axis=1) <= 0.03 * np.linalg.norm(Fc, axis=1))


@pytest.mark.parametrize("deposit", [0, 1])
def test_direct_is_the_no_bounce_force(oracle, deposit):
    # S2: the B = 0 run follows the same photons to their first hit and stops: its force is F_direct of any B, bit for bit
    th = W.draw_params(W.FAMILY_BOXWING, 2)
    sun = np.array([[0.2, 0.9, 0.3], [0.1, -0.95, -0.2], [0.7, 0.1, -0.7]], np.float32)
    for k in range(2):
        v, m = oracle.build_mesh(W.FAMILY_BOXWING, th[k], k=k)
        nb = oracle.forces(v, m, sun, 1 << 14, 0, seed=3, k=k, deposit=deposit)
        r = oracle.forces_split(v, m, sun, 1 << 14, 4, seed=3, k=k, deposit=deposit)
        full = oracle.forces(v, m, sun, 1 << 14, 4, seed=3, k=k, deposit=deposit)
        assert np.array_equal(r["F_direct"], nb["F"])
        assert np.array_equal(r["F"], full["F"])
        assert r["stats"] == full["stats"]
        # self-reflections between the panels and the bus are there, so the split is not trivial
        assert np.linalg.norm(r["F_indirect"]) > 1e-3 * np.linalg.norm(r["F"])


def test_direct_part_against_the_surface_quadrature(oracle):
    # S3: P12's independent surface integration with shadow rays is the direct force, whatever B
    th = W.draw_params(W.FAMILY_BOXWING, 1)
    v, m = oracle.build_mesh(W.FAMILY_BOXWING, th[0])
    sun = np.array([[0.1, -0.95, -0.2]], np.float32)
    r = oracle.forces_split(v, m, sun, 1 << 18, 4, seed=1)
    Fq = direct_force_by_surface_quadrature(v, m, sun[0])
    sig = oracle.forces(v, m, sun, 1 << 18, 0, seed=1)["sigma"][0]
    assert np.linalg.norm(r["F_direct"][0] - Fq) <= 4.0 * sig + 6e-3 * np.linalg.norm(Fq)


@pytest.mark.parametrize("B,ind", [(0, 0.0), (1, 1.0), (3, 1.0)])
def test_v_groove_split(oracle, B, ind):
    # S4: two mirrors at 90 degrees, sun along the bisector (P6): the first hits carry P A_p, the second hits another
    # P A_p -- which is all indirect
    h = np.sqrt(0.5)
    verts = np.concatenate([quad([0, -0.5, 0], [h, 0, h], [0, 1, 0]), quad([0, -0.5, 0], [-h, 0, h], [0, 1, 0])])
    r = oracle.forces_split(verts, const_mats(4, 0.0, 1.0, 0.0), np.array([[0, 0, 1]], np.float32), 1 << 12, B)
    Ap = np.sqrt(2.0)
    np.testing.assert_allclose(r["F_direct"][0], [0, 0, -P0 * Ap], rtol=1e-6, atol=1e-13)
    np.testing.assert_allclose(r["F_indirect"][0], [0, 0, -ind * P0 * Ap], rtol=1e-6, atol=1e-13)
