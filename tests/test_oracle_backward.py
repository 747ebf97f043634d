"""CPU pins of the oracle's backward estimator (the paper's Eq. 5: area-proportional surface
point, BRDF-sampled incoming direction, path tracing with next-event estimation toward the sun at every vertex,
BRDF-sampled outgoing direction) and its agreement with the forward tracer (R25).
No GPU."""
import numpy as np
import pytest

from paper_2602_10712_b200 import workloads as W
from helpers import P0, quad, const_mats, flat_plate_force, convex_polyhedron_force


def test_b1_flat_plate_is_exact(oracle):
    # every surface point of a lit plate receives the same pressure: no variance at all with the expected-value deposit
    verts, _ = oracle.build_mesh(W.FAMILY_PLATE, [0.3, 0.5, 0.2])
    mats = const_mats(2, 0.3, 0.5, 0.2)
    for om in ([0.3, 0.2, 0.8], [0.0, 0.0, 1.0], [0.5, -0.4, -0.6]):
        r = oracle.backward(verts, mats, om, 256, 3)
        Fc = flat_plate_force(om, [0, 0, 1], 1.0, 0.3, 0.5, 0.2)
        np.testing.assert_allclose(r["F"], Fc, rtol=3e-7, atol=1e-20)            # direction and materials are fp32 inputs
        assert r["sigma"] <= 1e-6 * np.linalg.norm(Fc)       # zero up to the cancellation in Q/N - F^2
        # analog deposit: the outgoing direction is drawn; same mean
        ra = oracle.backward(verts, mats, om, 1 << 14, 3, deposit=1)
        assert np.linalg.norm(ra["F"] - Fc) <= 4 * ra["sigma"] and ra["sigma"] > 0
    edge_on = oracle.backward(verts, mats, [1.0, 0.0, 0.0], 64, 2)
    assert np.all(edge_on["F"] == 0.0)


def test_b2_convex_polyhedron(oracle):
    verts = W.icosphere(2, 1.0)
    mats = W.dirichlet_materials(len(verts), 5)
    for om in W.fibonacci_sphere(4):
        r = oracle.backward(verts, mats, om, 1 << 14, 4, seed=2)
        Fc = convex_polyhedron_force(verts, mats, om)
        assert np.linalg.norm(r["F"] - Fc) <= 4 * r["sigma"], (r["F"], Fc)
        assert r["sigma"] < 0.05 * np.linalg.norm(Fc)
        # nothing is lit indirectly on a convex body: with B = 0 (no indirect paths at all) the same samples give the same force
        r0 = oracle.backward(verts, mats, om, 1 << 14, 0, seed=2)
        assert np.array_equal(r0["F"], r["F"])


def test_b3_shadow_rays(oracle):
    # a black plate hidden behind a larger mirror plate receives nothing; the front plate gives its closed form
    back = quad([-0.5, -0.5, 0.0], [1, 0, 0], [0, 1, 0])
    front = quad([-1.0, -1.0, 1.0], [2, 0, 0], [0, 2, 0])
    verts = np.concatenate([back, front])
    mats = np.concatenate([const_mats(2, 1.0, 0.0, 0.0), const_mats(2, 0.0, 1.0, 0.0)])
    r = oracle.backward(verts, mats, [0, 0, 1], 1 << 12, 0)
    Fc = flat_plate_force([0, 0, 1], [0, 0, 1], 4.0, 0.0, 1.0, 0.0)
    np.testing.assert_allclose(r["F"], Fc, rtol=2e-2, atol=1e-12)     # area-proportional sampling: 4/5 of the samples land on the front plate
    assert abs(r["F"][2] - Fc[2]) <= 4 * r["sigma"]


def test_b4_perpendicular_plates_indirect_light(oracle):
    """P7's scene: unit square A (rho_d = 1) in z = 0 lit from +z, black unit square B in x = 0 sharing an edge.  The
    light B receives is all indirect; the forward tracer and the backward estimator must agree on the total."""
    A = quad([0, 0, 0], [1, 0, 0], [0, 1, 0])
    Bq = quad([0, 0, 0], [0, 1, 0], [0, 0, 1])
    verts = np.concatenate([A, Bq])
    mats = np.concatenate([const_mats(2, 0.0, 0.0, 1.0), const_mats(2, 1.0, 0.0, 0.0)])
    sun = np.array([[0, 0, 1]], np.float32)
    fw = oracle.forces(verts, mats, sun, 1 << 18, 1, sampler=1)
    bw = oracle.backward(verts, mats, sun[0], 1 << 17, 1)
    assert np.linalg.norm(bw["F"] - fw["F"][0]) <= 4 * np.hypot(bw["sigma"], fw["sigma"][0])
    # direct part on A: P (0, 0, -5/3); the rest is what B absorbs: m = (-0.1213, 0, +0.1213) P (P7's quadrature)
    m = bw["F"] / P0 - np.array([0, 0, -5.0 / 3.0])
    assert np.linalg.norm(m - np.array([-0.1213, 0.0, 0.1213])) <= 4 * bw["sigma"] / P0 + 2e-4


@pytest.mark.parametrize("deposit", [0, 1])
def test_b5_forward_equals_backward_on_a_boxwing(oracle, deposit):
    """Box-wing with self-shadowing and inter-reflection, B = 4.  Lambertian + absorbing facets: the two estimators
    estimate the same force.  With specular facets: the same force once the forward tracer leaves out the light whose
    first reflection is specular (no_caustics), which no backward path with a delta sun can find."""
    th = W.draw_params(W.FAMILY_BOXWING, 2)
    sun = np.array([[0.2, 0.9, 0.3], [0.1, -0.95, -0.2]], np.float32)
    for k in range(2):
        v, m = oracle.build_mesh(W.FAMILY_BOXWING, th[k], k=k)
        md = m.copy(); md[:, 2] += md[:, 1]; md[:, 1] = 0.0                       # specular part turned diffuse
        for j in range(2):
            fw = oracle.forces(v, md, sun[j:j + 1], 1 << 17, 4, sampler=1, deposit=deposit, seed=7)
            bw = oracle.backward(v, md, sun[j], 1 << 17, 4, deposit=deposit, seed=7)
            assert np.linalg.norm(bw["F"] - fw["F"][0]) <= 4 * np.hypot(bw["sigma"], fw["sigma"][0]), (k, j)
            assert np.hypot(bw["sigma"], fw["sigma"][0]) < 0.02 * np.linalg.norm(fw["F"][0])
            fs = oracle.forces(v, m, sun[j:j + 1], 1 << 17, 4, sampler=1, deposit=deposit, seed=7, no_caustics=1)
            bs = oracle.backward(v, m, sun[j], 1 << 17, 4, deposit=deposit, seed=7)
            assert np.linalg.norm(bs["F"] - fs["F"][0]) <= 4 * np.hypot(bs["sigma"], fs["sigma"][0]), (k, j)


def test_b6_what_the_backward_estimator_cannot_see(oracle):
    # V-groove of two mirrors (P6): all indirect light is specularly reflected sun light.  Forward: 2 P A_p.
    # Backward: the direct P A_p only -- the documented blind spot (R25), and the reason BASELINE.json asks for the
    # forward form.
    h = np.sqrt(0.5)
    verts = np.concatenate([quad([0, -0.5, 0], [h, 0, h], [0, 1, 0]), quad([0, -0.5, 0], [-h, 0, h], [0, 1, 0])])
    mats = const_mats(4, 0.0, 1.0, 0.0)
    sun = np.array([[0, 0, 1]], np.float32)
    fw = oracle.forces(verts, mats, sun, 1 << 12, 2)
    bw = oracle.backward(verts, mats, sun[0], 1 << 12, 2)
    Ap = np.sqrt(2.0)
    np.testing.assert_allclose(fw["F"][0], [0, 0, -2 * P0 * Ap], rtol=1e-6, atol=1e-13)
    # z: both plates give the same, exactly; x: their contributions cancel only on average (area-proportional sampling)
    np.testing.assert_allclose(bw["F"][2], -1 * P0 * Ap, rtol=1e-7)
    assert abs(bw["F"][0]) <= 4 * bw["sigma"] and bw["F"][1] == 0.0
    nc = oracle.forces(verts, mats, sun, 1 << 12, 2, no_caustics=1)
    np.testing.assert_allclose(nc["F"][0], [0, 0, -1 * P0 * Ap], rtol=1e-6, atol=1e-13)
