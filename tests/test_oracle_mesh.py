"""CPU pins of the oracle's mesh generators against the geometry BASELINE.json's configs state
(sizes, areas, counts) and DESIGN.md "Mesh families".  No GPU."""
import numpy as np
import pytest

from paper_2602_10712_b200 import workloads as W


def areas(verts):
    v = verts.astype(float)
    return 0.5 * np.linalg.norm(np.cross(v[:, 1] - v[:, 0], v[:, 2] - v[:, 0]), axis=1)


def test_triangle_counts(oracle):
    for fam, T in W.TRI_COUNT.items():
        assert oracle.tri_count(fam) == T
        assert oracle.n_params(fam) == W.N_PARAMS[fam]
    assert 49000 <= W.TRI_COUNT[W.FAMILY_DETAILED] <= 51000          # "~50k triangles"
    assert W.TRI_COUNT[W.FAMILY_SAIL] >= 1_000_000 + 19_000          # "1M-triangle sail + 20k bus and booms"


def test_plate_vertices_exact(oracle):
    v, m = oracle.build_mesh(W.FAMILY_PLATE, [0.3, 0.5, 0.2])
    exp = np.array([[[-.5, -.5, 0], [.5, -.5, 0], [.5, .5, 0]], [[-.5, -.5, 0], [.5, .5, 0], [-.5, .5, 0]]],
                   np.float32)
    assert np.array_equal(v, exp)
    assert np.array_equal(m, np.tile(np.array([0.3, 0.5, 0.2], np.float32), (2, 1)))


def test_boxwing_geometry(oracle):
    L, phi = 5.5, 0.6
    v, m = oracle.build_mesh(W.FAMILY_BOXWING, [L, phi])
    a = areas(v)
    bus, pan = v[:12], v[12:]
    assert np.allclose(bus.reshape(-1, 3).min(0), [-.75, -.75, -1]) and np.allclose(bus.reshape(-1, 3).max(0), [.75, .75, 1])
    assert abs(a[:12].sum() - (2 * 1.5 * 1.5 + 4 * 1.5 * 2.0)) < 1e-5   # cuboid 1.5 x 1.5 x 2
    assert np.allclose(a[12:], 0.5 * 1.6 * np.float32(L), rtol=1e-6)    # two 1.6 m wide panels of length L
    py = np.abs(pan.reshape(-1, 3)[:, 1])
    assert abs(py.min() - 1.15) < 1e-6 and abs(py.max() - (1.15 + np.float32(L))) < 1e-5
    n = np.cross(pan[:, 1] - pan[:, 0], pan[:, 2] - pan[:, 0]).astype(float)
    n /= np.linalg.norm(n, axis=1, keepdims=True)
    # panel plane contains y and a(phi) = (cos phi, 0, sin phi) -> normal = +-(-sin phi, 0, cos phi)
    assert np.allclose(np.abs(n @ np.array([-np.sin(phi), 0, np.cos(phi)])), 1.0, atol=1e-6)
    # closed bus: area-weighted outward normals cancel
    nb = 0.5 * np.cross(bus[:, 1] - bus[:, 0], bus[:, 2] - bus[:, 0]).astype(float)
    cen = bus.mean(axis=1)
    nb = np.where((np.sum(nb * cen, axis=1) < 0)[:, None], -nb, nb)
    assert np.abs(nb.sum(0)).max() < 1e-6


def test_boxwing6_geometry_and_materials(oracle):
    th = np.array([0.3, 2.1, 6.0, 1.25, 0.4, 0.3], np.float32)
    v, m = oracle.build_mesh(W.FAMILY_BOXWING6, th)
    assert np.allclose(v[:12].reshape(-1, 3).max(0), [.75, .75, 1.25])
    n = np.cross(v[12:, 1] - v[12:, 0], v[12:, 2] - v[12:, 0]).astype(float)
    n /= np.linalg.norm(n, axis=1, keepdims=True)
    for rows, phi in ((n[:2], 0.3), (n[2:], 2.1)):                     # each panel has its own angle
        assert np.allclose(np.abs(rows @ np.array([-np.sin(phi), 0, np.cos(phi)])), 1.0, atol=1e-6)
    assert np.allclose(m[12:], [0.9 * 0.6, 0.4, 0.1 * 0.6], atol=1e-7)
    assert np.allclose(m[:12], [0.8 * 0.7, 0.2 * 0.7, 0.3], atol=1e-7)
    assert np.allclose(m.sum(1), 1.0, atol=2e-7)


def test_dirichlet_materials_moments(oracle):
    ms = np.concatenate([oracle.build_mesh(W.FAMILY_BOXWING, [4.0, 1.0], k=k, mesh_seed=2)[1] for k in range(400)])
    assert np.allclose(ms.sum(1), 1.0, atol=3e-7) and (ms > 0).all()
    assert np.allclose(ms.mean(0), 1 / 3, atol=0.01)                   # Dirichlet(2,2,2): mean 1/3
    assert np.allclose(ms.var(0), (1 / 3) * (2 / 3) / 7, atol=0.003)   # var = a(a0-a)/(a0^2 (a0+1))
    a = oracle.build_mesh(W.FAMILY_BOXWING, [4.0, 1.0], k=0, mesh_seed=2)[1]
    b = oracle.build_mesh(W.FAMILY_BOXWING, [4.0, 1.0], k=1, mesh_seed=2)[1]
    c = oracle.build_mesh(W.FAMILY_BOXWING, [4.0, 1.0], k=0, mesh_seed=3)[1]
    assert not np.array_equal(a, b) and not np.array_equal(a, c)


def test_detailed_spacecraft_geometry(oracle):
    td, pp = 0.8, 1.9
    v, m = oracle.build_mesh(W.FAMILY_DETAILED, [td, pp])
    a = areas(v)
    assert (a > 0).all()
    off = np.cumsum([0, 6912, 12160, 8704, 20480, 1584])
    bus, dish, cyl, wings, struts = (slice(off[i], off[i + 1]) for i in range(5))
    assert abs(a[bus].sum() - 16.5) < 1e-4
    c, R = 1 / (4 * 0.45), 1.2
    dish_exact = np.pi / (6 * c * c) * ((1 + 4 * c * c * R * R) ** 1.5 - 1)      # paraboloid z = c rho^2
    assert 0.995 * dish_exact < a[dish].sum() < dish_exact
    cyl_exact = 4 * (2 * np.pi * 0.05 * 1.5 + 2 * np.pi * 0.05 ** 2)
    assert 0.995 * cyl_exact < a[cyl].sum() < cyl_exact
    assert abs(a[wings].sum() - 8 * 1.6 * 2.0) < 1e-4
    # dish: apex at (0,0,2.6), axis tilted about x by theta_dish; rim centre = apex + c R^2 * axis
    dv = v[dish].reshape(-1, 3).astype(float)
    assert np.allclose(v[off[1], 0], [0, 0, 2.6])
    rim = dv[np.abs(np.linalg.norm(dv - [0, 0, 2.6], axis=1) - np.sqrt(R * R + (c * R * R) ** 2)) < 1e-5]
    axis = np.array([0, -np.sin(td), np.cos(td)])
    assert np.allclose(rim.mean(0), np.array([0, 0, 2.6]) + c * R * R * axis, atol=1e-5)
    # wings rotate about y by phi_pan and span |y| in [1.15, 1.15 + 4*2.0 + 3*0.1]
    wv = v[wings].reshape(-1, 3)
    assert abs(np.abs(wv[:, 1]).min() - 1.15) < 1e-6 and abs(np.abs(wv[:, 1]).max() - 9.45) < 1e-5
    assert np.abs(wv.astype(float) @ np.array([-np.sin(pp), 0, np.cos(pp)])).max() < 1e-6
    # every edge of the closed parts is shared by exactly two triangles (watertight strut 0)
    s0 = v[off[4]:off[4] + 132]
    keys = {}
    for t in s0:
        for e in range(3):
            k = tuple(sorted((tuple(t[e]), tuple(t[(e + 1) % 3]))))
            keys[k] = keys.get(k, 0) + 1
    assert set(keys.values()) == {2}
    assert np.allclose(m.sum(1), 1.0, atol=3e-7)


@pytest.fixture(scope="module")
def sail(oracle):
    return oracle.build_mesh(W.FAMILY_SAIL, [0.05], mesh_seed=2)


def test_sail_geometry(oracle, sail):
    v, m = sail
    nh = 2 * 707 * 707
    hv = v[:nh].reshape(-1, 3)
    assert np.allclose(hv[:, :2].min(0), -20) and np.allclose(hv[:, :2].max(0), 20)
    assert np.abs(hv[:, 2]).max() <= 0.05                                # amplitude 5 cm
    assert 0.005 < hv[:, 2].std() < 0.03 and abs(hv[:, 2].mean()) < 0.005
    assert len(np.unique(hv, axis=0)) == 708 * 708                       # shared vertices are bit-identical
    assert abs(areas(v[:nh]).sum() - 1600.0) < 1.0                       # wrinkles add < 0.1 % area
    assert np.array_equal(m, np.tile(np.array([0.08, 0.88, 0.04], np.float32), (len(v), 1)))
    bus = v[nh:nh + 19200].reshape(-1, 3)
    assert np.allclose(bus.min(0), [-.5, -.5, -1.2]) and np.allclose(bus.max(0), [.5, .5, -.2])
    booms = v[nh + 19200:].reshape(-1, 3)
    assert len(v) - nh - 19200 == 800
    assert abs(np.abs(booms[:, :2]).max() - 20.0) < 0.03 and abs(booms[:, 2].mean() + 0.1) < 1e-3


def test_sail_noise_depends_on_seed_and_amplitude(oracle, sail):
    nh = 2 * 707 * 707
    flat = oracle.build_mesh(W.FAMILY_SAIL, [0.0], mesh_seed=2)[0]
    assert np.all(flat[:nh, :, 2] == 0)
    assert np.array_equal(flat[nh:], sail[0][nh:])
    other = oracle.build_mesh(W.FAMILY_SAIL, [0.05], mesh_seed=3)[0]
    assert not np.array_equal(other[:nh], sail[0][:nh])
    dbl = oracle.build_mesh(W.FAMILY_SAIL, [0.1], mesh_seed=2)[0]
    assert np.allclose(dbl[:nh, :, 2], 2 * sail[0][:nh, :, 2], atol=1e-8)
