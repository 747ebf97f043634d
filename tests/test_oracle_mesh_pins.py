"""CPU pins of the oracle's mesh generators that do not come from the generator itself (task 2):
the sail's gradient noise, the placement of struts / cylinders / booms, and an independent evaluation of the
PLANE / POLAR / TUBE patch kinds written from DESIGN.md "Mesh families".  No GPU."""
import numpy as np
import pytest

from paper_2602_10712_b200 import workloads as W

NORM = 1.875 * np.sqrt(0.5)          # z = amp * fbm / (1.875 * sqrt(1/2))


def lattice_angle(oracle, ix, iy, octave, seed):
    """2 pi xi, xi from Philox4x32-10 (pinned by the known-answer vectors) at ctr (ix, iy, octave, 0xC0), key
    (seed lo, seed hi); ix, iy in two's complement; uniform map R4 written out here."""
    r = oracle.philox([ix & 0xFFFFFFFF, iy & 0xFFFFFFFF, octave, 0xC0], [seed & 0xFFFFFFFF, seed >> 32])
    xi = ((int(r[0]) >> 9) + 0.5) / 8388608.0
    return 2.0 * np.pi * xi


# ---- sail noise (fbm = sum_{o<4} 2^-o g_o(2^o x/8, 2^o y/8), quintic fade, gradient at angle 2 pi xi) ----

def test_sail_noise_vanishes_on_the_coarsest_lattice(oracle):
    # at (8a, 8b) every octave sits on a lattice corner, where gradient noise is exactly zero
    for a in range(-3, 4):
        for b in range(-3, 4):
            assert oracle.sail_height(8.0 * a, 8.0 * b, 0.05, 2) == 0.0
    assert oracle.sail_height(8.0, -16.0, 0.05, 77) == 0.0


@pytest.mark.parametrize("seed", [2, 5 + (9 << 32)])
@pytest.mark.parametrize("a,b", [(0, 0), (1, -2), (-3, 2)])
def test_sail_noise_half_cell_points(oracle, a, b, seed):
    """Points where only octave 0 contributes (octaves 1-3 sit on lattice corners), expanded by hand:
    fade(1/2) = 1/2, so the value is the mean of the corner dot products."""
    amp = 0.05
    ang = {(i, j): lattice_angle(oracle, a + i, b + j, 0, seed) for i in (0, 1) for j in (0, 1)}
    c = {k: np.cos(v) for k, v in ang.items()}
    s = {k: np.sin(v) for k, v in ang.items()}
    # (8a+4, 8b): fx = 1/2, fy = 0 -> 1/2 [c00 * 1/2] + 1/2 [c10 * (-1/2)]
    exp_x = 0.25 * (c[0, 0] - c[1, 0])
    assert abs(oracle.sail_height(8 * a + 4, 8 * b, amp, seed) - amp * exp_x / NORM) < 1e-15
    # (8a, 8b+4): fx = 0, fy = 1/2
    exp_y = 0.25 * (s[0, 0] - s[0, 1])
    assert abs(oracle.sail_height(8 * a, 8 * b + 4, amp, seed) - amp * exp_y / NORM) < 1e-15
    # (8a+4, 8b+4): all four corners, offsets (+-1/2, +-1/2)
    exp_c = 0.125 * ((c[0, 0] + s[0, 0]) + (-c[1, 0] + s[1, 0]) + (c[0, 1] - s[0, 1]) + (-c[1, 1] - s[1, 1]))
    assert abs(oracle.sail_height(8 * a + 4, 8 * b + 4, amp, seed) - amp * exp_c / NORM) < 1e-15


@pytest.mark.parametrize("a,b", [(0, 0), (-2, 1)])
def test_sail_noise_quarter_cell_point(oracle, a, b):
    """(8a+2, 8b): octave 0 at fx = 1/4 (quintic fade(1/4) = 53/512; the cubic 3t^2 - 2t^3 would give 5/32),
    octave 1 (weight 1/2, lattice (2a, 2b)) at fx = 1/2, octaves 2 and 3 on lattice corners."""
    amp, seed = 0.05, 2
    f = 53.0 / 512.0
    c00, c10 = np.cos(lattice_angle(oracle, a, b, 0, seed)), np.cos(lattice_angle(oracle, a + 1, b, 0, seed))
    o0 = 0.25 * c00 + f * (-0.75 * c10 - 0.25 * c00)
    d00, d10 = np.cos(lattice_angle(oracle, 2 * a, 2 * b, 1, seed)), np.cos(lattice_angle(oracle, 2 * a + 1, 2 * b, 1, seed))
    o1 = 0.25 * (d00 - d10)
    assert abs(oracle.sail_height(8 * a + 2, 8 * b, amp, seed) - amp * (o0 + 0.5 * o1) / NORM) < 1e-15
    # (8a, 8b+1): octave 0 at fy = 1/8, octave 1 at fy = 1/4, octave 2 at fy = 1/2, octave 3 on a corner
    f8 = (1 / 8) ** 3 * ((1 / 8) * ((1 / 8) * 6 - 15) + 10)
    s = lambda i, j, o: np.sin(lattice_angle(oracle, i, j, o, seed))
    p0 = 0.125 * s(a, b, 0) + f8 * (-0.875 * s(a, b + 1, 0) - 0.125 * s(a, b, 0))
    p1 = 0.25 * s(2 * a, 2 * b, 1) + f * (-0.75 * s(2 * a, 2 * b + 1, 1) - 0.25 * s(2 * a, 2 * b, 1))
    p2 = 0.25 * (s(4 * a, 4 * b, 2) - s(4 * a, 4 * b + 1, 2))
    assert abs(oracle.sail_height(8 * a, 8 * b + 1, amp, seed) - amp * (p0 + 0.5 * p1 + 0.25 * p2) / NORM) < 1e-15


def test_sail_noise_gradient_at_a_lattice_point(oracle):
    """Near a corner gradient noise is (lattice gradient) . (offset) up to O(h^3); octave o has weight 2^-o and
    frequency 2^o / 8, so every octave contributes its unit gradient / 8."""
    amp, seed, h = 0.05, 2, 1e-4
    for a, b in ((0, 0), (1, 1), (-2, 0)):
        g = np.zeros(2)
        for o in range(4):
            ang = lattice_angle(oracle, a << o, b << o, o, seed)
            g += np.array([np.cos(ang), np.sin(ang)]) / 8.0
        g *= amp / NORM
        x, y = 8.0 * a, 8.0 * b
        fd = np.array([oracle.sail_height(x + h, y, amp, seed) - oracle.sail_height(x - h, y, amp, seed),
                       oracle.sail_height(x, y + h, amp, seed) - oracle.sail_height(x, y - h, amp, seed)]) / (2 * h)
        assert np.allclose(fd, g, rtol=0, atol=1e-8), (fd, g)


def test_sail_noise_is_c2_across_cell_borders(oracle):
    """The quintic fade has zero first AND second derivative at 0 and 1, so the surface is C2 across the lattice
    lines (a cubic fade leaves a jump in the second derivative).  Third differences straddling the border x = 1
    (a lattice line of the finest octave) stay of the order h^3 * |f'''|."""
    amp, seed, h = 0.05, 2, 1e-3
    y = 0.37
    f = lambda x: oracle.sail_height(x, y, amp, seed)
    d2 = lambda x: (f(x + h) - 2 * f(x) + f(x - h)) / (h * h)
    left, right = d2(1.0 - 2 * h), d2(1.0 + 2 * h)
    inner_l, inner_r = d2(0.6 - 2 * h), d2(0.6 + 2 * h)          # same spacing inside a cell: scale of f''' * 4h
    assert abs(left - right) < 4 * max(abs(inner_l - inner_r), 1e-4)
    assert abs(f(1.0 + 1e-9) - f(1.0 - 1e-9)) < 1e-10            # C0
    d1 = lambda x: (f(x + h) - f(x - h)) / (2 * h)
    assert abs(d1(1.0 - h) - d1(1.0 + h)) < 2 * h * (abs(left) + abs(right) + 1e-3)   # C1


def test_sail_vertices_are_the_height_function(oracle):
    # the HFIELD patch samples sail_height at the PLANE grid points of [-20, 20]^2, 707 x 707 cells
    v, _ = oracle.build_mesh(W.FAMILY_SAIL, [0.05], mesh_seed=2)
    amp = float(np.float32(0.05))                                  # theta is fp32
    for t in (0, 1, 2 * 707 * 350 + 9, 2 * 707 * 707 - 1):
        for c in range(3):
            x, y, z = (float(q) for q in v[t, c])
            i, j = round((x + 20) * 707 / 40), round((y + 20) * 707 / 40)
            xe, ye = -20 + 40 * (i / 707), -20 + 40 * (j / 707)
            assert np.float32(xe) == v[t, c, 0] and np.float32(ye) == v[t, c, 1]
            assert np.float32(oracle.sail_height(xe, ye, amp, 2)) == v[t, c, 2]


# ---- placement of cylinders, struts and booms (DESIGN.md "Mesh families" table) ----

def axis_stats(pts, A, ez):
    """axial coordinate and distance from the axis through A along unit ez, for points [n,3]"""
    d = pts.astype(float) - np.asarray(A, float)
    ax = d @ np.asarray(ez, float)
    rad = np.linalg.norm(d - np.outer(ax, ez), axis=1)
    return ax, rad


def test_detailed_cylinders_and_struts_are_where_design_md_puts_them(oracle):
    td, pp = 0.8, 1.9
    v, _ = oracle.build_mesh(W.FAMILY_DETAILED, [td, pp])
    off = np.cumsum([0, 6912, 12160, 8704, 20480, 1584])
    # 4 capped cylinders r 0.05, length 1.5, from (+-0.5, +-0.5, -1) along -z; each = 64 x 16 tube (2048) + 2 caps (64 + 64)
    sg = [(1, 1), (-1, 1), (-1, -1), (1, -1)]
    for c in range(4):
        part = v[off[2] + 2176 * c: off[2] + 2176 * (c + 1)]
        A = np.array([0.5 * sg[c][0], 0.5 * sg[c][1], -1.0])
        ax, rad = axis_stats(part.reshape(-1, 3), A, [0, 0, -1])
        assert abs(ax.min()) < 1e-6 and abs(ax.max() - 1.5) < 1e-6
        tube = part[:2048].reshape(-1, 3)
        assert np.allclose(axis_stats(tube, A, [0, 0, -1])[1], 0.05, atol=1e-6)
        caps = part[2048:]
        assert np.allclose(caps[:64, 0], A, atol=1e-7) and np.allclose(caps[64:, 0], A + [0, 0, -1.5], atol=1e-6)
        assert len(np.unique(np.round(ax[: 2048 * 3], 5))) == 17                     # 16 segments along the axis
    # 12 capped hexagonal struts r 0.03, 6 x 10 (120) + 2 caps (6 + 6)
    apex = np.array([0, 0, 2.6])
    ends = []
    for s in range(4):
        A = np.array([0.6 * sg[s][0], 0.6 * sg[s][1], 1.0]); ends.append((A, apex))
    for s in range(4, 8):
        sx, sy = (-1.0 if s & 1 else 1.0), (1.0 if s < 6 else -1.0)
        A = np.array([0.3 * sx, 0.75 * sy, 0.0]); ends.append((A, A + [0, 0.4 * sy, 0]))
    for s in range(8, 12):
        sx, sy = (1.0 if s < 10 else -1.0), (-1.0 if s & 1 else 1.0)
        A = np.array([0.75 * sx, 0.4 * sy, 0.5]); ends.append((A, A + [1.0 * sx, 0, 0]))
    seen = set()
    for s, (A, B) in enumerate(ends):
        part = v[off[4] + 132 * s: off[4] + 132 * (s + 1)]
        L = np.linalg.norm(B - A)
        ez = (B - A) / L
        ax, rad = axis_stats(part.reshape(-1, 3), A, ez)
        assert abs(ax.min()) < 1e-6 and abs(ax.max() - L) < 1e-6, s
        assert np.allclose(axis_stats(part[:120].reshape(-1, 3), A, ez)[1], 0.03, atol=1e-6), s
        assert np.allclose(part[120:126, 0], A, atol=1e-6) and np.allclose(part[126:, 0], B, atol=1e-6), s
        seen.add(tuple(np.round(A, 3)))
    assert len(seen) == 12                                                           # twelve distinct feet
    # yoke struts bridge the 0.4 m gap between the bus face (|y| = 0.75) and the first panel (|y| = 1.15)
    assert all(abs(abs(B[1]) - 1.15) < 1e-12 for A, B in ends[4:8])


def test_sail_bus_and_booms_are_where_design_md_puts_them(oracle):
    v, _ = oracle.build_mesh(W.FAMILY_SAIL, [0.05], mesh_seed=2)
    nh = 2 * 707 * 707
    sg = [(1, 1), (-1, 1), (-1, -1), (1, -1)]
    for b in range(4):
        part = v[nh + 19200 + 200 * b: nh + 19200 + 200 * (b + 1)].reshape(-1, 3)
        ez = np.array([sg[b][0], sg[b][1], 0.0]) / np.sqrt(2.0)
        ax, rad = axis_stats(part, [0, 0, -0.1], ez)
        assert abs(ax.min()) < 1e-6 and abs(ax.max() - np.sqrt(800.0)) < 1e-5        # centre -> corner (20, 20)
        assert np.allclose(rad, 0.02 * np.sqrt(2.0), atol=2e-6)                      # square section 0.04 wide
        assert len(np.unique(np.round(ax, 4))) == 26                                 # 25 segments
    # the booms run 5 cm to 15 cm under the sheet (|z| <= 0.05) and clear of the bus top (z = -0.2)
    z = v[nh + 19200:].reshape(-1, 3)[:, 2]
    assert z.max() < -0.05 and z.min() > -0.2


# ---- an independent evaluation of the patch kinds, written from DESIGN.md "Mesh families" ----

def plane_patch(nu, nv, o, ex, ey):
    """PLANE(nu, nv): p(i, j) = o + (i/nu) ex + (j/nv) ey; cell c = j nu + i -> (p00, p10, p11), (p00, p11, p01)."""
    o, ex, ey = (np.asarray(q, float) for q in (o, ex, ey))
    p = lambda i, j: o + (i / nu) * ex + (j / nv) * ey
    tris = []
    for j in range(nv):
        for i in range(nu):
            tris += [[p(i, j), p(i + 1, j), p(i + 1, j + 1)], [p(i, j), p(i + 1, j + 1), p(i, j + 1)]]
    return np.array(tris)


def polar_patch(nr, ns, R, c, o, ex, ey, ez):
    """POLAR(nr, ns, R, c): q = (rho cos phi, rho sin phi, c rho^2), rho = R i / nr, phi = 2 pi (j mod ns) / ns;
    first the apex fan (q(0,0), q(1,j), q(1,j+1)), then rings i = 1 .. nr-1 of quads split like PLANE cells."""
    o, ex, ey, ez = (np.asarray(q, float) for q in (o, ex, ey, ez))

    def q(i, j):
        rho, phi = R * i / nr, 2 * np.pi * (j % ns) / ns
        return o + rho * np.cos(phi) * ex + rho * np.sin(phi) * ey + c * rho * rho * ez
    tris = [[q(0, 0), q(1, j), q(1, j + 1)] for j in range(ns)]
    for i in range(1, nr):
        for j in range(ns):
            tris += [[q(i, j), q(i + 1, j), q(i + 1, j + 1)], [q(i, j), q(i + 1, j + 1), q(i, j + 1)]]
    return np.array(tris)


def tube_patch(ns, nl, r, length, o, ex, ey, ez):
    """TUBE(ns, nl, r, len): q(i, j) = (r cos phi_i, r sin phi_i, len j / nl), phi_i = 2 pi (i mod ns) / ns."""
    o, ex, ey, ez = (np.asarray(q, float) for q in (o, ex, ey, ez))

    def q(i, j):
        phi = 2 * np.pi * (i % ns) / ns
        return o + r * np.cos(phi) * ex + r * np.sin(phi) * ey + (length * j / nl) * ez
    tris = []
    for j in range(nl):
        for i in range(ns):
            tris += [[q(i, j), q(i + 1, j), q(i + 1, j + 1)], [q(i, j), q(i + 1, j + 1), q(i, j + 1)]]
    return np.array(tris)


def ulp_diff(a, b):
    a32, b32 = np.asarray(a, np.float32), np.asarray(b, np.float32)
    return np.abs(a32.astype(np.float64) - b32.astype(np.float64)) / np.maximum(np.spacing(np.abs(b32)), np.float32(1e-45))


def test_patch_kinds_against_an_independent_evaluation(oracle):
    td, pp = 0.8, 1.9
    td32, pp32 = float(np.float32(td)), float(np.float32(pp))
    v, _ = oracle.build_mesh(W.FAMILY_DETAILED, [td, pp])
    off = np.cumsum([0, 6912, 12160, 8704, 20480, 1584])
    # PLANE: the bus' +x face (second face; 24 x 24 cells) spans y, z at x = +0.75
    face = plane_patch(24, 24, [0.75, -0.75, -1.0], [0, 1.5, 0], [0, 0, 2.0])
    assert ulp_diff(v[1152:2304], face).max() <= 2
    # PLANE: panel m = 2 of the -y wing: width 1.6 along a = (cos phi, 0, sin phi), y from -(1.15 + 4.2) outwards
    ca, sa = np.cos(pp32), np.sin(pp32)
    pan = plane_patch(32, 40, [-0.8 * ca, -(1.15 + 2.1 * 2), -0.8 * sa], [1.6 * ca, 0, 1.6 * sa], [0, -2.0, 0])
    assert ulp_diff(v[off[3] + 2560 * 6: off[3] + 2560 * 7], pan).max() <= 2
    # POLAR: the dish, apex (0, 0, 2.6), frame tilted about x by theta_dish
    cd, sd = np.cos(td32), np.sin(td32)
    dish = polar_patch(48, 128, 1.2, 1.0 / (4 * 0.45), [0, 0, 2.6], [1, 0, 0], [0, cd, sd], [0, -sd, cd])
    d = ulp_diff(v[off[1]:off[2]], dish)
    small = np.abs(dish) < 1e-6                  # coordinates that cancel to ~0: compare absolutely
    assert d[~small].max() <= 2 and np.abs(v[off[1]:off[2]][small] - dish[small]).max() < 1e-7
    # TUBE: cylinder 1 at (-0.5, 0.5, -1), frame (x, -y, -z)
    tube = tube_patch(64, 16, 0.05, 1.5, [-0.5, 0.5, -1.0], [1, 0, 0], [0, -1, 0], [0, 0, -1])
    assert ulp_diff(v[off[2] + 2176: off[2] + 2176 + 2048], tube).max() <= 2


# ---- the tie-break of O-step 4 (R11: equal t -> smallest triangle index) ----

def test_equal_t_goes_to_the_smallest_index(oracle):
    plate, _ = oracle.build_mesh(W.FAMILY_PLATE, [0.3, 0.5, 0.2])
    black, mirror = [1.0, 0.0, 0.0], [0.0, 1.0, 0.0]
    sun = np.array([[0.3, -0.2, 0.9]], np.float32)
    s = -sun[0].astype(float) / np.linalg.norm(sun[0].astype(float))
    for first, second in ((black, mirror), (mirror, black)):
        verts = np.concatenate([plate, plate])                   # triangles 2, 3 coincide with 0, 1
        mats = np.array([first, first, second, second], np.float32)
        r = oracle.forces(verts, mats, sun, 4096, 0, want_first_hit=True)
        fh = r["first_hit"]
        assert set(np.unique(fh)) == {-1, 0, 1}                  # misses, or the first copy; never 2 or 3
        alone = oracle.forces(plate, np.array([first, first], np.float32), sun, 4096, 0)
        assert np.array_equal(r["F"], alone["F"])
        # and the two materials do give different forces, so the choice is visible
        other = oracle.forces(plate, np.array([second, second], np.float32), sun, 4096, 0)
        assert np.linalg.norm(other["F"] - alone["F"]) > 0.1 * np.linalg.norm(alone["F"])
