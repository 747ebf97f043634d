"""GPU parity tests: the CUDA path, called through the C ABI (ctypes binding), against the CPU
oracle on the same seeded inputs.  Tolerances are BASELINE.json's: per-vector relative L2 <= 1e-4
when no ray diverged, else <= 1e-3 aggregate and within 4 sigma (helpers.assert_parity); integer
work (meshes up to 2 ulp, counters, hit ids) exactly or up to the counted divergent rays."""
import numpy as np
import pytest

from paper_2602_10712_b200 import workloads as W
from helpers import (P0, quad, const_mats, unit, flat_plate_force, convex_polyhedron_force, rel_l2,
                     oracle_pairs, assert_parity)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2602_10712_b200.binding import Context
    c = Context(0)
    yield c
    c.close()


def cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def ulp_diff(a, b):
    return np.abs(a.view(np.int32).astype(np.int64) - b.view(np.int32).astype(np.int64))


# ---------------------------------------------------------------- S0: mesh generator
@pytest.mark.parametrize("family", [W.FAMILY_PLATE, W.FAMILY_BOXWING, W.FAMILY_DETAILED,
                                    W.FAMILY_BOXWING6, W.FAMILY_SAIL, W.FAMILY_BOXWING_T])
def test_mesh_generator_matches_oracle(ctx, oracle, family):
    D = 3 if family != W.FAMILY_SAIL else 1
    th = W.draw_params(family, D)
    dz = ctx.srp_build_designs(family, th, mesh_seed=W.MESH_SEED)
    assert dz.D == D and np.array_equal(np.diff(dz.tri_offsets), [W.TRI_COUNT[family]] * D)
    k = D - 1
    v, m = dz.read_mesh(k)
    ov, om = oracle.build_mesh(family, th[k], k=k, mesh_seed=W.MESH_SEED)
    assert ulp_diff(v, ov).max() <= 2 and (v != ov).mean() < 1e-4       # fp64 evaluation on both sides
    assert ulp_diff(m, om).max() <= 2
    dz.free()


# ---------------------------------------------------------------- S1: LBVH structure
def check_bvh(nodes, perm, verts):
    T = len(perm)
    assert sorted(perm.tolist()) == list(range(T))                       # a permutation
    link = nodes[:, 12:14].copy().view(np.int32)
    seen = np.zeros(T, np.int32)
    stack = [(0, None, None)]
    n_visited = 0
    tri_lo = verts.min(axis=1)[perm]                                      # boxes of sorted triangles
    tri_hi = verts.max(axis=1)[perm]
    while stack:
        n, plo, phi = stack.pop()
        n_visited += 1
        for side in range(2):
            lo, hi = nodes[n, 6 * side:6 * side + 3], nodes[n, 6 * side + 3:6 * side + 6]
            if plo is not None and not (hi < lo).any():
                assert (lo >= plo - 1e-6).all() and (hi <= phi + 1e-6).all()   # child box inside parent box
            l = int(link[n, side])
            if l >= 0:
                stack.append((l, lo, hi))
            else:
                u = ~l
                first, cnt = u >> 3, (u & 7) + 1
                if (hi < lo).any():
                    continue                                              # empty box of a 1-triangle design
                seen[first:first + cnt] += 1
                eps = 1e-6 * (1 + np.abs(tri_hi[first:first + cnt]).max())
                assert (tri_lo[first:first + cnt] >= lo - eps).all() and (tri_hi[first:first + cnt] <= hi + eps).all()
    assert (seen == 1).all()                                              # every triangle in exactly one leaf
    return n_visited


def sah_cost(nodes):
    """Surface-area-heuristic cost of the tree: sum over reachable inner children of their box area plus, over leaf
    children, box area x triangles, in units of the root box's area."""
    link = nodes[:, 12:14].copy().view(np.int32)
    def area(lo, hi):
        d = np.maximum(hi - lo, 0.0)
        return d[0] * d[1] + d[1] * d[2] + d[0] * d[2]
    root = area(np.minimum(nodes[0, 0:3], nodes[0, 6:9]), np.maximum(nodes[0, 3:6], nodes[0, 9:12]))
    cost, stack = root, [0]
    while stack:
        n = stack.pop()
        for side in range(2):
            a = area(nodes[n, 6 * side:6 * side + 3], nodes[n, 6 * side + 3:6 * side + 6])
            l = int(link[n, side])
            if l >= 0:
                cost += a; stack.append(l)
            else:
                cost += a * (((~l) & 7) + 1)
    return cost / root


@pytest.mark.parametrize("builder", [0, 1])
def test_bvh_structure_detailed(ctx, builder):
    """Both builders (srp_options.bvh_builder: binned SAH, linear BVH): a permutation of the triangles, every triangle in
    exactly one leaf, every box inside its parent's and around its triangles."""
    th = W.draw_params(W.FAMILY_DETAILED, 2)
    ctx.srp_set_options(bvh_builder=builder)
    try:
        dz = ctx.srp_build_designs(W.FAMILY_DETAILED, th)
    finally:
        ctx.srp_set_options()
    for k in range(2):
        nodes, perm = dz.read_bvh(k)
        v, _ = dz.read_mesh(k)
        assert len(nodes) == len(perm) - 1                                # T-1 internal node records
        visited = check_bvh(nodes, perm, v)
        assert visited <= len(nodes)
    dz.free()


def test_sah_builder_is_reproducible_and_cheaper_than_lbvh(ctx):
    """Two builds give the same bytes (integer atomics and a scan: no dependence on arrival order); the SAH cost of
    the binned builder's tree is well below the linear BVH's on the detailed design; both give the same forces up to
    the photons whose closest hit is a tie."""
    th = W.draw_params(W.FAMILY_DETAILED, 1)
    sun = cuda(W.fibonacci_sphere(4))
    out = {}
    for builder in (0, 0, 1):
        ctx.srp_set_options(bvh_builder=builder)
        try:
            dz = ctx.srp_build_designs(W.FAMILY_DETAILED, th)
        finally:
            ctx.srp_set_options()
        nodes, perm = dz.read_bvh(0)
        F = ctx.srp_forces(dz, sun, 1 << 16, 4, 0).cpu().numpy()
        out.setdefault(builder, []).append((nodes, perm, F))
        dz.free()
    (n0, p0, F0), (n1, p1, F1) = out[0]
    assert np.array_equal(n0.view(np.uint32), n1.view(np.uint32)) and np.array_equal(p0, p1) and np.array_equal(F0, F1)
    nl, pl, Fl = out[1][0]
    c_sah, c_lbvh = sah_cost(n0), sah_cost(nl)
    assert c_sah < 0.8 * c_lbvh, (c_sah, c_lbvh)
    assert np.linalg.norm(F0 - Fl) <= 5e-4 * np.linalg.norm(Fl)          # a photon is 1e-4 of a force here


def test_small_designs_have_no_hierarchy(ctx):
    dz = ctx.srp_build_designs(W.FAMILY_BOXWING, W.draw_params(W.FAMILY_BOXWING, 4))
    nodes, perm = dz.read_bvh(2)
    assert len(nodes) == 0 and np.array_equal(perm, np.arange(16))
    dz.free()


@pytest.mark.parametrize("builder", [0, 1])
def test_bvh_mixed_sizes_and_duplicates(ctx, builder):
    """from_meshes with 1, 2, 3, 70 and 500 triangles in one batch; the 70 are 70 copies of one triangle
    (identical Morton keys -> index tie-break; identical centroids -> the SAH builder halves them by position)."""
    rng = np.random.default_rng(0)
    one = quad([0, 0, 0], [1, 0, 0], [0, 1, 0])[:1]
    three = rng.normal(size=(3, 3, 3)).astype(np.float32)
    dup = np.repeat(one, 70, axis=0)
    big = (rng.normal(size=(500, 1, 3)) + 0.1 * rng.normal(size=(500, 3, 3))).astype(np.float32)
    two = rng.normal(size=(2, 3, 3)).astype(np.float32)
    verts = np.concatenate([one, two, three, dup, big])
    mats = W.dirichlet_materials(len(verts), 1)
    off = np.cumsum([0, 1, 2, 3, 70, 500])
    ctx.srp_set_options(bvh_builder=builder)
    try:
        dz = ctx.srp_build_designs_from_meshes(verts, mats, off)
    finally:
        ctx.srp_set_options()
    for k in range(5):
        nodes, perm = dz.read_bvh(k)
        check_bvh(nodes, perm, verts[off[k]:off[k + 1]])
    dz.free()


@pytest.mark.parametrize("primary_mode,masks", [(1, 0), (2, 0), (1, 2), (2, 2)])
def test_forces_on_mixed_batch_match_oracle(ctx, oracle, primary_mode, masks):
    """One batch with a hierarchy holding designs of 1, 3, 70 (identical copies) and 500 random triangles: forces of
    every design against the oracle, per-ray and as beams (one-triangle root, empty child slot, equal Morton keys)."""
    rng = np.random.default_rng(0)
    one = quad([0, 0, 0], [1, 0, 0], [0, 1, 0])[:1]
    three = rng.normal(size=(3, 3, 3)).astype(np.float32)
    dup = np.repeat(one, 70, axis=0)
    big = (rng.normal(size=(500, 1, 3)) + 0.1 * rng.normal(size=(500, 3, 3))).astype(np.float32)
    verts = np.concatenate([one, three, dup, big])
    mats = W.dirichlet_materials(len(verts), 1)
    off = np.cumsum([0, 1, 3, 70, 500])
    dz = ctx.srp_build_designs_from_meshes(verts, mats, off)
    sun = W.fibonacci_sphere(6)
    N, B = 1 << 12, 3
    ctx.srp_set_options(primary_mode=primary_mode, escape_masks=masks)
    try:
        F = ctx.srp_forces(dz, cuda(sun), N, B, 4).cpu().numpy()
        st = ctx.srp_get_stats()
    finally:
        ctx.srp_set_options()
    assert st["launched"] == st["primary_miss"] + st["absorbed"] + st["escaped"] + st["capped"]
    for k in range(4):
        if k == 2:
            continue          # 70 coincident triangles: every hit is a 70-way tie in t, the winner is not unique (R11)
        r = oracle.forces(verts[off[k]:off[k + 1]], mats[off[k]:off[k + 1]], sun, N, B, seed=4, k=k)
        assert_parity(F[k], r["F"], r["sigma"], tol_agg=5e-3)
    # the coincident copies: whichever copy wins, the hit geometry is the plate's; materials differ per copy, so only
    # the direction-independent bound |F| <= 2 P A cos(theta) is checked
    for j in range(len(sun)):
        cos = abs(sun[j][2]) / np.linalg.norm(sun[j])
        assert np.linalg.norm(F[2, j]) <= 2.0 * P0 * 0.5 * cos * (1 + 1e-3) + 1e-12
    dz.free()


# ---------------------------------------------------------------- S3/S4: rays and closest hit
@pytest.mark.parametrize("family,N", [(W.FAMILY_BOXWING, 1 << 12), (W.FAMILY_DETAILED, 1 << 12),
                                      (W.FAMILY_SAIL, 1 << 10)])
def test_first_hits_bvh_equals_brute_equals_oracle(ctx, oracle, family, N):
    th = W.draw_params(family, 1)
    dz = ctx.srp_build_designs(family, th)
    sun = W.fibonacci_sphere(5)[1:4]
    pairs = np.array([[0, 0], [0, 1], [0, 2]], np.int32)
    a = ctx.srp_first_hits(dz, cuda(sun), pairs, N, seed=3, method=0).cpu().numpy()
    b = ctx.srp_first_hits(dz, cuda(sun), pairs, N, seed=3, method=1).cpu().numpy()
    ov, om = oracle.build_mesh(family, th[0], k=0)
    o = oracle.forces(ov, om, sun, N, 0, seed=3, k=0, want_first_hit=True)["first_hit"]
    # rays through an edge shared by two triangles may resolve either way in fp32: allow a handful
    assert (a != b).sum() <= 2
    assert (a != o).mean() <= 1e-3
    hit = o >= 0
    assert hit.any() and (~hit).any()
    assert ((a >= 0) != hit).sum() <= 2                                   # same silhouette
    dz.free()


# ---------------------------------------------------------------- S2-S7: forces, config slices
def run_pairs(ctx, dz, sun, pairs, N, B, seed=0):
    F = ctx.srp_forces_pairs(dz, cuda(sun), pairs, N, B, seed).cpu().numpy()
    return F, ctx.srp_get_stats()


def counters_close(st, ost, tol):
    for key in ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments"):
        assert abs(st[key] - ost[key]) <= tol, (key, st[key], ost[key])
    assert st["launched"] == ost["launched"]
    assert st["launched"] == st["primary_miss"] + st["absorbed"] + st["escaped"] + st["capped"]   # P8
    assert st["segments"] == sum(st["hits_at_depth"]) + st["primary_miss"] + st["escaped"]


def test_cfg1_flat_plate_full(ctx, oracle):
    cfg = W.CONFIGS["cfg1_plate"]
    th, sun = cfg.params(), cfg.sun_dirs()
    dz = ctx.srp_build_designs(cfg.family, th)
    F = ctx.srp_forces(dz, cuda(sun), cfg.N, cfg.B, cfg.seed).cpu().numpy()[0]
    st = ctx.srp_get_stats()
    ov, om = oracle.build_mesh(cfg.family, th[0])
    r = oracle.forces(ov, om, sun, cfg.N, cfg.B, seed=cfg.seed)
    assert assert_parity(F, r["F"], r["sigma"]) == 0
    assert rel_l2(F, r["F"]).max() < 1e-5
    counters_close(st, r["stats"], tol=2)
    for j in range(cfg.S):                                               # and the closed form itself
        Fc = flat_plate_force(sun[j], [0, 0, 1], 1.0, 0.3, 0.5, 0.2)
        if sun[j][2] > 0.1:
            assert np.linalg.norm(F[j] - Fc) < 3e-3 * np.linalg.norm(Fc)
    dz.free()


@pytest.mark.parametrize("name,n_pairs", [("cfg2_boxwing", 256), ("cfg4_sweep", 256)])
def test_small_design_configs_full_N(ctx, oracle, name, n_pairs):
    cfg = W.CONFIGS[name]
    th, sun = cfg.params(), cfg.sun_dirs()
    dz = ctx.srp_build_designs(cfg.family, th)
    rng = np.random.default_rng(5)
    pairs = np.stack([rng.integers(0, cfg.D, n_pairs), rng.integers(0, cfg.S, n_pairs)], 1).astype(np.int32)
    F, st = run_pairs(ctx, dz, sun, pairs, cfg.N, cfg.B, cfg.seed)
    meshes = {int(k): oracle.build_mesh(cfg.family, th[k], k=int(k)) for k in np.unique(pairs[:, 0])}
    Fo, sig, ost = oracle_pairs(oracle, meshes, pairs, sun, cfg.N, cfg.B, seed=cfg.seed)
    n_div = assert_parity(F, Fo, sig)
    assert n_div <= n_pairs // 20
    counters_close(st, ost, tol=n_pairs)            # <= ~1 divergent ray per pair at these sizes
    assert sum(st["hits_at_depth"][1:]) > 0         # bounces do happen (panel <-> bus)
    # the full job runs with the escape masks (above the photons-per-triangle rule; these sampled pairs are below
    # it, so the masks are forced): same photons and counters, same parity with the oracle
    assert st["mask_escapes"] == 0
    ctx.srp_set_options(escape_masks=2)
    try:
        Fm, sm = run_pairs(ctx, dz, sun, pairs, cfg.N, cfg.B, cfg.seed)
    finally:
        ctx.srp_set_options()
    for key in ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments", "hits_at_depth"):
        assert sm[key] == st[key], key
    assert sm["mask_escapes"] > 0.4 * sm["escaped"]
    assert np.abs(Fm - F).max() <= 2e-6 * np.abs(F).max()
    assert_parity(Fm, Fo, sig)
    dz.free()


@pytest.mark.parametrize("primary_mode,masks", [(1, 0), (2, 0), (1, 2), (2, 2)])   # primaries one by one / as beams
def test_cfg3_detailed_reduced_N(ctx, oracle, primary_mode, masks):                  # (auto picks by N / T); escape masks off / forced
    cfg = W.CONFIGS["cfg3_detailed"]
    th, sun = cfg.params(), cfg.sun_dirs()
    dz = ctx.srp_build_designs(cfg.family, th)
    N = 1 << 12
    rng = np.random.default_rng(6)
    pairs = np.stack([np.arange(cfg.D), rng.integers(0, cfg.S, cfg.D)], 1).astype(np.int32)   # one per design
    ctx.srp_set_options(primary_mode=primary_mode, escape_masks=masks)
    try:
        F, st = run_pairs(ctx, dz, sun, pairs, N, cfg.B, cfg.seed)
        psig = ctx.srp_path_signatures(dz, cuda(sun), pairs, N, cfg.B, cfg.seed).cpu().numpy().astype(np.uint64)
    finally:
        ctx.srp_set_options()
    assert (st["mask_escapes"] > 0.3 * st["escaped"]) if masks else st["mask_escapes"] == 0
    if primary_mode == 2:
        assert st["beam_tile_miss"] + st["beam_block_miss"] + st["beam_group_miss"] > 0.5 * st["launched"]
    else:
        assert st["beam_tile_miss"] + st["beam_block_miss"] + st["beam_group_miss"] + st["beam_fallback"] == 0
    meshes = {k: oracle.build_mesh(cfg.family, th[k], k=k) for k in range(cfg.D)}
    Fo, sig, ost, osig = oracle_pairs(oracle, meshes, pairs, sun, N, cfg.B, seed=cfg.seed, want_path_sig=True)
    n_div = (psig != osig).sum(axis=1)                     # divergent rays per pair
    print("cfg3 reduced N: divergent rays per pair", n_div.tolist())
    # fp32 hit points are ~1e-6 m off; with 2.5 cm dish facets a few photons per 1e5 segments cross a
    # facet edge the other way (measured: 3 of 65536 here).  BASELINE.json allows exactly this.
    assert n_div.sum() <= 8                                 # of 65536 photons
    assert_parity(F, Fo, sig, diverged=n_div > 0, tol_agg=1e-3 if n_div.sum() == 0 else 3e-3)
    counters_close(st, ost, tol=16)
    # the hierarchy changes nothing: brute force over all triangles gives the same forces
    ctx.srp_set_options(force_brute=1)
    Fb, stb = run_pairs(ctx, dz, sun, pairs[:4], N, cfg.B, cfg.seed)
    ctx.srp_set_options()
    assert rel_l2(Fb, F[:4]).max() < 1e-4
    dz.free()


@pytest.mark.parametrize("primary_mode,masks", [(1, 0), (2, 0), (1, 2)])
def test_cfg5_sail_reduced_N(ctx, oracle, primary_mode, masks):
    cfg = W.CONFIGS["cfg5_sail"]
    th = cfg.params()
    dz = ctx.srp_build_designs(cfg.family, th)
    N = 1 << 10
    # two grazing directions, two oblique, near-normal from both sides
    sun = np.array([[1, 0.2, 0.02], [0.3, -1, -0.03], [0.5, 0.4, 0.7], [-0.2, 0.6, -0.6],
                    [0.05, 0.02, 1], [0.01, -0.03, -1]], np.float32)
    pairs = np.stack([np.zeros(len(sun)), np.arange(len(sun))], 1).astype(np.int32)
    ctx.srp_set_options(primary_mode=primary_mode, escape_masks=masks)   # 2: ~1000 triangles per ray, every beam list overflows
    try:
        F, st = run_pairs(ctx, dz, sun, pairs, N, cfg.B, cfg.seed)
        psig = ctx.srp_path_signatures(dz, cuda(sun), pairs, N, cfg.B, cfg.seed).cpu().numpy().astype(np.uint64)
    finally:
        ctx.srp_set_options()
    meshes = {0: oracle.build_mesh(cfg.family, th[0], k=0)}
    Fo, sig, ost, osig = oracle_pairs(oracle, meshes, pairs, sun, N, cfg.B, seed=cfg.seed, want_path_sig=True)
    n_div = (psig != osig).sum(axis=1)
    print("cfg5 reduced N: divergent rays per pair", n_div.tolist())
    assert n_div.sum() <= 6
    # at N = 2^10 one photon is ~1e-3 of a force vector, so the aggregate bound scales with it
    assert_parity(F, Fo, sig, diverged=n_div > 0, tol_agg=1e-3 if n_div.sum() == 0 else 5e-3)
    counters_close(st, ost, tol=8)
    dz.free()


def test_sail_flat_limit_closed_form(ctx):
    """amplitude 0: the sail is a 40 x 40 m mirror-like plate; sun from +z sees only the sail (P2)."""
    dz = ctx.srp_build_designs(W.FAMILY_SAIL, np.array([[0.0]], np.float32))
    om = np.array([[0.1, 0.05, 1.0]], np.float32)
    F = ctx.srp_forces(dz, cuda(om), 1 << 16, 8, 0).cpu().numpy()[0, 0]
    Fc = flat_plate_force(om[0], [0, 0, 1], 1600.0, 0.08, 0.88, 0.04)
    assert np.linalg.norm(F - Fc) < 5e-3 * np.linalg.norm(Fc)
    dz.free()


# ---------------------------------------------------------------- closed forms through the CUDA path
def test_v_groove_on_gpu(ctx):
    h = np.sqrt(0.5)
    verts = np.concatenate([quad([0, -0.5, 0], [h, 0, h], [0, 1, 0]), quad([0, -0.5, 0], [-h, 0, h], [0, 1, 0])])
    dz = ctx.srp_build_designs_from_meshes(verts, const_mats(4, 0, 1, 0), [0, 4])
    om = cuda(np.array([[0, 0, 1]], np.float32))
    for B, factor, fate in ((0, 1.0, "capped"), (1, 2.0, "capped"), (2, 2.0, "escaped")):
        F = ctx.srp_forces(dz, om, 1 << 14, B, 0).cpu().numpy()[0, 0]
        np.testing.assert_allclose(F, [0, 0, -factor * P0 * np.sqrt(2.0)], rtol=2e-6, atol=1e-12)
        st = ctx.srp_get_stats()
        assert st["primary_miss"] == 0 and st[fate] == st["launched"] == 1 << 14
    dz.free()


def test_convex_polyhedron_with_bvh_on_gpu(ctx):
    verts = W.icosphere(3, 1.3)                                           # 1280 facets -> LBVH path
    mats = W.dirichlet_materials(len(verts), 7)
    dz = ctx.srp_build_designs_from_meshes(verts, mats, [0, len(verts)])
    sun = W.fibonacci_sphere(12)
    F = ctx.srp_forces(dz, cuda(sun), 1 << 18, 3, 1).cpu().numpy()[0]
    st = ctx.srp_get_stats()
    for j in range(len(sun)):
        Fc = convex_polyhedron_force(verts, mats, sun[j])
        assert rel_l2(F[j], Fc) < 1e-3
    # convex: nothing is hit twice -- except the ~1e-7 of fp32 rays that slip through the seam between two
    # facets (edge vectors are rounded) and bounce inside; counted, and bounded at 1e-5 of the hits
    assert sum(st["hits_at_depth"][1:]) <= 1e-5 * st["hits_at_depth"][0] and st["capped"] <= 2
    dz.free()


def test_occluded_facet_on_gpu(ctx):
    front = quad([-1, -1, 1.0], [2, 0, 0], [0, 2, 0])
    back = quad([-0.3, -0.3, 0.0], [0.6, 0, 0], [0, 0.6, 0])
    verts = np.concatenate([back, front])
    mats = np.concatenate([const_mats(2, 0.1, 0.8, 0.1), const_mats(2, 1, 0, 0)])
    dz = ctx.srp_build_designs_from_meshes(verts, mats, [0, 4])
    om = np.array([[0.05, 0.02, 1.0]], np.float32)
    prim = ctx.srp_first_hits(dz, cuda(om), np.array([[0, 0]], np.int32), 1 << 14, seed=0, method=0).cpu().numpy()
    assert not np.isin(prim, [0, 1]).any()
    F = ctx.srp_forces(dz, cuda(om), 1 << 14, 2, 0).cpu().numpy()[0, 0]
    Fc = flat_plate_force(om[0], [0, 0, 1], 4.0, 1.0, 0.0, 0.0)
    assert np.linalg.norm(F - Fc) < 3e-3 * np.linalg.norm(Fc)
    dz.free()


# ---------------------------------------------------------------- modes, determinism, API behaviour
@pytest.mark.parametrize("sampler,deposit,N", [(1, 0, 50000), (0, 1, 1 << 16), (1, 1, 1 << 16)])
def test_sampler_and_deposit_modes_match_oracle(ctx, oracle, sampler, deposit, N):
    th = W.draw_params(W.FAMILY_BOXWING, 3)
    sun = W.fibonacci_sphere(7)
    dz = ctx.srp_build_designs(W.FAMILY_BOXWING, th)
    ctx.srp_set_options(sampler=sampler, deposit=deposit, solar_pressure=9.12e-6)
    try:
        pairs = np.array([[k, j] for k in range(3) for j in range(7)], np.int32)
        F, st = run_pairs(ctx, dz, sun, pairs, N, 4, seed=11)
    finally:
        ctx.srp_set_options()
    meshes = {k: oracle.build_mesh(W.FAMILY_BOXWING, th[k], k=k) for k in range(3)}
    Fo, sig, ost = oracle_pairs(oracle, meshes, pairs, sun, N, 4, seed=11, sampler=sampler, deposit=deposit, P=9.12e-6)
    assert_parity(F, Fo, sig)
    counters_close(st, ost, tol=8)
    dz.free()


def test_bit_reproducible_and_pairs_equal_full(ctx):
    th = W.draw_params(W.FAMILY_DETAILED, 2)
    sun = cuda(W.fibonacci_sphere(16))
    dz = ctx.srp_build_designs(W.FAMILY_DETAILED, th)
    a = ctx.srp_forces(dz, sun, 1 << 14, 8, 2).cpu().numpy()
    b = ctx.srp_forces(dz, sun, 1 << 14, 8, 2).cpu().numpy()
    assert np.array_equal(a, b)                                          # integer accumulation: any schedule
    pairs = np.array([[1, 5], [0, 15], [1, 0]], np.int32)
    c = ctx.srp_forces_pairs(dz, sun, pairs, 1 << 14, 8, 2).cpu().numpy()
    assert np.array_equal(c, a[pairs[:, 0], pairs[:, 1]])
    d = ctx.srp_forces(dz, sun, 1 << 14, 8, 3).cpu().numpy()
    assert not np.array_equal(a, d)                                      # the seed matters
    dz.free()


def test_host_api_equals_device_api(ctx):
    th = W.draw_params(W.FAMILY_BOXWING6, 5)
    sun = W.fibonacci_sphere(9)
    dz = ctx.srp_build_designs(W.FAMILY_BOXWING6, th)
    a = ctx.srp_forces(dz, cuda(sun), 1 << 12, 4, 0).cpu().numpy()
    b = ctx.srp_forces_host(dz, sun, 1 << 12, 4, 0).numpy()
    assert np.array_equal(a, b)
    dz.free()


def test_edge_cases(ctx, oracle):
    from paper_2602_10712_b200.binding import SrpError
    th = W.draw_params(W.FAMILY_PLATE, 1)
    dz = ctx.srp_build_designs(W.FAMILY_PLATE, th)
    om = cuda(np.array([[1, 0, 0], [0, 0, 2.5], [0, 3, 0]], np.float32))      # edge-on, unnormalised, edge-on
    F = ctx.srp_forces(dz, om, 1 << 10, 0, 0).cpu().numpy()[0]
    assert np.all(F[0] == 0) and np.all(F[2] == 0)
    assert ctx.srp_get_stats()["launched"] == 1 << 10                    # edge-on pairs launch nothing
    np.testing.assert_allclose(F[1], flat_plate_force([0, 0, 1], [0, 0, 1], 1.0, 0.3, 0.5, 0.2), rtol=1e-5)
    F15 = ctx.srp_forces(dz, om, 1 << 10, 15, 0).cpu().numpy()[0]
    assert np.array_equal(F15, F)                                        # a plate never bounces twice
    with pytest.raises(SrpError):
        ctx.srp_forces(dz, om, 1000, 1, 0)                               # stratified needs 2^m
    with pytest.raises(SrpError):
        ctx.srp_forces(dz, om, 1 << 10, 16, 0)
    with pytest.raises(SrpError):
        ctx.srp_forces(dz, om, 0, 1, 0)
    with pytest.raises(SrpError):
        ctx.srp_build_designs(W.FAMILY_BOXWING, th)                      # wrong n_params
    with pytest.raises(SrpError):
        ctx.srp_build_designs(7, th)
    with pytest.raises(SrpError):
        ctx.srp_set_options(primary_mode=3)
    ctx.srp_set_options(instrumented=1)
    try:
        with pytest.raises(SrpError):                                    # torques come from the plain kernels only
            ctx.srp_forces_torques(dz, om, 1 << 10, 1, 0)
    finally:
        ctx.srp_set_options()
    ctx.srp_set_options(sampler=1)
    try:
        Fi = ctx.srp_forces(dz, om, 1000, 1, 0).cpu().numpy()[0]         # ragged N in i.i.d. mode
        assert ctx.srp_get_stats()["launched"] == 1000
    finally:
        ctx.srp_set_options()
    ov, omat = oracle.build_mesh(W.FAMILY_PLATE, th[0])
    r = oracle.forces(ov, omat, np.array([[0, 0, 2.5]], np.float32), 1000, 1, j0=1, sampler=1)
    assert rel_l2(Fi[1], r["F"][0]) < 1e-5
    dz.free()


def test_beams_equal_per_ray_primaries(ctx):
    """The beam tracer (shared BVH descent per block of rays, 2-D edge-function tests in the emitter frame,
    pooled bounce rays) follows the same photons as per-ray traversal: identical path signatures up to a
    handful of rays on facet edges, identical counters up to those, forces to 1e-6, on N from 1 ray
    (one lane) over ragged sub-blocks to several tiles, and on a sphere seen from 12 sides."""
    th = W.draw_params(W.FAMILY_DETAILED, 2)
    dz = ctx.srp_build_designs(W.FAMILY_DETAILED, th)
    sun = W.fibonacci_sphere(6)
    pairs = np.array([[k, j] for k in range(2) for j in range(6)], np.int32)
    for N, B in ((1, 2), (8, 2), (1 << 6, 3), (1 << 9, 8), (1 << 15, 8)):
        res = {}
        for mode in (1, 2):
            ctx.srp_set_options(primary_mode=mode)
            try:
                F, st = run_pairs(ctx, dz, sun, pairs, N, B, seed=5)
                sg = ctx.srp_path_signatures(dz, cuda(sun), pairs, N, B, 5).cpu().numpy().astype(np.uint64)
            finally:
                ctx.srp_set_options()
            res[mode] = (F, st, sg)
        n_div = int((res[1][2] != res[2][2]).sum())
        assert n_div <= max(2, N * len(pairs) // 100000), (N, n_div)
        for key in ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments"):
            assert abs(res[1][1][key] - res[2][1][key]) <= 4 * n_div, (N, key)
        assert res[2][1]["launched"] == N * len(pairs)
        if n_div == 0 and N >= 64:
            assert rel_l2(res[2][0], res[1][0]).max() < 1e-5
    dz.free()


@pytest.mark.parametrize("family,D,S,N,B", [(W.FAMILY_BOXWING, 8, 12, 1 << 14, 4), (W.FAMILY_BOXWING6, 8, 12, 1 << 16, 4),
                                            (W.FAMILY_PLATE, 1, 12, 1 << 10, 1), (W.FAMILY_BOXWING, 2, 5, 1, 4),
                                            (W.FAMILY_BOXWING, 2, 5, 16, 4)])
def test_small_design_beams_equal_brute_force(ctx, family, D, S, N, B):
    """Designs without a hierarchy: the tile / sub-block / group culling and the 2-D edge-function test of the
    primaries (small_beam_kernel) against Moller-Trumbore over all triangles for every segment (primary_mode 1)."""
    th = W.draw_params(family, D)
    sun = W.fibonacci_sphere(S)
    dz = ctx.srp_build_designs(family, th)
    pairs = np.array([[k, j] for k in range(D) for j in range(S)], np.int32)
    res = {}
    for mode in (0, 1):
        ctx.srp_set_options(primary_mode=mode)
        try:
            F, st = run_pairs(ctx, dz, sun, pairs, N, B, seed=4)
            sg = ctx.srp_path_signatures(dz, cuda(sun), pairs, N, B, 4).cpu().numpy().astype(np.uint64)
        finally:
            ctx.srp_set_options()
        res[mode] = (F, st, sg)
    n_div = int((res[0][2] != res[1][2]).sum())
    assert n_div <= max(1, N * len(pairs) // 1000000), n_div
    for key in ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments"):
        assert abs(res[0][1][key] - res[1][1][key]) <= 4 * n_div, key
    assert res[1][1]["beam_tile_miss"] + res[1][1]["beam_block_miss"] + res[1][1]["beam_group_miss"] == 0
    if N >= 1 << 10:
        assert res[0][1]["beam_tile_miss"] + res[0][1]["beam_block_miss"] + res[0][1]["beam_group_miss"] > 0
        nrm = np.linalg.norm(res[1][0], axis=1)
        err = np.linalg.norm(res[0][0] - res[1][0], axis=1)
        assert np.all(err <= 1e-4 * nrm + 1e-30) or n_div > 0
    dz.free()


@pytest.mark.parametrize("leaf_max", [1, 8])
def test_beams_with_other_leaf_sizes(ctx, leaf_max):
    """Single-triangle leaves fill the beam's leaf lists (a tile-level frontier of 32 nodes can add 64 leaves at
    once -- the list once held 64 and overflowed), 8-triangle leaves its candidate list: same photons either way."""
    th = W.draw_params(W.FAMILY_DETAILED, 1)
    ctx.srp_set_options(leaf_max=leaf_max)                        # read by srp_build_designs
    try:
        dz = ctx.srp_build_designs(W.FAMILY_DETAILED, th)
    finally:
        ctx.srp_set_options()
    sun = W.fibonacci_sphere(4)
    pairs = np.array([[0, j] for j in range(4)], np.int32)
    res = {}
    for mode in (1, 2):
        ctx.srp_set_options(primary_mode=mode)
        try:
            F, st = run_pairs(ctx, dz, sun, pairs, 1 << 16, 8, seed=0)
            sg = ctx.srp_path_signatures(dz, cuda(sun), pairs, 1 << 16, 8, 0).cpu().numpy().astype(np.uint64)
        finally:
            ctx.srp_set_options()
        res[mode] = (F, st, sg)
    n_div = int((res[1][2] != res[2][2]).sum())
    assert n_div <= 3, n_div
    for key in ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments"):
        assert abs(res[1][1][key] - res[2][1][key]) <= 4 * n_div, key
    dz.free()


def test_beam_auto_mode_and_determinism(ctx):
    """auto: beams when rays_per_dir >= 8 x triangles.  Beam results are bit-reproducible (integer
    accumulation; the pool order does not matter)."""
    verts = W.icosphere(3, 1.3)                                           # 1280 facets
    mats = W.dirichlet_materials(len(verts), 7)
    dz = ctx.srp_build_designs_from_meshes(verts, mats, [0, len(verts)])
    sun = cuda(W.fibonacci_sphere(5))
    a = ctx.srp_forces(dz, sun, 1 << 14, 3, 1).cpu().numpy()
    st = ctx.srp_get_stats()
    assert st["beam_tile_miss"] + st["beam_block_miss"] + st["beam_group_miss"] > 0       # 16384 >= 8 * 1280
    b = ctx.srp_forces(dz, sun, 1 << 14, 3, 1).cpu().numpy()
    assert np.array_equal(a, b)
    ctx.srp_forces(dz, sun, 1 << 12, 3, 1)
    st = ctx.srp_get_stats()
    assert st["beam_tile_miss"] + st["beam_block_miss"] + st["beam_group_miss"] + st["beam_fallback"] == 0
    dz.free()


# ---------------------------------------------------------------- torque (Eq. 4)
@pytest.mark.parametrize("family,D,S,N,B,mode", [
    (W.FAMILY_BOXWING, 3, 6, 1 << 14, 4, 0),        # small_beam_kernel
    (W.FAMILY_BOXWING6, 3, 6, 1 << 12, 4, 1),       # trace_kernel (all triangles, every segment)
    (W.FAMILY_DETAILED, 2, 3, 1 << 12, 8, 1),       # bvh_trace_kernel
    (W.FAMILY_DETAILED, 2, 3, 1 << 12, 8, 2),       # beam_trace_kernel: tile sums + pooled hits
])
def test_torque_matches_oracle(ctx, oracle, family, D, S, N, B, mode):
    """srp_forces_torques against the oracle's Eq. 4 on the same photons, off-origin centres of mass;
    the forces it returns are those of srp_forces."""
    th = W.draw_params(family, D)
    sun = W.fibonacci_sphere(S)
    x_com = np.array([[0.3, -0.2, 0.5], [-0.4, 0.1, 0.0], [0.0, 0.6, -0.7]], np.float32)[:D]
    dz = ctx.srp_build_designs(family, th)
    ctx.srp_set_options(primary_mode=mode)
    try:
        F, T = ctx.srp_forces_torques(dz, cuda(sun), N, B, seed=9, x_com=x_com)
        F0 = ctx.srp_forces(dz, cuda(sun), N, B, 9).cpu().numpy()
        pairs = np.array([[D - 1, 1], [0, S - 1]], np.int32)
        Fp, Tp = ctx.srp_forces_torques_pairs(dz, cuda(sun), pairs, N, B, seed=9, x_com=x_com)
    finally:
        ctx.srp_set_options()
    F, T = F.cpu().numpy(), T.cpu().numpy()
    assert rel_l2(F.reshape(-1, 3), F0.reshape(-1, 3)).max() < 1e-6
    assert np.array_equal(Tp.cpu().numpy(), T[pairs[:, 0], pairs[:, 1]])
    assert np.array_equal(Fp.cpu().numpy(), F[pairs[:, 0], pairs[:, 1]])
    for k in range(D):
        v, m = oracle.build_mesh(family, th[k], k=k)
        r = oracle.forces(v, m, sun, N, B, seed=9, k=k, x_com=x_com[k])
        assert_parity(F[k], r["F"], r["sigma"], tol_agg=3e-3)
        # same acceptance for the torque vectors, with their own standard error
        assert_parity(T[k], r["T"], r["sigma_T"], tol_agg=3e-3)
    dz.free()


def test_torque_closed_forms_on_gpu(ctx):
    """Off-centre plate: tau = (centroid - x_COM) x F; two-plate windmill: sign and lever arms; NULL x_com = origin."""
    p0 = np.array([1.5, -1.75, 0.5]); eu = np.array([1.0, 0, 0]); ev = np.array([0, 1.5, 0.3])
    verts = quad(p0, eu, ev)
    centroid = p0 + 0.5 * eu + 0.5 * ev
    normal = np.cross(eu, ev); area = np.linalg.norm(normal); normal /= area
    dz = ctx.srp_build_designs_from_meshes(verts, const_mats(2, 0.3, 0.5, 0.2), [0, 2])
    om = np.array([[0.3, 0.2, 0.8], [-0.5, 0.1, 0.6]], np.float32)
    xc = np.array([[0.2, 0.1, -0.4]], np.float32)
    F, T = ctx.srp_forces_torques(dz, cuda(om), 1 << 16, 1, seed=3, x_com=xc)
    F0, T0 = ctx.srp_forces_torques(dz, cuda(om), 1 << 16, 1, seed=3)
    F, T, T0 = F.cpu().numpy()[0], T.cpu().numpy()[0], T0.cpu().numpy()[0]
    for j in range(2):
        Fc = flat_plate_force(om[j], normal, area, 0.3, 0.5, 0.2)
        assert np.linalg.norm(T[j] - np.cross(centroid - xc[0], Fc)) < 5e-3 * np.linalg.norm(np.cross(centroid - xc[0], Fc))
        assert np.linalg.norm(T0[j] - np.cross(centroid, Fc)) < 5e-3 * np.linalg.norm(np.cross(centroid, Fc))
        np.testing.assert_allclose(T[j], T0[j] - np.cross(xc[0], F[j]), rtol=0, atol=2e-6 * np.linalg.norm(T0[j]))
    dz.free()
    black = quad([1.5, -0.5, 0.0], [1, 0, 0], [0, 1, 0])
    mirror = quad([-2.5, -0.5, 0.0], [1, 0, 0], [0, 1, 0])
    dz = ctx.srp_build_designs_from_meshes(np.concatenate([black, mirror]),
                                           np.concatenate([const_mats(2, 1, 0, 0), const_mats(2, 0, 1, 0)]), [0, 4])
    F, T = ctx.srp_forces_torques(dz, cuda(np.array([[0, 0, 1]], np.float32)), 1 << 16, 2, seed=1)
    T = T.cpu().numpy()[0, 0]
    assert np.linalg.norm(T - np.array([0, -2 * P0, 0])) < 5e-3 * 2 * P0
    dz.free()


# ---------------------------------------------------------------- thermal emitters (R22)
@pytest.mark.parametrize("family,D,N,B,deposit", [(W.FAMILY_BOXWING, 3, 1 << 12, 4, 0), (W.FAMILY_BOXWING6, 2, 1 << 12, 4, 1),
                                                  (W.FAMILY_DETAILED, 1, 1 << 9, 8, 0)])
def test_thermal_forces_match_oracle(ctx, oracle, family, D, N, B, deposit):
    """srp_thermal_forces against the oracle's emitters on the same Philox streams: a few facets per design radiate
    (both signs), brute-force and BVH designs, expected-value and analog deposits; counters agree."""
    th = W.draw_params(family, D)
    T = W.TRI_COUNT[family]
    rng = np.random.default_rng(3)
    power = np.zeros((D, T), np.float32)
    for k in range(D):
        idx = rng.choice(T, size=min(6, T), replace=False)
        power[k, idx] = rng.uniform(100.0, 700.0, len(idx)) * rng.choice([-1.0, 1.0], len(idx))
    dz = ctx.srp_build_designs(family, th)
    ctx.srp_set_options(deposit=deposit)
    try:
        F = ctx.srp_thermal_forces(dz, power.reshape(-1), N, B, seed=6).cpu().numpy()
        st = ctx.srp_get_stats()
    finally:
        ctx.srp_set_options()
    tot = None
    for k in range(D):
        v, m = oracle.build_mesh(family, th[k], k=k)
        r = oracle.thermal(v, m, power[k], N, B, seed=6, k=k, deposit=deposit)
        err = np.linalg.norm(F[k] - r["F"])
        assert err <= 1e-4 * np.linalg.norm(r["F"]) or err <= 4 * r["sigma"], (k, err, r["sigma"])
        assert err <= 3e-3 * np.linalg.norm(r["F"])
        tot = r["stats"] if tot is None else {a: ([x + y for x, y in zip(tot[a], b)] if isinstance(b, list) else tot[a] + b)
                                               for a, b in r["stats"].items()}
    assert st["launched"] == tot["launched"] == N * int((power != 0).sum())
    for key in ("primary_miss", "absorbed", "escaped", "capped", "segments"):
        assert abs(st[key] - tot[key]) <= 8, (key, st[key], tot[key])
    assert st["launched"] == st["primary_miss"] + st["absorbed"] + st["escaped"] + st["capped"]
    dz.free()


def test_thermal_closed_forms_on_gpu(ctx):
    """Isolated emitter: F = -(2/3) (W/c) n; emitter in a closed black cavity: no net force."""
    c = 299792458.0
    verts = quad([0, 0, 0], [1, 0, 0], [0, 0.5, 0.5])
    n = unit(np.cross([1, 0, 0], [0, 0.5, 0.5]))
    dz = ctx.srp_build_designs_from_meshes(verts, const_mats(2, 0.2, 0.5, 0.3), [0, 2])
    F = ctx.srp_thermal_forces(dz, [35000.0, 35000.0], 1 << 14, 3).cpu().numpy()[0]
    np.testing.assert_allclose(F, -(2.0 / 3.0) * 70000.0 / c * n, rtol=2e-6)
    F = ctx.srp_thermal_forces(dz, [0.0, -35000.0], 1 << 14, 3).cpu().numpy()[0]
    np.testing.assert_allclose(F, +(2.0 / 3.0) * 35000.0 / c * n, rtol=2e-6)
    assert ctx.srp_get_stats()["launched"] == 1 << 14
    F = ctx.srp_thermal_forces(dz, [0.0, 0.0], 1 << 10, 3).cpu().numpy()[0]
    assert np.all(F == 0) and ctx.srp_get_stats()["launched"] == 0
    dz.free()
    from test_oracle_thermal import box
    room = box([-1, -1, -1], [1, 1, 1], inward=True)
    emitter = quad([-0.2, -0.2, -0.3], [0.4, 0, 0], [0, 0.4, 0.1])
    verts = np.concatenate([room, emitter])
    power = np.zeros(len(verts), np.float32); power[-2:] = 500.0
    dz = ctx.srp_build_designs_from_meshes(verts, const_mats(len(verts), 1.0, 0.0, 0.0), [0, len(verts)])
    ctx.srp_set_options(deposit=1)
    try:
        F = ctx.srp_thermal_forces(dz, power, 1 << 14, 4).cpu().numpy()[0]
        st = ctx.srp_get_stats()
    finally:
        ctx.srp_set_options()
    assert st["absorbed"] == st["launched"] == 2 << 14
    assert np.linalg.norm(F) < 1e-5 * 1000.0 / c            # per-lane fp32 sums of +-d cancel to rounding
    dz.free()


# ---------------------------------------------------------------- full sizes, in bench.py's launch configuration
def test_cfg2_full_size_sampled_against_oracle(ctx, oracle):
    """The whole 256 x 1024 x 2^18 job in one srp_forces call (as bench.py launches it); 24 sampled
    outputs are recomputed by the oracle; the counters must balance over all 6.9e10 photons."""
    cfg = W.CONFIGS["cfg2_boxwing"]
    th, sun = cfg.params(), cfg.sun_dirs()
    dz = ctx.srp_build_designs(cfg.family, th)
    F = ctx.srp_forces(dz, cuda(sun), cfg.N, cfg.B, cfg.seed).cpu().numpy()
    st = ctx.srp_get_stats()
    assert st["launched"] == cfg.primaries
    assert st["launched"] == st["primary_miss"] + st["absorbed"] + st["escaped"] + st["capped"]
    assert st["segments"] == sum(st["hits_at_depth"]) + st["primary_miss"] + st["escaped"]
    assert np.isfinite(F).all()
    rng = np.random.default_rng(8)
    pairs = np.stack([rng.integers(0, cfg.D, 24), rng.integers(0, cfg.S, 24)], 1)
    meshes = {int(k): oracle.build_mesh(cfg.family, th[k], k=int(k)) for k in np.unique(pairs[:, 0])}
    Fo, sig, _ = oracle_pairs(oracle, meshes, pairs, sun, cfg.N, cfg.B, seed=cfg.seed)
    assert_parity(F[pairs[:, 0], pairs[:, 1]], Fo, sig)
    dz.free()


def test_cfg3_full_N_consistent_with_reduced_N_oracle(ctx, oracle):
    """Full N = 2^20 on 2 designs x 64 directions (same kernel and tile configuration as the full job);
    the oracle cannot finish 2^20 x 50k triangle tests per pair in seconds, so it is run at N = 2^12
    and the two estimates of the same force must agree within 4 sigma of the smaller sample."""
    cfg = W.CONFIGS["cfg3_detailed"]
    th, sun = cfg.params()[:2], cfg.sun_dirs()[::64]
    dz = ctx.srp_build_designs(cfg.family, th)
    F = ctx.srp_forces(dz, cuda(sun), cfg.N, cfg.B, cfg.seed).cpu().numpy()
    st = ctx.srp_get_stats()
    assert st["launched"] == 2 * len(sun) * cfg.N
    assert st["launched"] == st["primary_miss"] + st["absorbed"] + st["escaped"] + st["capped"]
    pairs = np.array([[0, 3], [1, 17], [0, 40], [1, 63]], np.int32)
    meshes = {k: oracle.build_mesh(cfg.family, th[k], k=k) for k in range(2)}
    Fo, sig, _ = oracle_pairs(oracle, meshes, pairs, sun, 1 << 12, cfg.B, seed=cfg.seed, sampler=1)
    err = np.linalg.norm(F[pairs[:, 0], pairs[:, 1]] - Fo, axis=1)
    assert np.all(err <= 4 * sig)
    # the full job also runs with the escape masks (its photons-per-triangle count is above the rule; this slice is
    # below it, so they are forced here): same photons, same counters, forces equal to fp32 rounding
    ctx.srp_set_options(escape_masks=2)
    try:
        Fm = ctx.srp_forces(dz, cuda(sun), cfg.N, cfg.B, cfg.seed).cpu().numpy()
        sm = ctx.srp_get_stats()
    finally:
        ctx.srp_set_options()
    for key in ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments", "hits_at_depth"):
        assert sm[key] == st[key], key
    assert sm["mask_escapes"] > 0.5 * sm["escaped"] and st["mask_escapes"] == 0
    assert np.abs(Fm - F).max() <= 2e-6 * np.abs(F).max()
    dz.free()


def test_cfg4_full_size_sampled_against_oracle(ctx, oracle):
    """The whole 4096 x 256 x 2^16 sweep in one srp_forces call (as bench.py launches it); 32 sampled
    outputs are recomputed by the oracle; the counters balance over all 6.9e10 photons."""
    cfg = W.CONFIGS["cfg4_sweep"]
    th, sun = cfg.params(), cfg.sun_dirs()
    dz = ctx.srp_build_designs(cfg.family, th)
    F = ctx.srp_forces(dz, cuda(sun), cfg.N, cfg.B, cfg.seed).cpu().numpy()
    st = ctx.srp_get_stats()
    assert st["launched"] == cfg.primaries
    assert st["launched"] == st["primary_miss"] + st["absorbed"] + st["escaped"] + st["capped"]
    assert st["segments"] == sum(st["hits_at_depth"]) + st["primary_miss"] + st["escaped"]
    assert np.isfinite(F).all()
    rng = np.random.default_rng(9)
    pairs = np.stack([rng.integers(0, cfg.D, 32), rng.integers(0, cfg.S, 32)], 1)
    meshes = {int(k): oracle.build_mesh(cfg.family, th[k], k=int(k)) for k in np.unique(pairs[:, 0])}
    Fo, sig, _ = oracle_pairs(oracle, meshes, pairs, sun, cfg.N, cfg.B, seed=cfg.seed)
    assert_parity(F[pairs[:, 0], pairs[:, 1]], Fo, sig)
    dz.free()


def test_cfg5_full_N_properties_and_reduced_N_oracle(ctx, oracle):
    """Full N = 2^20 on the 1M-triangle sail for 16 directions (bench.py's kernel and tile configuration).  The
    oracle cannot test 2^20 x 1e6 triangle pairs, so: photon bookkeeping balances exactly; the force is within 4 sigma
    of the oracle's N = 2^9 estimate on two directions; and near-normal incidence approaches the flat-sail closed
    form (5 cm wrinkles on 40 m change |F| by < 1 %)."""
    cfg = W.CONFIGS["cfg5_sail"]
    th = cfg.params()
    sun = np.concatenate([cfg.sun_dirs()[::293][:14], np.array([[0.02, 0.01, 1.0], [0.3, -0.2, 0.9]], np.float32)])
    dz = ctx.srp_build_designs(cfg.family, th)
    F = ctx.srp_forces(dz, cuda(sun), cfg.N, cfg.B, cfg.seed).cpu().numpy()[0]
    st = ctx.srp_get_stats()
    assert st["launched"] == len(sun) * cfg.N
    assert st["launched"] == st["primary_miss"] + st["absorbed"] + st["escaped"] + st["capped"]
    assert st["segments"] == sum(st["hits_at_depth"]) + st["primary_miss"] + st["escaped"]
    Fc = flat_plate_force(sun[14], [0, 0, 1], 1600.0, 0.08, 0.88, 0.04)
    assert np.linalg.norm(F[14] - Fc) < 1e-2 * np.linalg.norm(Fc)
    meshes = {0: oracle.build_mesh(cfg.family, th[0], k=0)}
    pairs = np.array([[0, 14], [0, 15]], np.int32)
    Fo, sig, _ = oracle_pairs(oracle, meshes, pairs, sun, 1 << 9, cfg.B, seed=cfg.seed, sampler=1)
    err = np.linalg.norm(F[pairs[:, 1]] - Fo, axis=1)
    assert np.all(err <= 4 * sig), (err, sig)
    dz.free()


def _same_stream_parity(ctx, oracle, cfg, dz, th, sun, pairs, N, max_div_fraction, label, **opts):
    """GPU forces (plain kernels, the launch configuration srp_forces picks for this N) against the oracle on the
    same Philox streams, photon paths compared through the path signatures; north_star's tolerances (1e-4 per vector
    where no photon diverged, else 4 sigma, 1e-3 aggregate).  Also: the instrumented build, which the signatures come
    from, gives the plain build's forces bit for bit, so the divergence count describes the forces that are checked."""
    import time
    ctx.srp_set_options(**opts)
    try:
        F, st = run_pairs(ctx, dz, sun, pairs, N, cfg.B, cfg.seed)
        psig = ctx.srp_path_signatures(dz, cuda(sun), pairs, N, cfg.B, cfg.seed).cpu().numpy().astype(np.uint64)
        ctx.srp_set_options(instrumented=1, **opts)
        Fi, sti = run_pairs(ctx, dz, sun, pairs, N, cfg.B, cfg.seed)
    finally:
        ctx.srp_set_options()
    assert np.array_equal(F, Fi)
    for key in ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments", "hits_at_depth"):
        assert st[key] == sti[key], key
    meshes = {int(k): oracle.build_mesh(cfg.family, th[k], k=int(k)) for k in np.unique(pairs[:, 0])}
    t0 = time.time()
    Fo, sig, ost, osig = oracle_pairs(oracle, meshes, pairs, sun, N, cfg.B, seed=cfg.seed, want_path_sig=True)
    n_div = (psig != osig).sum(axis=1)
    print("%s: %d pairs x N = %d, oracle %.0f s, divergent photons per pair %s" % (label, len(pairs), N, time.time() - t0, n_div.tolist()))
    assert n_div.sum() <= max_div_fraction * len(pairs) * N
    bad = assert_parity(F, Fo, sig, diverged=n_div > 0)              # tol_vec 1e-4, tol_agg 1e-3: BASELINE.json
    counters_close(st, ost, tol=4 * int(n_div.sum()) + 8)
    return bad, n_div


@pytest.mark.slow
def test_cfg3_full_N_same_stream_parity(ctx, oracle):
    """full N = 2^20, B = 8, one (design, direction) pair per host core (at most 16, the
    designs of the batch), oracle brute force over all 49 840 triangles on the same streams (~4 min per pair and core).
    The beam kernel and the bounce kernel run in the tile configuration of the full job, escape masks on."""
    import os
    cfg = W.CONFIGS["cfg3_detailed"]
    th, sun = cfg.params(), cfg.sun_dirs()
    n = max(4, min(16, os.cpu_count() or 4))
    rng = np.random.default_rng(11)
    pairs = np.stack([np.arange(n) % cfg.D, rng.integers(0, cfg.S, n)], 1).astype(np.int32)
    dz = ctx.srp_build_designs(cfg.family, th)
    _same_stream_parity(ctx, oracle, cfg, dz, th, sun, pairs, cfg.N, 2e-4, "cfg3 full N", escape_masks=2)
    st = ctx.srp_get_stats()
    assert st["beam_tile_miss"] > 0 and st["loop_rounds"] >= 1        # beams + ray queue were in play
    dz.free()


@pytest.mark.slow
def test_cfg5_sail_N14_same_stream_parity(ctx, oracle):
    """N = 2^14 on 8 directions (two grazing, two oblique, near-normal from both sides, two of
    the workload's Fibonacci directions), B = 8, oracle brute force over all 1 019 698 triangles (~4 min per
    direction and core)."""
    cfg = W.CONFIGS["cfg5_sail"]
    th = cfg.params()
    sun = np.concatenate([np.array([[1, 0.2, 0.02], [0.3, -1, -0.03], [0.5, 0.4, 0.7], [-0.2, 0.6, -0.6],
                                    [0.05, 0.02, 1], [0.01, -0.03, -1]], np.float32), cfg.sun_dirs()[[517, 3011]]])
    pairs = np.stack([np.zeros(len(sun)), np.arange(len(sun))], 1).astype(np.int32)
    dz = ctx.srp_build_designs(cfg.family, th)
    _same_stream_parity(ctx, oracle, cfg, dz, th, sun, pairs, 1 << 14, 2e-4, "cfg5 N = 2^14")
    dz.free()


# ---------------------------------------------------------------- per-sample designs (NEXT-3)
@pytest.mark.parametrize("family,M,N,B,sampler,deposit", [
    (W.FAMILY_BOXWING, 40, 1 << 10, 4, 0, 0),        # 16 triangles per record, each over hundreds of grid cells (rasterised by a warp)
    (W.FAMILY_BOXWING_T, 24, 1 << 10, 4, 0, 0),      # 1280 triangles: the paper's "1 k faces" (rasterised by a thread each)
    (W.FAMILY_BOXWING_T, 6, 1 << 11, 4, 0, 0),       # a 64 x 32 grid
    (W.FAMILY_BOXWING_T, 4, 1 << 12, 3, 0, 0),       # 64 KB of grid beside the triangles: one block per SM
    (W.FAMILY_BOXWING_T, 2, 1 << 13, 2, 0, 0),       # a grid that does not fit: every primary against every triangle
    (W.FAMILY_PLATE, 16, 1 << 7, 2, 0, 0),           # 2 triangles, 16 x 8 cells
    (W.FAMILY_BOXWING_T, 8, 1000, 3, 1, 1),          # i.i.d. sampler (N need not be a power of two), analog deposit
])
def test_per_sample_designs_match_oracle(ctx, oracle, family, M, N, B, sampler, deposit):
    """srp_forces_per_sample: every record its own design AND its own direction, brute force over all triangles.
    Record m against the oracle's forward tracer on design m (k = m in the Philox counters, direction index 0)."""
    import torch
    th = W.draw_params(family, M)
    sun = W.random_directions(M)
    ctx.srp_set_options(sampler=sampler, deposit=deposit)
    try:
        F = ctx.srp_forces_per_sample(family, cuda(th), cuda(sun), N, B, seed=5).cpu().numpy()
        st = ctx.srp_get_stats()
    finally:
        ctx.srp_set_options()
    assert st["launched"] == M * N
    assert st["launched"] == st["primary_miss"] + st["absorbed"] + st["escaped"] + st["capped"]
    Fo, sig, tot = [], [], None
    for m in range(M):
        v, mt = oracle.build_mesh(family, th[m], k=m)
        r = oracle.forces(v, mt, sun[m:m + 1], N, B, seed=5, k=m, j0=0, sampler=sampler, deposit=deposit)
        Fo.append(r["F"][0]); sig.append(r["sigma"][0])
        tot = r["stats"] if tot is None else {a: ([x + y for x, y in zip(tot[a], b)] if isinstance(b, list) else tot[a] + b)
                                             for a, b in r["stats"].items()}
    assert_parity(F, np.array(Fo), np.array(sig), tol_agg=3e-3)      # N = 2^10: one photon is ~1e-3 of a vector (R24)
    counters_close(st, tot, tol=8)
    # the same records through the designs + pairs interface (direction index m instead of 0: other photons, same forces)
    if family == W.FAMILY_BOXWING and sampler == 0:
        dz = ctx.srp_build_designs(family, th)
        pairs = np.stack([np.arange(M), np.arange(M)], 1).astype(np.int32)
        Fp = ctx.srp_forces_pairs(dz, cuda(sun), pairs, 1 << 16, B, 5).cpu().numpy()
        assert np.all(np.linalg.norm(F - Fp, axis=1) <= 5.0 * np.array(sig) + 1e-3 * np.linalg.norm(Fp, axis=1))
        dz.free()


def test_new_entry_points_reject_bad_arguments(ctx):
    """SRP_ERR_INVALID / SRP_ERR_UNSUPPORTED before any launch: per-sample records, split, workspace."""
    import ctypes
    import torch
    from paper_2602_10712_b200.binding import SrpError
    L, h = ctx.lib, ctx.handle
    th = cuda(W.draw_params(W.FAMILY_BOXWING_T, 4))
    sun = cuda(W.random_directions(4))
    out = torch.empty((4, 3), dtype=torch.float32, device="cuda")
    ok = lambda *a: L.srp_forces_per_sample(h, *a)
    assert ok(W.FAMILY_BOXWING_T, th.data_ptr(), 2, sun.data_ptr(), 4, 1 << 10, 4, 0, 2, out.data_ptr()) == 0
    assert ok(W.FAMILY_BOXWING_T, th.data_ptr(), 3, sun.data_ptr(), 4, 1 << 10, 4, 0, 2, out.data_ptr()) == -1     # n_params
    assert ok(W.FAMILY_BOXWING_T, th.data_ptr(), 2, sun.data_ptr(), 0, 1 << 10, 4, 0, 2, out.data_ptr()) == -1     # M
    assert ok(W.FAMILY_BOXWING_T, th.data_ptr(), 2, sun.data_ptr(), 4, 1000, 4, 0, 2, out.data_ptr()) == -1        # stratified: 2^m
    assert ok(W.FAMILY_BOXWING_T, th.data_ptr(), 2, sun.data_ptr(), 4, 1 << 10, 16, 0, 2, out.data_ptr()) == -1    # B
    assert ok(W.FAMILY_BOXWING_T, None, 2, sun.data_ptr(), 4, 1 << 10, 4, 0, 2, out.data_ptr()) == -1              # null
    assert ok(W.FAMILY_DETAILED, th.data_ptr(), 2, sun.data_ptr(), 4, 1 << 10, 4, 0, 2, out.data_ptr()) == -4      # 49 840 triangles
    assert ok(9, th.data_ptr(), 2, sun.data_ptr(), 4, 1 << 10, 4, 0, 2, out.data_ptr()) == -1                      # family
    torch.cuda.synchronize()
    dz = ctx.srp_build_designs(W.FAMILY_BOXWING, W.draw_params(W.FAMILY_BOXWING, 2))
    assert L.srp_forces_split(h, dz.handle, sun.data_ptr(), 4, 1 << 10, 2, 0, out.data_ptr(), None) == -1
    assert L.srp_forces_split_pairs(h, dz.handle, sun.data_ptr(), 4, None, 2, 1 << 10, 2, 0, out.data_ptr(), out.data_ptr()) == -1
    buf = torch.empty(ctx.srp_workspace_bytes_min() + 4096, dtype=torch.uint8, device="cuda")
    assert L.srp_set_workspace(h, ctypes.c_void_p(buf.data_ptr() + 8), buf.numel() - 8) == -1                     # alignment
    assert L.srp_set_workspace(h, None, 4096) == -1 and L.srp_set_workspace(h, ctypes.c_void_p(buf.data_ptr()), 0) == -1
    assert L.srp_set_workspace(h, None, 0) == 0
    assert L.srp_launch_count(h, None) == -1
    with pytest.raises(ValueError):
        ctx.srp_forces_pairs(dz, sun, np.array([[0, 0], [2, 1]], np.int32), 1 << 10, 2)                           # design 2 of 2
    with pytest.raises(ValueError):
        ctx.srp_forces(dz, sun.cpu(), 1 << 10, 2)                                                                  # a CPU tensor is no device pointer
    with pytest.raises(ValueError):
        ctx.srp_build_designs_from_meshes(W.icosphere(0), np.full((20, 3), 0.5, np.float32), [0, 20])              # materials sum to 1.5
    # a pair list the binding did not see: out-of-range entries are clamped on the device, nothing is read out of bounds
    bad = torch.tensor([[7, 9], [-3, 0]], dtype=torch.int32, device="cuda")
    assert L.srp_forces_pairs(h, dz.handle, sun.data_ptr(), 4, bad.data_ptr(), 2, 1 << 10, 2, 0, out.data_ptr()) == 0
    torch.cuda.synchronize()
    assert torch.isfinite(out[:2]).all()
    # a zero sun direction gives a zero force, not NaN
    z = cuda(np.array([[0, 0, 0], [0, 0, 1]], np.float32))
    F = ctx.srp_forces(dz, z, 1 << 10, 2).cpu().numpy()
    assert np.all(F[:, 0] == 0.0) and np.all(np.isfinite(F)) and np.linalg.norm(F[0, 1]) > 0
    dz.free()


def test_large_accumulations_do_not_wrap(ctx):
    """The fixed-point scale is chosen per call (R21): a mirror plate deposits 2 per photon, which wrapped the 2^-32
    accumulators at N = 2^30 photons per direction.  And torque arms are summed in units of the design's extent, so a
    mesh given in millimetres gives 1e6 times the force and 1e9 times the torque of the same mesh in metres (area x arm)
    instead of wrapping (arms of ~1e3 mesh units times 2^20 photons used to exceed the accumulators' range)."""
    plate = quad([-0.5, -0.5, 0.0], [1, 0, 0], [0, 1, 0])
    dz = ctx.srp_build_designs_from_meshes(plate, const_mats(2, 0.0, 1.0, 0.0), [0, 2])
    sun = cuda(np.array([[0, 0, 1]], np.float32))
    F = ctx.srp_forces(dz, sun, 1 << 30, 1, 0).cpu().numpy()[0, 0]
    np.testing.assert_allclose(F, [0, 0, -2 * P0], rtol=1e-5, atol=1e-12)
    dz.free()
    # the same off-centre plate in metres and in millimetres: torque scales with length^3 (area x arm)
    res = []
    for s in (1.0, 1000.0):
        v = quad([1.5 * s, -1.75 * s, 0.5 * s], [1.0 * s, 0, 0], [0, 1.5 * s, 0.3 * s])
        d = ctx.srp_build_designs_from_meshes(v, const_mats(2, 0.3, 0.5, 0.2), [0, 2])
        Fm, Tm = ctx.srp_forces_torques(d, cuda(np.array([[0.3, 0.2, 0.8]], np.float32)), 1 << 20, 1, seed=3)
        res.append((Fm.cpu().numpy()[0, 0], Tm.cpu().numpy()[0, 0]))
        d.free()
    assert np.allclose(res[1][0], res[0][0] * 1e6, rtol=2e-4)
    assert np.allclose(res[1][1], res[0][1] * 1e9, rtol=2e-4)


def test_force_maps_direct_and_indirect(ctx):
    """PAPER.md:394 force maps from srp_forces_split.  A convex body has no indirect light (its map is the closed
    form of P3, direct = total exactly); the box-wing has some."""
    verts = W.icosphere(2, 1.0)
    mats = W.dirichlet_materials(len(verts), 3)
    dz = ctx.srp_build_designs_from_meshes(verts, mats, [0, len(verts)])
    total, direct = ctx.force_maps(dz, 4, 8, 1 << 14, 3, seed=1)
    sun = W.latlong_directions(4, 8)
    t = total.cpu().numpy().reshape(-1, 3)
    for j in range(len(sun)):
        assert rel_l2(t[j], convex_polyhedron_force(verts, mats, sun[j])) < 5e-3
    assert float((total - direct).abs().max()) <= 1e-3 * float(total.abs().max())
    dz.free()
    dz = ctx.srp_build_designs(W.FAMILY_BOXWING, W.draw_params(W.FAMILY_BOXWING, 2))
    total, direct = ctx.force_maps(dz, 4, 8, 1 << 14, 4, seed=1)
    indirect = total - direct
    assert tuple(total.shape) == (2, 4, 8, 3)
    assert float(indirect.abs().max()) > 1e-3 * float(total.abs().max())
    assert float(indirect.abs().max()) < float(direct.abs().max())
    dz.free()


@pytest.mark.parametrize("family,D,S,N,B,mode,deposit", [
    (W.FAMILY_BOXWING, 3, 6, 1 << 14, 4, 0, 0),        # small_beam_kernel
    (W.FAMILY_BOXWING6, 3, 6, 1 << 12, 4, 1, 1),       # trace_kernel (all triangles, every segment), analog deposit
    (W.FAMILY_DETAILED, 2, 3, 1 << 12, 8, 1, 0),       # bvh_trace_kernel
    (W.FAMILY_DETAILED, 2, 3, 1 << 12, 8, 2, 0),       # beam_trace_kernel (all direct) + bounce_trace_kernel
])
def test_direct_indirect_split_matches_oracle(ctx, oracle, family, D, S, N, B, mode, deposit):
    """srp_forces_split against the oracle's split on the same photons: the total is srp_forces' (same photons),
    the direct part is the B = 0 force bit for bit, and both parts match the oracle."""
    th = W.draw_params(family, D)
    sun = W.fibonacci_sphere(S)
    dz = ctx.srp_build_designs(family, th)
    ctx.srp_set_options(primary_mode=mode, deposit=deposit)
    try:
        F, Fd = ctx.srp_forces_split(dz, cuda(sun), N, B, seed=4)
        F0 = ctx.srp_forces(dz, cuda(sun), N, B, 4).cpu().numpy()
        Fnb = ctx.srp_forces(dz, cuda(sun), N, 0, 4).cpu().numpy()
        pairs = np.array([[D - 1, 1], [0, S - 1]], np.int32)
        Fp, Fdp = ctx.srp_forces_split_pairs(dz, cuda(sun), pairs, N, B, seed=4)
    finally:
        ctx.srp_set_options()
    F, Fd = F.cpu().numpy(), Fd.cpu().numpy()
    assert rel_l2(F.reshape(-1, 3), F0.reshape(-1, 3)).max() < 1e-6
    # direct == "NB": bit for bit where a photon's lane is fixed by its index; trace_kernel hands rays
    # to lanes as they fall free, so its per-lane fp32 partial sums group differently
    if family == W.FAMILY_BOXWING6:
        assert rel_l2(Fd.reshape(-1, 3), Fnb.reshape(-1, 3)).max() < 2e-6
    else:
        assert np.array_equal(Fd, Fnb)
    assert np.array_equal(Fp.cpu().numpy(), F[pairs[:, 0], pairs[:, 1]])
    assert np.array_equal(Fdp.cpu().numpy(), Fd[pairs[:, 0], pairs[:, 1]])
    some_indirect = False
    for k in range(D):
        v, m = oracle.build_mesh(family, th[k], k=k)
        r = oracle.forces_split(v, m, sun, N, B, seed=4, k=k, deposit=deposit)
        sig = oracle.forces(v, m, sun, N, B, seed=4, k=k, deposit=deposit)["sigma"]
        assert_parity(F[k], r["F"], sig, tol_agg=3e-3)
        assert_parity(Fd[k], r["F_direct"], sig, tol_agg=3e-3)
        ind_o, ind_g = r["F_indirect"], F[k].astype(float) - Fd[k].astype(float)
        # the indirect part is a small difference of two large sums: compare it on the scale of the total
        assert np.all(np.linalg.norm(ind_g - ind_o, axis=1) <= 4.0 * sig + 1e-4 * np.linalg.norm(r["F"], axis=1))
        some_indirect |= bool(np.any(np.linalg.norm(ind_o, axis=1) > 1e-3 * np.linalg.norm(r["F"], axis=1)))
    assert some_indirect
    dz.free()


def test_workspace_from_the_caller_and_launch_count(ctx):
    """srp_set_workspace: the ray queue of the beam / bounce loop lives in a torch tensor; a small one means more
    rounds of the loop and the same forces bit for bit; one below srp_workspace_bytes_min is refused.
    srp_launch_count / srp_stats.kernel_launches count this library's kernels."""
    import torch
    from paper_2602_10712_b200.binding import SrpError
    th = W.draw_params(W.FAMILY_DETAILED, 1)
    sun = cuda(W.fibonacci_sphere(8))
    dz = ctx.srp_build_designs(W.FAMILY_DETAILED, th)
    ctx.srp_set_options(primary_mode=2)
    try:
        n0 = ctx.srp_launch_count()
        F0 = ctx.srp_forces(dz, sun, 1 << 18, 8, 2).cpu().numpy()
        st0 = ctx.srp_get_stats()
        n1 = ctx.srp_launch_count()
        assert st0["loop_rounds"] >= 1 and st0["queued_rays"] > 0
        assert st0["kernel_launches"] == n1 - n0 >= 3 + 3 * st0["loop_rounds"] - 1
        need = ctx.srp_workspace_bytes_min()
        with pytest.raises(SrpError):
            ctx.srp_set_workspace(torch.empty(need // 2, dtype=torch.uint8, device="cuda"))
        ws = torch.empty(need + (1 << 16), dtype=torch.uint8, device="cuda")
        ctx.srp_set_workspace(ws)
        F1 = ctx.srp_forces(dz, sun, 1 << 18, 8, 2).cpu().numpy()
        st1 = ctx.srp_get_stats()
        assert np.array_equal(F0, F1)
        # queued_rays counts slots (a few stay unfilled per beam warp and round), so it moves a little with the layout
        assert st1["loop_rounds"] >= 1 and abs(st1["queued_rays"] - st0["queued_rays"]) <= 0.2 * st0["queued_rays"]
        ctx.srp_set_options(primary_mode=2, plain_launches=1)
        F2 = ctx.srp_forces(dz, sun, 1 << 18, 8, 2).cpu().numpy()
        assert np.array_equal(F0, F2)
    finally:
        ctx.srp_set_workspace(None)
        ctx.srp_set_options()
    dz.free()


# ---------------------------------------------------------------- escape masks (escape_mask.cu)
def _mask_meshes():
    """Meshes that stress the mask build: a sphere (convex: every outward direction escapes), an open-topped room
    with a box in it, entered through the opening (inside, almost nothing escapes), two facing finely tessellated
    plates (coplanar neighbours by the thousand, everything opposite within a narrow cone), a random triangle soup
    (no structure at all)."""
    from test_oracle_thermal import box
    rng = np.random.default_rng(11)

    def tess(o, u, v, n):                                   # n x n quads, normal u x v
        o, u, v = (np.asarray(x, float) for x in (o, u, v))
        return np.concatenate([quad(o + u * i / n + v * j / n, u / n, v / n) for i in range(n) for j in range(n)])

    sphere = W.icosphere(3, 1.0)
    walls = [tess([-2, -2, -2], [0, 4, 0], [0, 0, 4], 6), tess([2, -2, -2], [0, 0, 4], [0, 4, 0], 6),     # normals inward
             tess([-2, -2, -2], [0, 0, 4], [4, 0, 0], 6), tess([-2, 2, -2], [4, 0, 0], [0, 0, 4], 6),
             tess([-2, -2, -2], [4, 0, 0], [0, 4, 0], 6)]
    room = np.concatenate(walls + [box([-0.5, -0.4, -1.3], [0.4, 0.5, 0.6])])
    plates = np.concatenate([tess([-1, -1, 0], [2, 0, 0], [0, 2, 0], 24), tess([-1, -1, 0.7], [0, 2, 0], [2, 0, 0], 24)])
    c = rng.uniform(-1, 1, (1500, 1, 3))
    soup = (c + rng.normal(0, 0.15, (1500, 3, 3))).astype(np.float32)
    return {"sphere": sphere, "room": room.astype(np.float32), "plates": plates.astype(np.float32), "soup": soup}


@pytest.mark.parametrize("name", ["sphere", "room", "plates", "soup", "detailed", "sail", "boxwing", "boxwing6", "plate"])
def test_escape_masks_change_no_photon(ctx, name):
    """The masks only say "no triangle lies this way": with them forced on, every photon follows the same path
    (identical signatures) and all photon counters agree; the forces agree to fp32 rounding (a lane that skips a
    traversal takes its next ray earlier, so the per-lane fp32 partial sums group the same deposits differently);
    only the share of escaped rays that never walked the BVH (mask_escapes) differs."""
    rng = np.random.default_rng(3)
    if name == "detailed":
        dz = ctx.srp_build_designs(W.FAMILY_DETAILED, W.draw_params(W.FAMILY_DETAILED, 3))
        D = 3
    elif name == "sail":
        dz = ctx.srp_build_designs(W.FAMILY_SAIL, np.array([[0.8]], np.float32))
        D = 1
    elif name in ("boxwing", "boxwing6", "plate"):              # no hierarchy: masks from all pairs of triangles
        fam = {"boxwing": W.FAMILY_BOXWING, "boxwing6": W.FAMILY_BOXWING6, "plate": W.FAMILY_PLATE}[name]
        D = 1 if name == "plate" else 5
        dz = ctx.srp_build_designs(fam, W.draw_params(fam, D))
    else:
        verts = _mask_meshes()[name]
        mats = np.tile(np.array([[0.2, 0.5, 0.3]], np.float32), (len(verts), 1))
        dz = ctx.srp_build_designs_from_meshes(verts, mats, [0, len(verts)])
        D = 1
    sun = W.fibonacci_sphere(7)
    pairs = np.array([[k, j] for k in range(D) for j in range(7)], np.int32)
    N, B = 1 << 13, 6
    res = {}
    for mode in (1, 2):
        for masks in (0, 2):
            ctx.srp_set_options(primary_mode=mode, escape_masks=masks)
            try:
                F, st = run_pairs(ctx, dz, sun, pairs, N, B, seed=9)
                sg = ctx.srp_path_signatures(dz, cuda(sun), pairs, N, B, 9).cpu().numpy()
            finally:
                ctx.srp_set_options()
            res[mode, masks] = (F, st, sg)
        (F0, s0, g0), (F2, s2, g2) = res[mode, 0], res[mode, 2]
        assert np.array_equal(g0, g2), (name, mode, int((g0 != g2).sum()))
        assert np.abs(F2 - F0).max() <= 2e-6 * np.abs(F0).max(), (name, mode)
        for key in ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments", "hits_at_depth"):
            assert s0[key] == s2[key], (name, mode, key)
        assert s0["mask_escapes"] == 0
        print(name, "mode", mode, "escaped", s2["escaped"], "by mask", s2["mask_escapes"])
        if name == "sphere":
            assert s2["mask_escapes"] == s2["escaped"] > 0          # convex: no bounce ray needs a traversal
        if name == "room":                                          # sun 0 looks into the opening: photons bounce inside
            assert s2["capped"] + s2["absorbed"] > 0 and sum(s2["hits_at_depth"][2:]) > 0
        if name in ("detailed", "plates"):
            assert s2["mask_escapes"] > 0.3 * s2["escaped"]
        if name in ("boxwing", "boxwing6") and mode == 2:            # mode 1 is the brute-force kernel: no masks
            assert s2["mask_escapes"] > 0.5 * s2["escaped"]
        if name == "plate":
            assert s2["mask_escapes"] == s2["escaped"] or mode == 1
    dz.free()


def test_escape_masks_thermal_and_auto_rule(ctx):
    """Thermal emitters use the same masks (emitted rays and their bounces); the default option builds them only
    when the call traces >= 32768 photons per triangle."""
    th = W.draw_params(W.FAMILY_DETAILED, 1)
    rng = np.random.default_rng(4)
    power = np.zeros(W.TRI_COUNT[W.FAMILY_DETAILED], np.float32)
    power[rng.choice(len(power), 64, replace=False)] = 50.0
    out = {}
    for masks in (0, 2):
        dz = ctx.srp_build_designs(W.FAMILY_DETAILED, th)
        ctx.srp_set_options(escape_masks=masks)
        try:
            F = ctx.srp_thermal_forces(dz, power, 1 << 12, 4, seed=2).cpu().numpy()
            out[masks] = (F, ctx.srp_get_stats())
        finally:
            ctx.srp_set_options()
        dz.free()
    assert rel_l2(out[2][0], out[0][0]).max() < 2e-6
    for key in ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments"):
        assert out[0][1][key] == out[2][1][key], key
    assert out[0][1]["mask_escapes"] == 0 < out[2][1]["mask_escapes"]
    # auto: 2 pairs x 2^12 rays on 49 840 triangles is far below the rule, 2^20 rays x 2048 pairs is above it
    sun = W.fibonacci_sphere(2048)
    dz = ctx.srp_build_designs(W.FAMILY_DETAILED, th)
    ctx.srp_forces(dz, cuda(sun[:2]), 1 << 12, 4, 0)
    assert ctx.srp_get_stats()["mask_escapes"] == 0
    pairs = np.stack([np.zeros(2048), np.arange(2048)], 1).astype(np.int32)
    ctx.srp_forces_pairs(dz, cuda(sun), pairs, 1 << 20, 1, 0)
    assert ctx.srp_get_stats()["mask_escapes"] > 0
    ctx.srp_forces(dz, cuda(sun[:2]), 1 << 12, 4, 0)               # once built they stay with the handle
    assert ctx.srp_get_stats()["mask_escapes"] > 0
    dz.free()


@pytest.mark.parametrize("gap", [2e-5, 1e-3])
def test_escape_masks_see_a_plate_hovering_above_the_emitter(ctx, gap):
    """Coplanar pruning must not swallow real geometry: a 2 m plate hovering 20 um (and 1 mm) above another, both
    finely tessellated.  The lower plate radiates upwards; all but the photons leaving through the rim gap
    (<= gap / size of them) are absorbed by the plate above -- with the masks as without."""
    def tess(o, u, v, n):
        o, u, v = (np.asarray(x, float) for x in (o, u, v))
        return np.concatenate([quad(o + u * i / n + v * j / n, u / n, v / n) for i in range(n) for j in range(n)])
    lower = tess([-1, -1, 0], [2, 0, 0], [0, 2, 0], 8)            # normal +z
    upper = tess([-1, -1, gap], [0, 2, 0], [2, 0, 0], 5)          # normal -z
    verts = np.concatenate([lower, upper]).astype(np.float32)
    mats = const_mats(len(verts), 1.0, 0.0, 0.0)
    power = np.zeros(len(verts), np.float32); power[:len(lower)] = 10.0
    res = {}
    for masks in (0, 2):
        dz = ctx.srp_build_designs_from_meshes(verts, mats, [0, len(verts)])
        ctx.srp_set_options(escape_masks=masks)
        try:
            F = ctx.srp_thermal_forces(dz, power, 1 << 10, 2, seed=1).cpu().numpy()
            res[masks] = (F, ctx.srp_get_stats())
        finally:
            ctx.srp_set_options()
        dz.free()
    for key in ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments"):
        assert res[0][1][key] == res[2][1][key], key
    st = res[2][1]
    assert st["launched"] == len(lower) << 10
    assert st["absorbed"] >= (1.0 - 4 * gap) * st["launched"]
    assert np.abs(res[2][0] - res[0][0]).max() <= 2e-6 * np.abs(res[0][0]).max() + 1e-30


# ---------------------------------------------------------------- glossy specular lobes (R23)
def _glossy_cases():
    """(name, verts, mats, offsets, shininess): small designs (no hierarchy), a sphere and the open room (hierarchy,
    many bounces), every facet with its own exponent from {mirror, 0, 3, 40, 800}."""
    rng = np.random.default_rng(21)
    out = {}
    th = W.draw_params(W.FAMILY_BOXWING, 3)
    out["boxwing"] = (W.FAMILY_BOXWING, th)
    room = _mask_meshes()["room"]
    out["room"] = (room, np.tile(np.array([[0.15, 0.7, 0.15]], np.float32), (len(room), 1)))
    sph = W.icosphere(3, 1.0)
    out["sphere"] = (sph, W.dirichlet_materials(len(sph), 2))
    return out, rng


@pytest.mark.parametrize("deposit", [0, 1])
@pytest.mark.parametrize("name,mode", [("boxwing", 0), ("boxwing", 1), ("room", 1), ("room", 2), ("sphere", 2)])
def test_glossy_forces_match_oracle(ctx, oracle, name, mode, deposit):
    cases, rng = _glossy_cases()
    if name == "boxwing":
        family, th = cases[name]
        dz = ctx.srp_build_designs(family, th)
        meshes = {k: oracle.build_mesh(family, th[k], k=k) for k in range(len(th))}
    else:
        verts, mats = cases[name]
        dz = ctx.srp_build_designs_from_meshes(verts, mats, [0, len(verts)])
        meshes = {0: (verts, mats)}
    sumT = int(dz.tri_offsets[-1])
    sh = rng.choice([-1.0, 0.0, 3.0, 40.0, 800.0], sumT).astype(np.float32)
    ctx.srp_designs_set_shininess(dz, sh)
    sun = W.fibonacci_sphere(5)
    pairs = np.array([[k, j] for k in range(dz.D) for j in range(5)], np.int32)
    N, B = 1 << 12, 5
    ctx.srp_set_options(primary_mode=mode, deposit=deposit, escape_masks=2)
    try:
        F, st = run_pairs(ctx, dz, sun, pairs, N, B, seed=8)
        psig = ctx.srp_path_signatures(dz, cuda(sun), pairs, N, B, 8).cpu().numpy().astype(np.uint64)
    finally:
        ctx.srp_set_options()
    Fo = np.zeros((len(pairs), 3)); sig = np.zeros(len(pairs)); n_div = np.zeros(len(pairs), int)
    ost = None
    for q, (k, j) in enumerate(pairs):
        v, m = meshes[int(k)]
        off = int(dz.tri_offsets[k])
        r = oracle.forces(v, m, sun[j:j + 1], N, B, seed=8, k=int(k), j0=int(j), deposit=deposit, want_path_sig=True,
                          shininess=sh[off:off + len(v)])
        Fo[q], sig[q] = r["F"][0], r["sigma"][0]
        n_div[q] = int((psig[q] != r["path_sig"][0]).sum())
        ost = r["stats"] if ost is None else {kk: (vv + r["stats"][kk] if not isinstance(vv, list) else
                                                   [a + b for a, b in zip(vv, r["stats"][kk])]) for kk, vv in ost.items()}
    print(name, "mode", mode, "deposit", deposit, "divergent rays", int(n_div.sum()), "of", N * len(pairs))
    assert n_div.sum() <= 3e-4 * N * len(pairs) + 2
    assert_parity(F, Fo, sig, diverged=n_div > 0, tol_agg=1e-3 if n_div.sum() == 0 else 5e-3)
    counters_close(st, ost, tol=4 * int(n_div.sum()) + 2)
    # removing the shininess restores the mirrors
    ctx.srp_designs_set_shininess(dz, None)
    ctx.srp_set_options(primary_mode=mode, deposit=deposit)
    try:
        F0, _ = run_pairs(ctx, dz, sun, pairs[:3], N, B, seed=8)
    finally:
        ctx.srp_set_options()
    for q, (k, j) in enumerate(pairs[:3]):
        v, m = meshes[int(k)]
        r = oracle.forces(v, m, sun[j:j + 1], N, B, seed=8, k=int(k), j0=int(j), deposit=deposit)
        assert rel_l2(F0[q], r["F"][0]).max() < 1e-3
    dz.free()


def test_glossy_closed_forms_on_gpu(ctx):
    """G1 / G3 through the CUDA path: mean cosine (n+1)/(n+2) at normal incidence, lobe axis at 50 degrees."""
    verts = quad([-0.5, -0.5, 0], [1, 0, 0], [0, 1, 0])
    dz = ctx.srp_build_designs_from_meshes(verts, const_mats(2, 0.0, 1.0, 0.0), [0, 2])
    for ns in (0.0, 10.0):
        ctx.srp_designs_set_shininess(dz, [ns, ns])
        F = ctx.srp_forces(dz, cuda(np.array([[0, 0, 1]], np.float32)), 1 << 18, 1, 0).cpu().numpy()[0, 0]
        Fc = np.array([0, 0, -P0 * (1.0 + (ns + 1.0) / (ns + 2.0))])
        assert np.linalg.norm(F - Fc) < 4e-3 * P0, (ns, F, Fc)
    th = np.radians(50.0)
    om = np.array([np.sin(th) * np.cos(0.7), np.sin(th) * np.sin(0.7), np.cos(th)])
    refl = -om + 2 * np.cos(th) * np.array([0, 0, 1.0])
    ctx.srp_designs_set_shininess(dz, [400.0, 400.0])
    F = ctx.srp_forces(dz, cuda(om[None].astype(np.float32)), 1 << 18, 1, 0).cpu().numpy()[0, 0]
    Fc = P0 * np.cos(th) * (-om - (401.0 / 402.0) * refl)
    assert np.linalg.norm(F - Fc) < 2e-3 * np.linalg.norm(Fc)
    dz.free()


def test_glossy_thermal_matches_oracle(ctx, oracle):
    th = W.draw_params(W.FAMILY_BOXWING6, 2)
    dz = ctx.srp_build_designs(W.FAMILY_BOXWING6, th)
    rng = np.random.default_rng(2)
    sh = rng.choice([-1.0, 1.0, 25.0], 32).astype(np.float32)
    power = np.zeros((2, 16), np.float32); power[:, :12] = 40.0
    ctx.srp_designs_set_shininess(dz, sh)
    N, B = 1 << 12, 4
    F = ctx.srp_thermal_forces(dz, power.reshape(-1), N, B, seed=3).cpu().numpy()
    st = ctx.srp_get_stats()
    tot = 0
    for k in range(2):
        v, m = oracle.build_mesh(W.FAMILY_BOXWING6, th[k], k=k)
        r = oracle.thermal(v, m, power[k], N, B, seed=3, k=k, shininess=sh[16 * k:16 * k + 16])
        assert np.linalg.norm(F[k] - r["F"]) <= 4 * r["sigma"] + 1e-4 * np.linalg.norm(r["F"])
        assert np.linalg.norm(F[k] - r["F"]) <= 2e-3 * np.linalg.norm(r["F"])
        tot += r["stats"]["segments"]
    assert abs(st["segments"] - tot) <= 1e-3 * tot


@pytest.mark.parametrize("deposit", [0, 1])
@pytest.mark.parametrize("name,mode", [("boxwing", 0), ("room", 2)])
def test_glossy_torque_matches_oracle(ctx, oracle, name, mode, deposit):
    """The torque builds of the kernels with glossy facets and both deposit rules (every template combination the
    launcher can pick is exercised somewhere: this covers TORQUE x GLOSSY x ANALOG)."""
    cases, rng = _glossy_cases()
    if name == "boxwing":
        family, th = cases[name]
        th = th[:2]
        dz = ctx.srp_build_designs(family, th)
        meshes = {k: oracle.build_mesh(family, th[k], k=k) for k in range(len(th))}
    else:
        verts, mats = cases[name]
        dz = ctx.srp_build_designs_from_meshes(verts, mats, [0, len(verts)])
        meshes = {0: (verts, mats)}
    sumT = int(dz.tri_offsets[-1])
    sh = rng.choice([-1.0, 2.0, 60.0], sumT).astype(np.float32)
    ctx.srp_designs_set_shininess(dz, sh)
    sun = W.fibonacci_sphere(4)
    x_com = np.array([[0.3, -0.2, 0.5], [-0.4, 0.1, 0.0]], np.float32)[:dz.D]
    N, B = 1 << 12, 4
    ctx.srp_set_options(primary_mode=mode, deposit=deposit, escape_masks=2)
    try:
        F, T = ctx.srp_forces_torques(dz, cuda(sun), N, B, seed=12, x_com=x_com)
    finally:
        ctx.srp_set_options()
    F, T = F.cpu().numpy(), T.cpu().numpy()
    for k in range(dz.D):
        v, m = meshes[k]
        off = int(dz.tri_offsets[k])
        r = oracle.forces(v, m, sun, N, B, seed=12, k=k, deposit=deposit, x_com=x_com[k], shininess=sh[off:off + len(v)])
        assert_parity(F[k], r["F"], r["sigma"], tol_agg=3e-3)
        assert_parity(T[k], r["T"], r["sigma_T"], tol_agg=3e-3)
    dz.free()


def _random_mask_mesh(seed):
    """Random meshes for the mask stress test: a sparse soup of small triangles, scattered boxes (outward and inward
    normals, touching and nested), a paraboloid bowl (either winding) with objects inside and across it, stacks of
    tessellated near-coplanar plates with gaps from 1e-5 to 0.3."""
    from test_oracle_thermal import box
    rng = np.random.default_rng(100 + seed)
    kind = seed % 4
    if kind == 0:
        n = int(rng.integers(100, 3000)); sz = rng.uniform(0.01, 0.2)
        verts = (rng.uniform(-1, 1, (n, 1, 3)) + rng.normal(0, sz, (n, 3, 3))).astype(np.float32)
    elif kind == 1:
        bs = []
        for _ in range(int(rng.integers(6, 40))):
            lo = rng.uniform(-1, 1, 3)
            bs.append(box(lo, lo + rng.uniform(0.05, 0.6, 3), inward=bool(rng.integers(0, 2))))
        verts = np.concatenate(bs)
    elif kind == 2:
        n, depth, flip = int(rng.integers(8, 40)), rng.uniform(0.1, 1.5), bool(rng.integers(0, 2))
        P = lambda a, b: np.array([-1 + 2 * a / n, -1 + 2 * b / n, depth * ((-1 + 2 * a / n) ** 2 + (-1 + 2 * b / n) ** 2)])
        tris = []
        for i in range(n):
            for j in range(n):
                p00, p10, p11, p01 = P(i, j), P(i + 1, j), P(i + 1, j + 1), P(i, j + 1)
                tris += [[p00, p11, p10], [p00, p01, p11]] if flip else [[p00, p10, p11], [p00, p11, p01]]
        verts = np.concatenate([np.array(tris, np.float32), box([-0.1, -0.1, 0.5], [0.1, 0.1, 0.7]),
                                quad([-0.02, -1.2, 0.0], [0, 2.4, 0.9], [0.04, 0, 0])])
    else:
        ps, z = [], 0.0
        for _ in range(int(rng.integers(2, 6))):
            n, s, off = int(rng.integers(3, 14)), rng.uniform(0.3, 1.0), rng.uniform(-0.3, 0.3, 2)
            ps += [quad([off[0] - s + 2 * s * i / n, off[1] - s + 2 * s * j / n, z], [2 * s / n, 0, 0], [0, 2 * s / n, 0])
                   for i in range(n) for j in range(n)]
            z += 10 ** rng.uniform(-5, -0.5)
        verts = np.concatenate(ps).astype(np.float32)
    return verts.astype(np.float32)


@pytest.mark.parametrize("seed", range(16))
def test_escape_masks_random_meshes(ctx, seed):
    """Conservativeness of the mask build on geometry it was not tuned on: with the masks forced on, every photon
    path signature and every counter equals the run without masks."""
    verts = _random_mask_mesh(seed)
    mats = np.tile(np.array([[0.1, 0.6, 0.3]], np.float32), (len(verts), 1))
    dz = ctx.srp_build_designs_from_meshes(verts, mats, [0, len(verts)])
    sun = W.fibonacci_sphere(6) if seed % 3 else np.array([[0, 0, 1], [0, 0, -1], [1, 0, 0.01], [0.3, 0.3, 0.9], [0, 1, 0],
                                                            [-1, -1, -1]], np.float32)
    pairs = np.array([[0, j] for j in range(6)], np.int32)
    res = {}
    for masks in (0, 2):
        ctx.srp_set_options(primary_mode=1 + seed % 2, escape_masks=masks)
        try:
            F, st = run_pairs(ctx, dz, sun, pairs, 1 << 12, 6, seed=seed)
            sg = ctx.srp_path_signatures(dz, cuda(sun), pairs, 1 << 12, 6, seed).cpu().numpy()
        finally:
            ctx.srp_set_options()
        res[masks] = (F, st, sg)
    assert np.array_equal(res[0][2], res[2][2])
    for key in ("launched", "primary_miss", "absorbed", "escaped", "capped", "segments", "hits_at_depth"):
        assert res[0][1][key] == res[2][1][key], key
    assert np.abs(res[2][0] - res[0][0]).max() <= 2e-6 * np.abs(res[0][0]).max() + 1e-30
    dz.free()
