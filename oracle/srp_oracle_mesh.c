/*
 * srp_oracle_mesh.c -- TEST INFRASTRUCTURE ONLY.  CPU oracle, part 1 of 2:
 * the parametric "design parameters -> triangle mesh with per-face material"
 * map (Sec. 3.2: "The spacecraft is given as a mapping from
 * design parameters to triangle meshes with per-face Phong material
 * parameters").  The paper leaves the map to the user; the five
 * synthetic families are BASELINE.json's configs, laid out in DESIGN.md
 * "Mesh families" -- every number below is restated from that section.
 *
 * Everything is evaluated in fp64 and rounded once to fp32 (the mesh the
 * tracer sees is the fp32 one).  Compile with -ffp-contract=off so that the
 * arithmetic is plain IEEE and reproducible.
 *
 * A design is a list of PATCHES in a fixed order; triangles are numbered patch
 * by patch.  Patch kinds (local coordinates, then world = o + x*ex + y*ey + z*ez):
 *   PLANE (nu,nv):  p(i,j) = (i/nu, j/nv, 0) with ex, ey the full edge vectors.
 *                   cell c = j*nu+i -> tris (p00,p10,p11), (p00,p11,p01).
 *   HFIELD(nu,nv):  PLANE whose world z is replaced by amp*fbm(x,y)/norm.
 *   POLAR (nr,ns,R,c): q(i,j) = (rho cos phi, rho sin phi, c rho^2),
 *                   rho = R*i/nr, phi = 2 pi (j mod ns)/ns.  First ns tris: the
 *                   fan (q(0,0), q(1,j), q(1,j+1)); then ring i=1..nr-1, sector
 *                   j: (q(i,j), q(i+1,j), q(i+1,j+1)), (q(i,j), q(i+1,j+1), q(i,j+1)).
 *   TUBE  (ns,nl,r,len): q(i,j) = (r cos phi_i, r sin phi_i, len*j/nl);
 *                   cell c = j*ns+i -> (q(i,j), q(i+1,j), q(i+1,j+1)),
 *                   (q(i,j), q(i+1,j+1), q(i,j+1)).
 * The sail's gradient noise is defined by DESIGN.md, not by the paper; it is pinned
 * through srp_oracle_sail_height (tests/test_oracle_mesh.py: exact zeros on the
 * coarsest lattice, hand-expanded values at half- and quarter-cell points, the
 * lattice gradient, C2 continuity of the quintic fade).
 */
#include <stdlib.h>
#include <string.h>
#include "srp_oracle_common.h"

enum { FAM_PLATE = 0, FAM_BOXWING = 1, FAM_DETAILED = 2, FAM_BOXWING6 = 3, FAM_SAIL = 4, FAM_BOXWING_T = 5 };
enum { PK_PLANE = 0, PK_HFIELD = 1, PK_POLAR = 2, PK_TUBE = 3 };
enum { MAT_DIRICHLET = 0, MAT_FIXED = 1 };

typedef struct {
    int kind, n0, n1;      /* PLANE/HFIELD: nu,nv; POLAR: nr,ns; TUBE: ns,nl */
    orc_v3 o, ex, ey, ez;
    double a, b;           /* POLAR: R, c;  TUBE: r, len;  HFIELD: amp, unused */
    int mat_class;         /* index into the family's fixed materials */
} orc_patch;

#define ORC_MAX_PATCHES 64
#define ORC_TWO_PI 6.283185307179586476925286766559

static long patch_tris(const orc_patch *p)
{
    switch (p->kind) {
    case PK_PLANE: case PK_HFIELD: return 2L * p->n0 * p->n1;
    case PK_POLAR: return (long)p->n1 + 2L * (p->n0 - 1) * p->n1;
    default:       return 2L * p->n0 * p->n1;
    }
}

static orc_patch mk_plane(int nu, int nv, orc_v3 o, orc_v3 ex, orc_v3 ey, int mc)
{
    orc_patch p; memset(&p, 0, sizeof p);
    p.kind = PK_PLANE; p.n0 = nu; p.n1 = nv; p.o = o; p.ex = ex; p.ey = ey;
    p.ez = orc_mk(0, 0, 0); p.mat_class = mc;
    return p;
}
static orc_patch mk_polar(int nr, int ns, double R, double c, orc_v3 o, orc_v3 ex, orc_v3 ey,
                          orc_v3 ez, int mc)
{
    orc_patch p; memset(&p, 0, sizeof p);
    p.kind = PK_POLAR; p.n0 = nr; p.n1 = ns; p.a = R; p.b = c;
    p.o = o; p.ex = ex; p.ey = ey; p.ez = ez; p.mat_class = mc;
    return p;
}
static orc_patch mk_tube(int ns, int nl, double r, double len, orc_v3 o, orc_v3 ex, orc_v3 ey,
                         orc_v3 ez, int mc)
{
    orc_patch p; memset(&p, 0, sizeof p);
    p.kind = PK_TUBE; p.n0 = ns; p.n1 = nl; p.a = r; p.b = len;
    p.o = o; p.ex = ex; p.ey = ey; p.ez = ez; p.mat_class = mc;
    return p;
}

/* Cuboid centred at c with half extents (hx,hy,hz); face order -x,+x,-y,+y,-z,+z;
 * each face a PLANE of n x n cells. */
static int add_cuboid(orc_patch *out, orc_v3 c, double hx, double hy, double hz, int n, int mc)
{
    orc_v3 lo = orc_mk(c.x - hx, c.y - hy, c.z - hz);
    orc_v3 X = orc_mk(2.0 * hx, 0, 0), Y = orc_mk(0, 2.0 * hy, 0), Z = orc_mk(0, 0, 2.0 * hz);
    out[0] = mk_plane(n, n, lo, Y, Z, mc);
    out[1] = mk_plane(n, n, orc_mk(c.x + hx, lo.y, lo.z), Y, Z, mc);
    out[2] = mk_plane(n, n, lo, X, Z, mc);
    out[3] = mk_plane(n, n, orc_mk(lo.x, c.y + hy, lo.z), X, Z, mc);
    out[4] = mk_plane(n, n, lo, X, Y, mc);
    out[5] = mk_plane(n, n, orc_mk(lo.x, lo.y, c.z + hz), X, Y, mc);
    return 6;
}

/* A solar panel: width 1.6 along a(phi) = (cos phi, 0, sin phi), centred on the
 * y axis, from y = sgn*y0 to sgn*(y0+len). */
static orc_patch mk_panel(double phi, double sgn, double y0, double len, int nu, int nv, int mc)
{
    double ca = cos(phi), sa = sin(phi);
    orc_v3 o = orc_mk(-0.8 * ca, sgn * y0, -0.8 * sa);
    orc_v3 ex = orc_mk(1.6 * ca, 0, 1.6 * sa);
    orc_v3 ey = orc_mk(0, sgn * len, 0);
    return mk_plane(nu, nv, o, ex, ey, mc);
}

/* Closed prism along the unit axis ez from point A: tube + cap at A + cap at A+len*ez. */
static int add_capped_tube(orc_patch *out, int ns, int nl, double r, double len, orc_v3 A,
                           orc_v3 ex, orc_v3 ey, orc_v3 ez, int mc)
{
    orc_v3 B = orc_add(A, orc_scale(ez, len));
    out[0] = mk_tube(ns, nl, r, len, A, ex, ey, ez, mc);
    out[1] = mk_polar(1, ns, r, 0.0, A, ex, ey, ez, mc);
    out[2] = mk_polar(1, ns, r, 0.0, B, ex, ey, ez, mc);
    return 3;
}

static const double SGN4[4][2] = { {1, 1}, {-1, 1}, {-1, -1}, {1, -1} };

/* Builds the patch list of one design.  theta = the design's fp32 parameters. */
static int family_patches(int family, const float *theta, orc_patch *P)
{
    int n = 0;
    switch (family) {
    case FAM_PLATE:
        P[n++] = mk_plane(1, 1, orc_mk(-0.5, -0.5, 0), orc_mk(1, 0, 0), orc_mk(0, 1, 0), 0);
        break;
    case FAM_BOXWING: {
        double L = (double)theta[0], phi = (double)theta[1];
        n += add_cuboid(P + n, orc_mk(0, 0, 0), 0.75, 0.75, 1.0, 1, 0);
        P[n++] = mk_panel(phi, 1.0, 1.15, L, 1, 1, 0);
        P[n++] = mk_panel(phi, -1.0, 1.15, L, 1, 1, 0);
        break;
    }
    case FAM_BOXWING_T: {   /* the box-wing of FAM_BOXWING, tessellated: "a representative satellite model (1 k faces)" */
        double L = (double)theta[0], phi = (double)theta[1];
        n += add_cuboid(P + n, orc_mk(0, 0, 0), 0.75, 0.75, 1.0, 8, 0);
        P[n++] = mk_panel(phi, 1.0, 1.15, L, 8, 16, 0);
        P[n++] = mk_panel(phi, -1.0, 1.15, L, 8, 16, 0);
        break;
    }
    case FAM_BOXWING6: {
        double phi1 = (double)theta[0], phi2 = (double)theta[1], L = (double)theta[2];
        double asp = (double)theta[3];
        n += add_cuboid(P + n, orc_mk(0, 0, 0), 0.75, 0.75, asp, 1, 0);
        P[n++] = mk_panel(phi1, 1.0, 1.15, L, 1, 1, 1);
        P[n++] = mk_panel(phi2, -1.0, 1.15, L, 1, 1, 1);
        break;
    }
    case FAM_DETAILED: {
        double td = (double)theta[0], pp = (double)theta[1];
        double cd = cos(td), sd = sin(td);
        n += add_cuboid(P + n, orc_mk(0, 0, 0), 0.75, 0.75, 1.0, 24, 0);
        P[n++] = mk_polar(48, 128, 1.2, 1.0 / (4.0 * 0.45), orc_mk(0, 0, 2.6), orc_mk(1, 0, 0),
                          orc_mk(0, cd, sd), orc_mk(0, -sd, cd), 0);
        for (int c = 0; c < 4; ++c)
            n += add_capped_tube(P + n, 64, 16, 0.05, 1.5,
                                 orc_mk(0.5 * SGN4[c][0], 0.5 * SGN4[c][1], -1.0),
                                 orc_mk(1, 0, 0), orc_mk(0, -1, 0), orc_mk(0, 0, -1), 0);
        for (int w = 0; w < 2; ++w)
            for (int m = 0; m < 4; ++m)
                P[n++] = mk_panel(pp, w == 0 ? 1.0 : -1.0, 1.15 + 2.1 * (double)m, 2.0, 32, 40, 0);
        for (int s = 0; s < 12; ++s) {
            orc_v3 A, ez, ex, ey; double len;
            if (s < 4) {            /* dish supports: bus top -> dish vertex */
                A = orc_mk(0.6 * SGN4[s][0], 0.6 * SGN4[s][1], 1.0);
                orc_v3 d = orc_sub(orc_mk(0, 0, 2.6), A);
                len = sqrt(orc_dot(d, d));
                ez = orc_mk(d.x / len, d.y / len, d.z / len);
            } else if (s < 8) {     /* yoke struts across the 0.4 m gap */
                double sx = (s & 1) ? -1.0 : 1.0, sy = (s < 6) ? 1.0 : -1.0;
                A = orc_mk(0.3 * sx, 0.75 * sy, 0.0);
                ez = orc_mk(0, sy, 0); len = 0.4;
            } else {                /* outriggers on the +-x faces */
                double sx = (s < 10) ? 1.0 : -1.0, sy = (s & 1) ? -1.0 : 1.0;
                A = orc_mk(0.75 * sx, 0.4 * sy, 0.5);
                ez = orc_mk(sx, 0, 0); len = 1.0;
            }
            orc_basis(ez, &ex, &ey);
            n += add_capped_tube(P + n, 6, 10, 0.03, len, A, ex, ey, ez, 0);
        }
        break;
    }
    case FAM_SAIL: {
        orc_patch h = mk_plane(707, 707, orc_mk(-20, -20, 0), orc_mk(40, 0, 0), orc_mk(0, 40, 0), 0);
        h.kind = PK_HFIELD; h.a = (double)theta[0];
        P[n++] = h;
        n += add_cuboid(P + n, orc_mk(0, 0, -0.7), 0.5, 0.5, 0.5, 40, 0);
        for (int b = 0; b < 4; ++b) {
            double inv = 1.0 / sqrt(2.0);
            orc_v3 ez = orc_mk(SGN4[b][0] * inv, SGN4[b][1] * inv, 0), ex, ey;
            orc_basis(ez, &ex, &ey);
            P[n++] = mk_tube(4, 25, 0.02 * sqrt(2.0), sqrt(800.0), orc_mk(0, 0, -0.1), ex, ey, ez, 0);
        }
        break;
    }
    default: return -1;
    }
    return n;
}

/* ---- sail height field: 4-octave 2-D gradient noise ---- */
static double lattice_angle(int ix, int iy, int oct, uint64_t mesh_seed)
{
    uint32_t ctr[4] = { (uint32_t)ix, (uint32_t)iy, (uint32_t)oct, 0xC0u };
    uint32_t key[2] = { (uint32_t)mesh_seed, (uint32_t)(mesh_seed >> 32) }, r[4];
    orc_philox4x32_10(ctr, key, r);
    return ORC_TWO_PI * orc_uniform(r[0]);
}
static double fade5(double t) { return t * t * t * (t * (t * 6.0 - 15.0) + 10.0); }
static double corner_dot(int ix, int iy, int oct, uint64_t seed, double dx, double dy)
{
    double ang = lattice_angle(ix, iy, oct, seed);
    return cos(ang) * dx + sin(ang) * dy;
}
static double gnoise(double X, double Y, int oct, uint64_t seed)
{
    double fxl = floor(X), fyl = floor(Y);
    int ix = (int)fxl, iy = (int)fyl;
    double fx = X - fxl, fy = Y - fyl;
    double n00 = corner_dot(ix, iy, oct, seed, fx, fy);
    double n10 = corner_dot(ix + 1, iy, oct, seed, fx - 1.0, fy);
    double n01 = corner_dot(ix, iy + 1, oct, seed, fx, fy - 1.0);
    double n11 = corner_dot(ix + 1, iy + 1, oct, seed, fx - 1.0, fy - 1.0);
    double u = fade5(fx), v = fade5(fy);
    double a = n00 + u * (n10 - n00);
    double b = n01 + u * (n11 - n01);
    return a + v * (b - a);
}
static double sail_height(double x, double y, double amp, uint64_t seed)
{
    double f = 0.0, w = 1.0, s = 1.0;
    for (int oct = 0; oct < 4; ++oct) {
        f += w * gnoise(s * x / 8.0, s * y / 8.0, oct, seed);
        w *= 0.5; s *= 2.0;
    }
    return amp * f / (1.875 * sqrt(0.5));
}

/* Height of the sail's surface above (x, y), exported so that the noise can be pinned on its own. */
double srp_oracle_sail_height(double x, double y, double amp, uint64_t mesh_seed)
{
    return sail_height(x, y, amp, mesh_seed);
}

/* ---- vertex of a patch ---- */
static orc_v3 to_world(const orc_patch *p, double x, double y, double z)
{
    return orc_mk(p->o.x + x * p->ex.x + y * p->ey.x + z * p->ez.x,
                  p->o.y + x * p->ex.y + y * p->ey.y + z * p->ez.y,
                  p->o.z + x * p->ex.z + y * p->ey.z + z * p->ez.z);
}
static orc_v3 patch_vertex(const orc_patch *p, int i, int j, uint64_t seed)
{
    switch (p->kind) {
    case PK_PLANE:
        return to_world(p, (double)i / p->n0, (double)j / p->n1, 0.0);
    case PK_HFIELD: {
        orc_v3 w = to_world(p, (double)i / p->n0, (double)j / p->n1, 0.0);
        w.z = sail_height(w.x, w.y, p->a, seed);
        return w;
    }
    case PK_POLAR: {
        double rho = p->a * (double)i / p->n0;
        double phi = ORC_TWO_PI * (double)(j % p->n1) / p->n1;
        return to_world(p, rho * cos(phi), rho * sin(phi), p->b * rho * rho);
    }
    default: {
        double phi = ORC_TWO_PI * (double)(i % p->n0) / p->n0;
        return to_world(p, p->a * cos(phi), p->a * sin(phi), p->b * (double)j / p->n1);
    }
    }
}

/* The three vertices of triangle t (patch-local index) of patch p. */
static void patch_triangle(const orc_patch *p, long t, uint64_t seed, orc_v3 v[3])
{
    int i, j, h;
    if (p->kind == PK_POLAR) {
        int ns = p->n1;
        if (t < ns) {
            v[0] = patch_vertex(p, 0, 0, seed);
            v[1] = patch_vertex(p, 1, (int)t, seed);
            v[2] = patch_vertex(p, 1, (int)t + 1, seed);
            return;
        }
        t -= ns; h = (int)(t & 1); t >>= 1;
        i = 1 + (int)(t / ns); j = (int)(t % ns);
    } else {
        int nu = p->n0;
        h = (int)(t & 1); t >>= 1;
        j = (int)(t / nu); i = (int)(t % nu);
    }
    if (p->kind == PK_POLAR) {           /* (i,j) = (ring, sector): ring is the first index */
        v[0] = patch_vertex(p, i, j, seed);
        if (h == 0) { v[1] = patch_vertex(p, i + 1, j, seed); v[2] = patch_vertex(p, i + 1, j + 1, seed); }
        else        { v[1] = patch_vertex(p, i + 1, j + 1, seed); v[2] = patch_vertex(p, i, j + 1, seed); }
    } else {
        v[0] = patch_vertex(p, i, j, seed);
        if (h == 0) { v[1] = patch_vertex(p, i + 1, j, seed); v[2] = patch_vertex(p, i + 1, j + 1, seed); }
        else        { v[1] = patch_vertex(p, i + 1, j + 1, seed); v[2] = patch_vertex(p, i, j + 1, seed); }
    }
}

/* ---- per-facet material ---- */
static void dirichlet222(long f, int k, uint64_t mesh_seed, double m[3])
{
    uint32_t key[2] = { (uint32_t)mesh_seed, (uint32_t)(mesh_seed >> 32) };
    uint32_t c0[4] = { (uint32_t)f, (uint32_t)k, 0u, 0xB0u }, c1[4] = { (uint32_t)f, (uint32_t)k, 1u, 0xB0u };
    uint32_t r0[4], r1[4];
    orc_philox4x32_10(c0, key, r0);
    orc_philox4x32_10(c1, key, r1);
    double g0 = -log(orc_uniform(r0[0]) * orc_uniform(r0[1]));
    double g1 = -log(orc_uniform(r0[2]) * orc_uniform(r0[3]));
    double g2 = -log(orc_uniform(r1[0]) * orc_uniform(r1[1]));
    double s = g0 + g1 + g2;
    m[0] = g0 / s; m[1] = g1 / s; m[2] = g2 / s;
}

int srp_oracle_n_params(int family)
{
    switch (family) {
    case FAM_PLATE: return 3; case FAM_BOXWING: return 2; case FAM_DETAILED: return 2;
    case FAM_BOXWING6: return 6; case FAM_SAIL: return 1; case FAM_BOXWING_T: return 2; default: return -1;
    }
}

long srp_oracle_tri_count(int family)
{
    static const float zero[8] = {0};
    orc_patch P[ORC_MAX_PATCHES];
    int n = family_patches(family, zero, P);
    if (n < 0) return -1;
    long T = 0;
    for (int q = 0; q < n; ++q) T += patch_tris(&P[q]);
    return T;
}

/*
 * Mesh of design k of a batch.  theta: the design's n_params fp32 parameters.
 * verts: float[T][3][3] (v0,v1,v2), mats: float[T][3] = (alpha, rho_s, rho_d).
 * Returns T, or -1 on a bad family.
 */
long srp_oracle_build_mesh(int family, const float *theta, int k, uint64_t mesh_seed,
                           float *verts, float *mats)
{
    orc_patch P[ORC_MAX_PATCHES];
    int n = family_patches(family, theta, P);
    if (n < 0) return -1;
    double fixed[2][3] = { {0, 0, 0}, {0, 0, 0} };
    int mat_mode = MAT_DIRICHLET;
    if (family == FAM_PLATE) {
        mat_mode = MAT_FIXED;
        fixed[0][0] = theta[0]; fixed[0][1] = theta[1]; fixed[0][2] = theta[2];
    } else if (family == FAM_SAIL) {
        mat_mode = MAT_FIXED;
        fixed[0][0] = 0.08; fixed[0][1] = 0.88; fixed[0][2] = 0.04;
    } else if (family == FAM_BOXWING6) {
        mat_mode = MAT_FIXED;
        double rs = (double)theta[4], rd = (double)theta[5];
        fixed[1][0] = 0.9 * (1.0 - rs); fixed[1][1] = rs; fixed[1][2] = 0.1 * (1.0 - rs);
        fixed[0][0] = 0.8 * (1.0 - rd); fixed[0][1] = 0.2 * (1.0 - rd); fixed[0][2] = rd;
    }
    long f = 0;
    for (int q = 0; q < n; ++q) {
        long nt = patch_tris(&P[q]);
        for (long t = 0; t < nt; ++t, ++f) {
            orc_v3 v[3];
            patch_triangle(&P[q], t, mesh_seed, v);
            for (int c = 0; c < 3; ++c) {
                verts[f * 9 + c * 3 + 0] = (float)v[c].x;
                verts[f * 9 + c * 3 + 1] = (float)v[c].y;
                verts[f * 9 + c * 3 + 2] = (float)v[c].z;
            }
            double m[3];
            if (mat_mode == MAT_DIRICHLET) dirichlet222(f, k, mesh_seed, m);
            else { m[0] = fixed[P[q].mat_class][0]; m[1] = fixed[P[q].mat_class][1]; m[2] = fixed[P[q].mat_class][2]; }
            mats[f * 3 + 0] = (float)m[0]; mats[f * 3 + 1] = (float)m[1]; mats[f * 3 + 2] = (float)m[2];
        }
    }
    return f;
}
