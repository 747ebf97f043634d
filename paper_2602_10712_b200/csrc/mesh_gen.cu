// mesh_gen.cu -- S0 of the hot path: design parameters theta_k -> triangle soup with per-facet
// (alpha, rho_s, rho_d)  ("mapping from design parameters to triangle meshes with
// per-face Phong material parameters"; the five families are BASELINE.json's configs, defined in
// DESIGN.md "Mesh families").
//
// Two kernels: (1) one thread per design expands theta into a table of parametric patches,
// (2) one thread per triangle evaluates its three vertices and its material.  Geometry is
// evaluated in fp64 and rounded once to fp32; this file is compiled with --fmad=false so that
// the arithmetic is plain IEEE (a one-off build step, not the hot loop).
#include "srp_internal.cuh"

namespace {

enum { PK_PLANE = 0, PK_HFIELD = 1, PK_POLAR = 2, PK_TUBE = 3 };
constexpr int MAX_PATCHES = 64;
constexpr double TWO_PI = 6.283185307179586476925286766559;

struct d3 { double x, y, z; };
__device__ inline d3 mk(double x, double y, double z) { d3 r; r.x = x; r.y = y; r.z = z; return r; }

struct Patch {
    int kind, n0, n1, mat_class;
    d3 o, ex, ey, ez;
    double a, b;
};

__device__ inline long long patch_tris(const Patch &p)
{
    if (p.kind == PK_POLAR) return (long long)p.n1 + 2LL * (p.n0 - 1) * p.n1;
    return 2LL * p.n0 * p.n1;
}

__device__ inline void philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                              uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
__device__ inline double uniform(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }

__device__ inline void basis(d3 s, d3 &u, d3 &v)
{
    double sign = copysign(1.0, s.z);
    double a = -1.0 / (sign + s.z);
    double b = s.x * s.y * a;
    u = mk(1.0 + sign * s.x * s.x * a, sign * b, -sign * s.x);
    v = mk(b, sign + s.y * s.y * a, -s.y);
}

__device__ inline Patch plane(int nu, int nv, d3 o, d3 ex, d3 ey, int mc)
{
    Patch p; p.kind = PK_PLANE; p.n0 = nu; p.n1 = nv; p.mat_class = mc;
    p.o = o; p.ex = ex; p.ey = ey; p.ez = mk(0, 0, 0); p.a = 0; p.b = 0;
    return p;
}
__device__ inline Patch polar(int nr, int ns, double R, double c, d3 o, d3 ex, d3 ey, d3 ez, int mc)
{
    Patch p; p.kind = PK_POLAR; p.n0 = nr; p.n1 = ns; p.mat_class = mc;
    p.o = o; p.ex = ex; p.ey = ey; p.ez = ez; p.a = R; p.b = c;
    return p;
}
__device__ inline Patch tube(int ns, int nl, double r, double len, d3 o, d3 ex, d3 ey, d3 ez, int mc)
{
    Patch p; p.kind = PK_TUBE; p.n0 = ns; p.n1 = nl; p.mat_class = mc;
    p.o = o; p.ex = ex; p.ey = ey; p.ez = ez; p.a = r; p.b = len;
    return p;
}

// cuboid centred at c, half extents h; faces -x,+x,-y,+y,-z,+z, n x n cells each
__device__ int cuboid(Patch *out, d3 c, double hx, double hy, double hz, int n, int mc)
{
    d3 lo = mk(c.x - hx, c.y - hy, c.z - hz);
    d3 X = mk(2.0 * hx, 0, 0), Y = mk(0, 2.0 * hy, 0), Z = mk(0, 0, 2.0 * hz);
    out[0] = plane(n, n, lo, Y, Z, mc);
    out[1] = plane(n, n, mk(c.x + hx, lo.y, lo.z), Y, Z, mc);
    out[2] = plane(n, n, lo, X, Z, mc);
    out[3] = plane(n, n, mk(lo.x, c.y + hy, lo.z), X, Z, mc);
    out[4] = plane(n, n, lo, X, Y, mc);
    out[5] = plane(n, n, mk(lo.x, lo.y, c.z + hz), X, Y, mc);
    return 6;
}

// solar panel of width 1.6 along a(phi) = (cos phi, 0, sin phi), from y = sgn*y0 to sgn*(y0+len)
__device__ Patch panel(double phi, double sgn, double y0, double len, int nu, int nv, int mc)
{
    double ca = cos(phi), sa = sin(phi);
    return plane(nu, nv, mk(-0.8 * ca, sgn * y0, -0.8 * sa), mk(1.6 * ca, 0, 1.6 * sa),
                 mk(0, sgn * len, 0), mc);
}

__device__ int capped_tube(Patch *out, int ns, int nl, double r, double len, d3 A, d3 ex, d3 ey,
                           d3 ez, int mc)
{
    d3 B = mk(A.x + ez.x * len, A.y + ez.y * len, A.z + ez.z * len);
    out[0] = tube(ns, nl, r, len, A, ex, ey, ez, mc);
    out[1] = polar(1, ns, r, 0.0, A, ex, ey, ez, mc);
    out[2] = polar(1, ns, r, 0.0, B, ex, ey, ez, mc);
    return 3;
}

__device__ int family_patches(int family, const float *theta, Patch *P)
{
    const double SG[4][2] = { {1, 1}, {-1, 1}, {-1, -1}, {1, -1} };
    int n = 0;
    switch (family) {
    case SRP_FAMILY_PLATE:
        P[n++] = plane(1, 1, mk(-0.5, -0.5, 0), mk(1, 0, 0), mk(0, 1, 0), 0);
        break;
    case SRP_FAMILY_BOXWING: {
        double L = (double)theta[0], phi = (double)theta[1];
        n += cuboid(P + n, mk(0, 0, 0), 0.75, 0.75, 1.0, 1, 0);
        P[n++] = panel(phi, 1.0, 1.15, L, 1, 1, 0);
        P[n++] = panel(phi, -1.0, 1.15, L, 1, 1, 0);
        break;
    }
    case SRP_FAMILY_BOXWING_T: {          // the box-wing, tessellated to ~1 k faces
        double L = (double)theta[0], phi = (double)theta[1];
        n += cuboid(P + n, mk(0, 0, 0), 0.75, 0.75, 1.0, 8, 0);
        P[n++] = panel(phi, 1.0, 1.15, L, 8, 16, 0);
        P[n++] = panel(phi, -1.0, 1.15, L, 8, 16, 0);
        break;
    }
    case SRP_FAMILY_BOXWING6: {
        double phi1 = (double)theta[0], phi2 = (double)theta[1], L = (double)theta[2];
        double asp = (double)theta[3];
        n += cuboid(P + n, mk(0, 0, 0), 0.75, 0.75, asp, 1, 0);
        P[n++] = panel(phi1, 1.0, 1.15, L, 1, 1, 1);
        P[n++] = panel(phi2, -1.0, 1.15, L, 1, 1, 1);
        break;
    }
    case SRP_FAMILY_DETAILED: {
        double td = (double)theta[0], pp = (double)theta[1];
        double cd = cos(td), sd = sin(td);
        n += cuboid(P + n, mk(0, 0, 0), 0.75, 0.75, 1.0, 24, 0);
        P[n++] = polar(48, 128, 1.2, 1.0 / (4.0 * 0.45), mk(0, 0, 2.6), mk(1, 0, 0), mk(0, cd, sd),
                       mk(0, -sd, cd), 0);
        for (int c = 0; c < 4; ++c)
            n += capped_tube(P + n, 64, 16, 0.05, 1.5, mk(0.5 * SG[c][0], 0.5 * SG[c][1], -1.0),
                             mk(1, 0, 0), mk(0, -1, 0), mk(0, 0, -1), 0);
        for (int w = 0; w < 2; ++w)
            for (int m = 0; m < 4; ++m)
                P[n++] = panel(pp, w == 0 ? 1.0 : -1.0, 1.15 + 2.1 * (double)m, 2.0, 32, 40, 0);
        for (int s = 0; s < 12; ++s) {
            d3 A, ez, ex, ey; double len;
            if (s < 4) {
                A = mk(0.6 * SG[s][0], 0.6 * SG[s][1], 1.0);
                d3 d = mk(0.0 - A.x, 0.0 - A.y, 2.6 - A.z);
                len = sqrt(d.x * d.x + d.y * d.y + d.z * d.z);
                ez = mk(d.x / len, d.y / len, d.z / len);
            } else if (s < 8) {
                double sx = (s & 1) ? -1.0 : 1.0, sy = (s < 6) ? 1.0 : -1.0;
                A = mk(0.3 * sx, 0.75 * sy, 0.0);
                ez = mk(0, sy, 0); len = 0.4;
            } else {
                double sx = (s < 10) ? 1.0 : -1.0, sy = (s & 1) ? -1.0 : 1.0;
                A = mk(0.75 * sx, 0.4 * sy, 0.5);
                ez = mk(sx, 0, 0); len = 1.0;
            }
            basis(ez, ex, ey);
            n += capped_tube(P + n, 6, 10, 0.03, len, A, ex, ey, ez, 0);
        }
        break;
    }
    case SRP_FAMILY_SAIL: {
        Patch h = plane(707, 707, mk(-20, -20, 0), mk(40, 0, 0), mk(0, 40, 0), 0);
        h.kind = PK_HFIELD; h.a = (double)theta[0];
        P[n++] = h;
        n += cuboid(P + n, mk(0, 0, -0.7), 0.5, 0.5, 0.5, 40, 0);
        for (int b = 0; b < 4; ++b) {
            double inv = 1.0 / sqrt(2.0);
            d3 ez = mk(SG[b][0] * inv, SG[b][1] * inv, 0), ex, ey;
            basis(ez, ex, ey);
            P[n++] = tube(4, 25, 0.02 * sqrt(2.0), sqrt(800.0), mk(0, 0, -0.1), ex, ey, ez, 0);
        }
        break;
    }
    default: break;
    }
    return n;
}

// ---- sail height field: 4 octaves of 2-D gradient noise ----
__device__ double corner_dot(int ix, int iy, int oct, uint32_t k0, uint32_t k1, double dx, double dy)
{
    uint32_t r[4];
    philox((uint32_t)ix, (uint32_t)iy, (uint32_t)oct, 0xC0u, k0, k1, r);
    double ang = TWO_PI * uniform(r[0]);
    return cos(ang) * dx + sin(ang) * dy;
}
__device__ inline double fade5(double t) { return t * t * t * (t * (t * 6.0 - 15.0) + 10.0); }
__device__ double gnoise(double X, double Y, int oct, uint32_t k0, uint32_t k1)
{
    double fxl = floor(X), fyl = floor(Y);
    int ix = (int)fxl, iy = (int)fyl;
    double fx = X - fxl, fy = Y - fyl;
    double n00 = corner_dot(ix, iy, oct, k0, k1, fx, fy);
    double n10 = corner_dot(ix + 1, iy, oct, k0, k1, fx - 1.0, fy);
    double n01 = corner_dot(ix, iy + 1, oct, k0, k1, fx, fy - 1.0);
    double n11 = corner_dot(ix + 1, iy + 1, oct, k0, k1, fx - 1.0, fy - 1.0);
    double u = fade5(fx), v = fade5(fy);
    double a = n00 + u * (n10 - n00);
    double b = n01 + u * (n11 - n01);
    return a + v * (b - a);
}
__device__ double sail_height(double x, double y, double amp, uint32_t k0, uint32_t k1)
{
    double f = 0.0, w = 1.0, s = 1.0;
    for (int oct = 0; oct < 4; ++oct) {
        f += w * gnoise(s * x / 8.0, s * y / 8.0, oct, k0, k1);
        w *= 0.5; s *= 2.0;
    }
    return amp * f / (1.875 * sqrt(0.5));
}

__device__ inline d3 to_world(const Patch &p, double x, double y, double z)
{
    return mk(p.o.x + x * p.ex.x + y * p.ey.x + z * p.ez.x,
              p.o.y + x * p.ex.y + y * p.ey.y + z * p.ez.y,
              p.o.z + x * p.ex.z + y * p.ey.z + z * p.ez.z);
}

__device__ d3 patch_vertex(const Patch &p, int i, int j, uint32_t k0, uint32_t k1)
{
    if (p.kind == PK_PLANE) return to_world(p, (double)i / p.n0, (double)j / p.n1, 0.0);
    if (p.kind == PK_HFIELD) {
        d3 w = to_world(p, (double)i / p.n0, (double)j / p.n1, 0.0);
        w.z = sail_height(w.x, w.y, p.a, k0, k1);
        return w;
    }
    if (p.kind == PK_POLAR) {
        double rho = p.a * (double)i / p.n0;
        double phi = TWO_PI * (double)(j % p.n1) / p.n1;
        return to_world(p, rho * cos(phi), rho * sin(phi), p.b * rho * rho);
    }
    double phi = TWO_PI * (double)(i % p.n0) / p.n0;
    return to_world(p, p.a * cos(phi), p.a * sin(phi), p.b * (double)j / p.n1);
}

__global__ void patch_table_kernel(int family, const float *theta, int D, int n_params,
                                   Patch *patches, int *n_patches)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= D) return;
    int n = family_patches(family, theta + (size_t)k * n_params, patches + (size_t)k * MAX_PATCHES);
    if (k == 0) *n_patches = n;
}

__global__ void __launch_bounds__(128)
mesh_triangles_kernel(int family, const float *theta, int D, int n_params, uint32_t k0, uint32_t k1,
                      long long T, const Patch *patches, const int *n_patches, float *verts, float *mats,
                      uint32_t k_offset /* index of design 0 in the Philox counters of the material draws */)
{
    long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= (long long)D * T) return;
    const int k = (int)(g / T);
    long long t = g - (long long)k * T;
    const long long f = t;
    const Patch *P = patches + (size_t)k * MAX_PATCHES;
    int q = 0;
    const int np = *n_patches;
    for (; q < np - 1; ++q) {
        long long nt = patch_tris(P[q]);
        if (t < nt) break;
        t -= nt;
    }
    const Patch p = P[q];
    int i, j, h;
    d3 v0, v1, v2;
    if (p.kind == PK_POLAR && t < p.n1) {
        v0 = patch_vertex(p, 0, 0, k0, k1);
        v1 = patch_vertex(p, 1, (int)t, k0, k1);
        v2 = patch_vertex(p, 1, (int)t + 1, k0, k1);
    } else {
        if (p.kind == PK_POLAR) {
            t -= p.n1; h = (int)(t & 1); t >>= 1;
            i = 1 + (int)(t / p.n1); j = (int)(t % p.n1);
        } else {
            h = (int)(t & 1); t >>= 1;
            j = (int)(t / p.n0); i = (int)(t % p.n0);
        }
        v0 = patch_vertex(p, i, j, k0, k1);
        if (h == 0) { v1 = patch_vertex(p, i + 1, j, k0, k1); v2 = patch_vertex(p, i + 1, j + 1, k0, k1); }
        else        { v1 = patch_vertex(p, i + 1, j + 1, k0, k1); v2 = patch_vertex(p, i, j + 1, k0, k1); }
    }
    float *o = verts + (size_t)g * 9;
    o[0] = (float)v0.x; o[1] = (float)v0.y; o[2] = (float)v0.z;
    o[3] = (float)v1.x; o[4] = (float)v1.y; o[5] = (float)v1.z;
    o[6] = (float)v2.x; o[7] = (float)v2.y; o[8] = (float)v2.z;

    const float *th = theta + (size_t)k * n_params;
    double m0, m1, m2;
    if (family == SRP_FAMILY_PLATE) {
        m0 = th[0]; m1 = th[1]; m2 = th[2];
    } else if (family == SRP_FAMILY_SAIL) {
        m0 = 0.08; m1 = 0.88; m2 = 0.04;
    } else if (family == SRP_FAMILY_BOXWING6) {
        double rs = (double)th[4], rd = (double)th[5];
        if (p.mat_class == 1) { m0 = 0.9 * (1.0 - rs); m1 = rs; m2 = 0.1 * (1.0 - rs); }
        else                  { m0 = 0.8 * (1.0 - rd); m1 = 0.2 * (1.0 - rd); m2 = rd; }
    } else {                                   // per-facet Dirichlet(2,2,2)
        uint32_t r0[4], r1[4];
        philox((uint32_t)f, (uint32_t)k + k_offset, 0u, 0xB0u, k0, k1, r0);
        philox((uint32_t)f, (uint32_t)k + k_offset, 1u, 0xB0u, k0, k1, r1);
        double g0 = -log(uniform(r0[0]) * uniform(r0[1]));
        double g1 = -log(uniform(r0[2]) * uniform(r0[3]));
        double g2 = -log(uniform(r1[0]) * uniform(r1[1]));
        double s = g0 + g1 + g2;
        m0 = g0 / s; m1 = g1 / s; m2 = g2 / s;
    }
    float *mo = mats + (size_t)g * 3;
    mo[0] = (float)m0; mo[1] = (float)m1; mo[2] = (float)m2;
}

} // namespace

long long srp_family_tris_host(int family)
{
    switch (family) {
    case SRP_FAMILY_PLATE: return 2;
    case SRP_FAMILY_BOXWING: case SRP_FAMILY_BOXWING6: return 16;
    case SRP_FAMILY_DETAILED: return 6 * 2 * 24 * 24 + (128 + 2 * 47 * 128) + 4 * (2 * 64 * 16 + 2 * 64)
                                     + 8 * 2 * 32 * 40 + 12 * (2 * 6 * 10 + 2 * 6);
    case SRP_FAMILY_SAIL: return 2LL * 707 * 707 + 6 * 2 * 40 * 40 + 4 * 2 * 4 * 25;
    case SRP_FAMILY_BOXWING_T: return 6 * 2 * 8 * 8 + 2 * 2 * 8 * 16;
    default: return -1;
    }
}

cudaError_t srp_launch_mesh_gen(int family, const float *theta, int D, int n_params,
                                unsigned long long mesh_seed, long long T, float *verts, float *mats,
                                cudaMemPool_t pool, unsigned k_offset, cudaStream_t stream)
{
    Patch *patches = nullptr; int *n_patches = nullptr;
    cudaError_t e = cudaMallocFromPoolAsync((void **)&patches, sizeof(Patch) * MAX_PATCHES * (size_t)D, pool, stream);
    if (e != cudaSuccess) return e;
    e = cudaMallocFromPoolAsync((void **)&n_patches, sizeof(int), pool, stream);
    if (e != cudaSuccess) { cudaFreeAsync(patches, stream); return e; }
    patch_table_kernel<<<(D + 63) / 64, 64, 0, stream>>>(family, theta, D, n_params, patches, n_patches);
    long long total = (long long)D * T;
    mesh_triangles_kernel<<<(unsigned)((total + 127) / 128), 128, 0, stream>>>(
        family, theta, D, n_params, (uint32_t)mesh_seed, (uint32_t)(mesh_seed >> 32), T, patches,
        n_patches, verts, mats, k_offset);
    e = cudaGetLastError();
    cudaFreeAsync(patches, stream);
    cudaFreeAsync(n_patches, stream);
    return e;
}
