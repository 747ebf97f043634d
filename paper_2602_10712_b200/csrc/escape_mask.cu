// escape_mask.cu -- per-triangle "escape masks" (part of S1, the per-design build).
//
// Most bounce rays leave the spacecraft for good (91 % on the detailed config), yet each one walks the whole
// chain of BVH nodes that contain its origin before that is known.  For every triangle t and each of its two
// sides these kernels mark the direction bins (a cube map of the sphere, 6 x 6 cells per face, 216 bins) in which
// SOME ray that starts on t could hit another triangle; a bounce ray whose direction falls in an unmarked bin
// escapes, and the tracer counts it as such without a traversal.  The masks are conservative, so no result changes
// (R20): a triangle f is left out for side s of t only if all its vertices lie behind t's plane or are
// coplanar with it (within 1e-6 x the design's extent, the fp32 rounding of the vertices, plus 1e-4 rad x the
// clearance between the two: coplanar neighbours, which exact arithmetic never hits); otherwise every bin that
// meets the cone of directions from t's bounding sphere to the bounding sphere of f -- or of a whole BVH subtree,
// once that cone is narrow -- is marked.
//
// Designs with a BVH: one warp per cluster of 32 neighbouring triangles, depth-first over the design's BVH2
// (escape_mask_kernel).  Designs without (T <= 64): all pairs of triangles (escape_mask_small_kernel).
#include <cfloat>
#include "srp_internal.cuh"
#include "escape_bins.cuh"

namespace {

constexpr int ESC_STACK = 96;
#ifndef ESC_MAX_VISITS_DEF
#define ESC_MAX_VISITS_DEF 2000
#endif
constexpr int ESC_MAX_VISITS = ESC_MAX_VISITS_DEF;      // beyond this the triangle sits in cluttered surroundings: mark everything
#ifndef ESC_SIN_DESCEND_DEF
#define ESC_SIN_DESCEND_DEF 0.5f
#endif
constexpr float ESC_SIN_DESCEND = ESC_SIN_DESCEND_DEF;  // subtrees seen under a wider cone than this are opened.  0.5 / 2000 visits
                                                        // against 0.25 / 4000: the build of cfg3's 16 designs 114 -> 62 ms AND 4 % more
                                                        // escapes resolved (fewer clusters run into the visit cap and mark everything)
#ifndef ESC_SIN_SHARED_DEF
#define ESC_SIN_SHARED_DEF 0.8f
#endif
constexpr float ESC_SIN_SHARED = ESC_SIN_SHARED_DEF;   // leaf triangles seen from the cluster under a narrower cone share one cone
constexpr float ESC_ANGLE_EPS = 1.0e-4f;  // a triangle within this angle of the plane (seen from t) counts as coplanar

struct BinTable {                          // per block, in shared memory
    float cx[ESC_BINS], cy[ESC_BINS], cz[ESC_BINS];   // bin centre directions
    float cosb[ESC_BINS], sinb[ESC_BINS];             // angular radius of the bin about its centre
};

__device__ inline float3 cube_dir(int face, float s, float t)
{
    // face = 2 * axis + (negative ? 1 : 0); (s, t) = the other two coordinates over |major|, in axis order
    const float m = (face & 1) ? -1.0f : 1.0f;
    float3 d;
    if ((face >> 1) == 0) d = make_float3(m, s, t);
    else if ((face >> 1) == 1) d = make_float3(s, m, t);
    else d = make_float3(s, t, m);
    const float il = rsqrtf(d.x * d.x + d.y * d.y + d.z * d.z);
    return make_float3(d.x * il, d.y * il, d.z * il);
}

__device__ inline void fill_bin_table(BinTable &B)
{
    for (int b = threadIdx.x; b < ESC_BINS; b += blockDim.x) {
        const int face = b / (ESC_GRID * ESC_GRID), cell = b % (ESC_GRID * ESC_GRID);
        const int is = cell % ESC_GRID, it = cell / ESC_GRID;
        const float s0 = -1.0f + 2.0f * is / ESC_GRID, s1 = -1.0f + 2.0f * (is + 1) / ESC_GRID;
        const float t0 = -1.0f + 2.0f * it / ESC_GRID, t1 = -1.0f + 2.0f * (it + 1) / ESC_GRID;
        const float3 c = cube_dir(face, 0.5f * (s0 + s1), 0.5f * (t0 + t1));
        // the cell is a convex spherical quadrilateral: its farthest point from c is a corner
        float cmin = 1.0f;
        const float ss[2] = { s0, s1 }, tt[2] = { t0, t1 };
        for (int a = 0; a < 4; ++a) {
            const float3 k = cube_dir(face, ss[a & 1], tt[a >> 1]);
            cmin = fminf(cmin, c.x * k.x + c.y * k.y + c.z * k.z);
        }
        cmin = fmaxf(cmin - 2.0e-4f, -1.0f);              // slack for fp32 binning at cell borders
        B.cx[b] = c.x; B.cy[b] = c.y; B.cz[b] = c.z;
        B.cosb[b] = cmin; B.sinb[b] = sqrtf(fmaxf(0.0f, 1.0f - cmin * cmin));
    }
}

// The masks under construction: one 64-bit word per cube face (36 cells) and side, so that every index below is
// a compile-time constant and the words stay in registers.
struct FaceMasks { unsigned long long p[6], m[6]; };

constexpr unsigned FULLW = 0xffffffffu;

// The 216 bins that meet the cone (axis a, sin / cos of the half-angle), computed by the whole warp (lane l tests
// cells l and l + 32 of every face the cone can reach) and OR-ed into the masks of the lanes that see the occluder.
// A cube face spans 54.74 deg about its axis, so a face whose axis is farther than that plus the cone from a is skipped.
__device__ __forceinline__ void mark_cone(const BinTable &B, float3 a, float sina, float cosa, bool plus, bool minus,
                                          FaceMasks &M, int lane)
{
    const float cf = 0.57735f, sf = 0.81650f;                    // cos / sin of the face's angular radius
    const float cface = cosa * cf - sina * sf - 1.0e-3f;          // cos(alpha + 54.74 deg)
    const float fa[6] = { a.x, -a.x, a.y, -a.y, a.z, -a.z };
#pragma unroll
    for (int face = 0; face < 6; ++face) {
        if (fa[face] < cface) continue;                           // warp-uniform
        bool h0, h1 = false;
        {
            const int b = face * ESC_GRID * ESC_GRID + lane;      // cells 0..31
            // angle(a, centre_b) <= alpha + beta_b  <=>  dot >= cos(alpha + beta_b)   (alpha <= pi/2, beta < pi/4)
            h0 = a.x * B.cx[b] + a.y * B.cy[b] + a.z * B.cz[b] >= cosa * B.cosb[b] - sina * B.sinb[b];
        }
        if (lane < ESC_GRID * ESC_GRID - 32) {   // (compile-time grid: at most 32 more cells)
            const int b = face * ESC_GRID * ESC_GRID + 32 + lane; // cells 32..35
            h1 = a.x * B.cx[b] + a.y * B.cy[b] + a.z * B.cz[b] >= cosa * B.cosb[b] - sina * B.sinb[b];
        }
        const unsigned long long bits = (unsigned long long)__ballot_sync(FULLW, h0) |
                                        ((unsigned long long)__ballot_sync(FULLW, h1) << 32);
        if (plus) M.p[face] |= bits;
        if (minus) M.m[face] |= bits;
    }
}

// Per-lane version (leaf level, where every lane has its own cone about its own triangle).
__device__ __forceinline__ void mark_cone_lane(const BinTable &B, float3 a, float sina, float cosa, bool plus, bool minus, FaceMasks &M)
{
    const float cf = 0.57735f, sf = 0.81650f;
    const float cface = cosa * cf - sina * sf - 1.0e-3f;
    const float fa[6] = { a.x, -a.x, a.y, -a.y, a.z, -a.z };
#pragma unroll
    for (int face = 0; face < 6; ++face) {
        if (fa[face] < cface) continue;
        unsigned long long bits = 0ULL;
#pragma unroll 1
        for (int cell = 0; cell < ESC_GRID * ESC_GRID; ++cell) {
            const int b = face * ESC_GRID * ESC_GRID + cell;
            if (a.x * B.cx[b] + a.y * B.cy[b] + a.z * B.cz[b] >= cosa * B.cosb[b] - sina * B.sinb[b]) bits |= 1ULL << cell;
        }
        if (plus) M.p[face] |= bits;
        if (minus) M.m[face] |= bits;
    }
}

// One WARP per cluster of 32 consecutive (Morton-sorted, hence neighbouring) triangles of a design: the warp walks
// the BVH once for the cluster's bounding sphere -- node loads, cone widths and the marked bins are warp-uniform --
// and every lane applies its own triangle's plane to decide which of its two masks an occluder goes into.
__global__ void __launch_bounds__(128)
escape_mask_kernel(const DesignsDev dz, unsigned *esc)
{
    __shared__ BinTable B;
    __shared__ int s_stack[4][ESC_STACK];
    fill_bin_table(B);
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int k = blockIdx.y;
    const long long tbase = dz.tri_off[k];
    const int T = (int)(dz.tri_off[k + 1] - tbase);
    const int first_t = (blockIdx.x * 4 + warp) * 32;
    if (first_t >= T) return;
    const int t = first_t + lane;
    const bool live = t < T;
    const float4 *tri = dz.tri + 3 * tbase;
    const float4 *nodes = dz.nodes + 4 * tbase;
    int *stack = s_stack[warp];
    FaceMasks M;
#pragma unroll
    for (int w = 0; w < 6; ++w) M.p[w] = M.m[w] = 0ULL;

    const int tt = live ? t : first_t;                              // idle lanes copy the first triangle
    const float4 q0 = tri[3 * tt], q1 = tri[3 * tt + 1], q2 = tri[3 * tt + 2];
    float3 n = make_float3(q1.y * q2.z - q1.z * q2.y, q1.z * q2.x - q1.x * q2.z, q1.x * q2.y - q1.y * q2.x);
    const float nl = sqrtf(n.x * n.x + n.y * n.y + n.z * n.z);
    bool all = !(nl > 0.0f);                                       // degenerate facet (never a source): mark all
    if (!all) { n.x /= nl; n.y /= nl; n.z /= nl; } else n = make_float3(0.f, 0.f, 1.f);
    const float3 ct = make_float3(q0.x + (q1.x + q2.x) * (1.0f / 3.0f), q0.y + (q1.y + q2.y) * (1.0f / 3.0f),
                                  q0.z + (q1.z + q2.z) * (1.0f / 3.0f));
    float rt = 0.0f;                                               // bounding sphere of t about its centroid
    {
        const float3 v[3] = { make_float3(q0.x, q0.y, q0.z), make_float3(q0.x + q1.x, q0.y + q1.y, q0.z + q1.z),
                              make_float3(q0.x + q2.x, q0.y + q2.y, q0.z + q2.z) };
        for (int a = 0; a < 3; ++a) {
            const float dx = v[a].x - ct.x, dy = v[a].y - ct.y, dz_ = v[a].z - ct.z;
            rt = fmaxf(rt, sqrtf(dx * dx + dy * dy + dz_ * dz_));
        }
    }
    // the cluster's bounding sphere: mean of the centroids, radius = farthest lane sphere
    float3 cc = ct;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        cc.x += __shfl_xor_sync(FULLW, cc.x, o); cc.y += __shfl_xor_sync(FULLW, cc.y, o); cc.z += __shfl_xor_sync(FULLW, cc.z, o);
    }
    cc.x *= (1.0f / 32.0f); cc.y *= (1.0f / 32.0f); cc.z *= (1.0f / 32.0f);
    float rc = sqrtf((ct.x - cc.x) * (ct.x - cc.x) + (ct.y - cc.y) * (ct.y - cc.y) + (ct.z - cc.z) * (ct.z - cc.z)) + rt;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) rc = fmaxf(rc, __shfl_xor_sync(FULLW, rc, o));
    rc *= 1.0002f;
    const float4 blo = dz.box[2 * k], bhi = dz.box[2 * k + 1];
    const float eps = 1.0e-6f * (fmaxf(fabsf(blo.x), fabsf(bhi.x)) + fmaxf(fabsf(blo.y), fabsf(bhi.y)) +
                                 fmaxf(fabsf(blo.z), fabsf(bhi.z)));
    const float pd = n.x * q0.x + n.y * q0.y + n.z * q0.z;          // plane: n . x = pd

    int sp = 0, visits = 0;                                         // warp-uniform
    bool giveup = false, fullp = false, fullm = false;               // per lane: this side's mask is already full
    if (T > 1) { if (lane == 0) stack[0] = 0; sp = 1; }
    __syncwarp();
    while (sp > 0) {
        const int node = stack[--sp];
        __syncwarp();
        if (++visits > ESC_MAX_VISITS) { giveup = true; break; }
        if ((visits & 31) == 0) {                                   // a side whose mask is full has nothing to gain
            const unsigned long long cells = ESC_CELLS;
            bool fp_ = true, fm_ = true;
#pragma unroll
            for (int w = 0; w < 6; ++w) { fp_ = fp_ && (M.p[w] & cells) == cells; fm_ = fm_ && (M.m[w] & cells) == cells; }
            fullp = fp_; fullm = fm_;
            if (__all_sync(FULLW, fullp && fullm)) break;
        }
        const float4 n0 = __ldg(nodes + 4 * node), n1 = __ldg(nodes + 4 * node + 1), n2 = __ldg(nodes + 4 * node + 2),
                     n3 = __ldg(nodes + 4 * node + 3);
        const float bl[2][3] = { { n0.x, n0.y, n0.z }, { n1.z, n1.w, n2.x } };
        const float bh[2][3] = { { n0.w, n1.x, n1.y }, { n2.y, n2.z, n2.w } };
        const int link[2] = { __float_as_int(n3.x), __float_as_int(n3.y) };
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            if (!(bl[c][0] <= bh[c][0])) continue;                  // the empty slot of a one-triangle design
            const float cx = 0.5f * (bl[c][0] + bh[c][0]), cy = 0.5f * (bl[c][1] + bh[c][1]), cz = 0.5f * (bl[c][2] + bh[c][2]);
            const float hx = 0.5f * (bh[c][0] - bl[c][0]), hy = 0.5f * (bh[c][1] - bl[c][1]), hz = 0.5f * (bh[c][2] - bl[c][2]);
            // signed distance range of the box from THIS lane's plane
            const float dc = n.x * cx + n.y * cy + n.z * cz - pd;
            const float dr = fabsf(n.x) * hx + fabsf(n.y) * hy + fabsf(n.z) * hz;
            // slab half-width: geometry this close to the plane counts as coplanar with the triangle (R20).  eps covers
            // the fp32 rounding of the vertices; the angular term covers the error of the fp32 normal (from 5 cm
            // edges of vertices rounded to 1e-6 m: ~2e-5 rad) and grows with the CLEARANCE between the triangle and
            // the box, not with the box's size: a facet hovering just above the triangle keeps a slab of eps
            const float mx = fmaxf(fabsf(cx - ct.x) - hx, 0.0f), my = fmaxf(fabsf(cy - ct.y) - hy, 0.0f),
                        mz = fmaxf(fabsf(cz - ct.z) - hz, 0.0f);
            const float clear = fmaxf(sqrtf(mx * mx + my * my + mz * mz) - rt, 0.0f);
            const float slab = eps + ESC_ANGLE_EPS * clear;
            bool plus = dc + dr > slab, minus = dc - dr < -slab;
            if (link[c] >= 0 && (plus || minus)) {
                // the box of a tilted flat patch is fat; the subtree's own plane slab (lbvh.cu) is not.  If the
                // patch is parallel to this lane's plane within the angular margin, measure with the patch's normal
                // (an area-weighted mean, far more accurate than one small triangle's).  "Parallel" is judged to the
                // accuracy of this triangle's own fp32 normal, ang = min(ESC_ANGLE_EPS, 4 eps / rt) -- a large
                // triangle has an accurate normal -- so its own vertices deviate by at most ang * rt <= 4 eps from
                // its centroid's offset
                const float4 pn = __ldg(dz.nplane + 2 * (tbase + link[c])), pm = __ldg(dz.nplane + 2 * (tbase + link[c]) + 1);
                const float kx = n.y * pn.z - n.z * pn.y, ky = n.z * pn.x - n.x * pn.z, kz = n.x * pn.y - n.y * pn.x;
                const float ang = fminf(ESC_ANGLE_EPS, 4.0f * eps / rt);
                if (kx * kx + ky * ky + kz * kz <= ang * ang) {
                    const bool same = n.x * pn.x + n.y * pn.y + n.z * pn.z > 0.0f;
                    const float pc = pn.x * ct.x + pn.y * ct.y + pn.z * ct.z;
                    const float lo_d = same ? pn.w - pc : pc - pm.x, hi_d = same ? pm.x - pc : pc - pn.w;
                    const float slab_n = 2.0f * eps + ang * rt + ESC_ANGLE_EPS * clear;
                    plus = hi_d > slab_n; minus = lo_d < -slab_n;
                }
            }
            plus = plus && !fullp; minus = minus && !fullm;
            if (!__any_sync(FULLW, plus || minus)) continue;        // within every lane's slab (or nothing to gain): skip
            if (link[c] >= 0) {
                const float R = sqrtf(hx * hx + hy * hy + hz * hz);
                const float dx = cx - cc.x, dy = cy - cc.y, dzz = cz - cc.z;
                const float dist = sqrtf(dx * dx + dy * dy + dzz * dzz);
                const float sina = (R + rc) * 1.0001f / dist;
                if (!(sina < ESC_SIN_DESCEND)) {                    // wide cone (or NaN): open the subtree
                    if (sp < ESC_STACK) { if (lane == 0) stack[sp] = link[c]; ++sp; } else giveup = true;
                    continue;
                }
                // narrow enough: one cone from the cluster's sphere, its bins computed by the warp together
                const float il = 1.0f / dist;
                mark_cone(B, make_float3(dx * il, dy * il, dzz * il), sina, sqrtf(1.0f - sina * sina), plus, minus, M, lane);
            } else {                                                // leaf: its triangles, exactly
                const unsigned u = (unsigned)~link[c];
                const int first = (int)(u >> 3), cnt = (int)(u & 7u) + 1;
#pragma unroll 1
                for (int f = first; f < first + cnt; ++f) {
                    const float4 p0 = __ldg(tri + 3 * f), p1 = __ldg(tri + 3 * f + 1), p2 = __ldg(tri + 3 * f + 2);
                    const float3 v0 = make_float3(p0.x, p0.y, p0.z), v1 = make_float3(p0.x + p1.x, p0.y + p1.y, p0.z + p1.z),
                                 v2 = make_float3(p0.x + p2.x, p0.y + p2.y, p0.z + p2.z);
                    const float d0 = n.x * v0.x + n.y * v0.y + n.z * v0.z - pd, d1 = n.x * v1.x + n.y * v1.y + n.z * v1.z - pd,
                                d2 = n.x * v2.x + n.y * v2.y + n.z * v2.z - pd;
                    // clearance between the two triangles' bounding spheres (v0's distance less f's longest edge
                    // bounds f's nearest point from below)
                    const float e1l = sqrtf(p1.x * p1.x + p1.y * p1.y + p1.z * p1.z), e2l = sqrtf(p2.x * p2.x + p2.y * p2.y + p2.z * p2.z);
                    const float v0d = sqrtf((v0.x - ct.x) * (v0.x - ct.x) + (v0.y - ct.y) * (v0.y - ct.y) + (v0.z - ct.z) * (v0.z - ct.z));
                    const float slab_f = eps + ESC_ANGLE_EPS * fmaxf(v0d - fmaxf(e1l, e2l) - rt, 0.0f);
                    const bool fp = f != t && !fullp && fmaxf(d0, fmaxf(d1, d2)) > slab_f,
                               fm = f != t && !fullm && fminf(d0, fminf(d1, d2)) < -slab_f;
                    if (!__any_sync(FULLW, fp || fm)) continue;
                    const float3 cf = make_float3((v0.x + v1.x + v2.x) * (1.0f / 3.0f), (v0.y + v1.y + v2.y) * (1.0f / 3.0f),
                                                  (v0.z + v1.z + v2.z) * (1.0f / 3.0f));
                    float rf = 0.0f;
                    {
                        const float3 vv[3] = { v0, v1, v2 };
                        for (int a = 0; a < 3; ++a) {
                            const float ex = vv[a].x - cf.x, ey = vv[a].y - cf.y, ez = vv[a].z - cf.z;
                            rf = fmaxf(rf, sqrtf(ex * ex + ey * ey + ez * ez));
                        }
                    }
                    {   // not too close to the cluster: one shared cone (cheap)
                        const float gx = cf.x - cc.x, gy = cf.y - cc.y, gz = cf.z - cc.z;
                        const float gd = sqrtf(gx * gx + gy * gy + gz * gz);
                        const float gs = (rf + rc) * 1.0002f / gd;
                        if (gs < ESC_SIN_SHARED) {
                            const float gi = 1.0f / gd;
                            mark_cone(B, make_float3(gx * gi, gy * gi, gz * gi), gs, sqrtf(1.0f - gs * gs), fp, fm, M, lane);
                            continue;
                        }
                    }
                    // near field: every lane's own cone, from its triangle's sphere to f's
                    const float dx = cf.x - ct.x, dy = cf.y - ct.y, dzz = cf.z - ct.z;
                    const float dist = sqrtf(dx * dx + dy * dy + dzz * dzz);
                    const float sina = (rf + rt) * 1.0002f / dist;
                    if (!(fp || fm)) continue;
                    {   // nothing to add if this lane's masks of the sides that see f are full already
                        const unsigned long long cells = ESC_CELLS;
                        bool fullp = true, fullm = true;
#pragma unroll
                        for (int w = 0; w < 6; ++w) { fullp = fullp && (M.p[w] & cells) == cells; fullm = fullm && (M.m[w] & cells) == cells; }
                        if ((!fp || fullp) && (!fm || fullm)) continue;
                    }
                    if (!(sina < 1.0f)) {                           // touching / overlapping spheres: every direction
#pragma unroll
                        for (int w = 0; w < 6; ++w) { if (fp) M.p[w] = ~0ULL; if (fm) M.m[w] = ~0ULL; }
                        continue;
                    }
                    const float il = 1.0f / dist;
                    mark_cone_lane(B, make_float3(dx * il, dy * il, dzz * il), sina, sqrtf(1.0f - sina * sina), fp, fm, M);
                }
            }
        }
        __syncwarp();
    }
    if (giveup) all = true;                                         // cluttered surroundings: no escapes claimed
    if (!live) return;
    // pack: bit (face * 36 + cell) of the 216-bit mask of each side
    unsigned *out = esc + (size_t)(tbase + t) * (2 * ESC_WORDS);
    unsigned wp[ESC_WORDS + 2], wm[ESC_WORDS + 2];
#pragma unroll
    for (int w = 0; w < ESC_WORDS + 2; ++w) wp[w] = wm[w] = 0u;
#pragma unroll
    for (int face = 0; face < 6; ++face) {
        const int pos = face * ESC_GRID * ESC_GRID, w0 = pos >> 5, sh = pos & 31;
        const unsigned long long cells = ESC_CELLS;
        const unsigned long long a = M.p[face] & cells, b = M.m[face] & cells;
        wp[w0] |= (unsigned)(a << sh); wm[w0] |= (unsigned)(b << sh);
        if (w0 + 1 <= ESC_WORDS) { wp[w0 + 1] |= (unsigned)(a >> (32 - sh)); wm[w0 + 1] |= (unsigned)(b >> (32 - sh)); }
        if (sh != 0 && w0 + 2 <= ESC_WORDS) { wp[w0 + 2] |= (unsigned)(a >> (64 - sh)); wm[w0 + 2] |= (unsigned)(b >> (64 - sh)); }
    }
#pragma unroll
    for (int w = 0; w < ESC_WORDS; ++w) { out[w] = all ? 0xffffffffu : wp[w]; out[ESC_WORDS + w] = all ? 0xffffffffu : wm[w]; }
}

// design of global triangle position g: tri_off[k] <= g < tri_off[k + 1]
__device__ inline int find_design_of(const long long *off, int D, long long g)
{
    int lo = 0, hi = D;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (off[mid] <= g) lo = mid; else hi = mid;
    }
    return lo;
}

// ---- designs without a hierarchy (T <= 64): one warp per triangle t, every other triangle f tested exactly enough.
// The directions from a point of t to a point of f are the cone over the Minkowski difference f - t, the convex hull
// of the 9 vertex differences.  A bin of the cube map is the pyramid {d_m >= 0, s0 d_m <= d_s <= s1 d_m,
// t0 d_m <= d_t <= t1 d_m}; if all 9 differences lie outside one of its 5 planes, so does the whole cone, and the bin
// stays clear.  Otherwise it is marked (conservative: only the bin's own planes are tried as separators).  Which
// side of t sees f is decided as in small_beam_kernel's facet-side masks (R20).  Lane l owns bins l, l + 32, ...
__global__ void __launch_bounds__(128)
escape_mask_small_kernel(const DesignsDev dz, long long sumT, unsigned *esc)
{
    const long long g = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;     // global triangle position
    const int lane = threadIdx.x & 31;
    if (g >= sumT) return;
    const int k = find_design_of(dz.tri_off, dz.D, g);
    const long long tbase = dz.tri_off[k];
    const int T = (int)(dz.tri_off[k + 1] - tbase), t = (int)(g - tbase);
    const float4 *tri = dz.tri + 3 * tbase;
    const float4 q0 = __ldg(tri + 3 * t), q1 = __ldg(tri + 3 * t + 1), q2 = __ldg(tri + 3 * t + 2);
    const float3 a[3] = { make_float3(q0.x, q0.y, q0.z), make_float3(q0.x + q1.x, q0.y + q1.y, q0.z + q1.z),
                          make_float3(q0.x + q2.x, q0.y + q2.y, q0.z + q2.z) };
    float3 n = make_float3(q1.y * q2.z - q1.z * q2.y, q1.z * q2.x - q1.x * q2.z, q1.x * q2.y - q1.y * q2.x);
    const float il = rsqrtf(n.x * n.x + n.y * n.y + n.z * n.z);
    n = make_float3(n.x * il, n.y * il, n.z * il);
    const float4 blo = dz.box[2 * k], bhi = dz.box[2 * k + 1];
    const float eps = 1.0e-6f * (fmaxf(fabsf(blo.x), fabsf(bhi.x)) + fmaxf(fabsf(blo.y), fabsf(bhi.y)) +
                                 fmaxf(fabsf(blo.z), fabsf(bhi.z)));
    constexpr int ROUNDS = (ESC_BINS + 31) / 32;
    unsigned mp[ROUNDS], mm[ROUNDS];                                 // bit r of lane l = bin 32 r + l, front / back side
#pragma unroll
    for (int r = 0; r < ROUNDS; ++r) mp[r] = mm[r] = 0u;
    for (int f = 0; f < T; ++f) {
        if (f == t) continue;
        const float4 p0 = __ldg(tri + 3 * f), p1 = __ldg(tri + 3 * f + 1), p2 = __ldg(tri + 3 * f + 2);
        const float3 b[3] = { make_float3(p0.x, p0.y, p0.z), make_float3(p0.x + p1.x, p0.y + p1.y, p0.z + p1.z),
                              make_float3(p0.x + p2.x, p0.y + p2.y, p0.z + p2.z) };
        const float r0 = n.x * (p0.x - q0.x) + n.y * (p0.y - q0.y) + n.z * (p0.z - q0.z);
        const float d0 = r0, d1 = r0 + n.x * p1.x + n.y * p1.y + n.z * p1.z, d2 = r0 + n.x * p2.x + n.y * p2.y + n.z * p2.z;
        const bool fp = fmaxf(d0, fmaxf(d1, d2)) > eps, fm = fminf(d0, fminf(d1, d2)) < -eps;
        if (!fp && !fm) continue;                                    // coplanar with t: never hit from t
        float3 v[9];
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) v[3 * i + j] = make_float3(b[i].x - a[j].x, b[i].y - a[j].y, b[i].z - a[j].z);
#pragma unroll
        for (int r = 0; r < ROUNDS; ++r) {
            const int bin = 32 * r + lane;
            if (bin >= ESC_BINS) break;
            const int face = bin / (ESC_GRID * ESC_GRID), cell = bin % (ESC_GRID * ESC_GRID);
            const int is = cell % ESC_GRID, it = cell / ESC_GRID;
            const float s0 = -1.0f + 2.0f * is / ESC_GRID, s1 = -1.0f + 2.0f * (is + 1) / ESC_GRID;
            const float t0 = -1.0f + 2.0f * it / ESC_GRID, t1 = -1.0f + 2.0f * (it + 1) / ESC_GRID;
            const float sg = (face & 1) ? -1.0f : 1.0f;
            bool out_m = true, out_s0 = true, out_s1 = true, out_t0 = true, out_t1 = true;
#pragma unroll
            for (int c = 0; c < 9; ++c) {
                // (m, s, t) components in the face's axis order (escape_bins.cuh)
                const float dm = sg * (face < 2 ? v[c].x : face < 4 ? v[c].y : v[c].z);
                const float ds = face < 2 ? v[c].y : v[c].x;
                const float dt = face < 4 ? v[c].z : v[c].y;
                const float tol = 1.0e-5f * (fabsf(dm) + fabsf(ds) + fabsf(dt));   // bin edges and esc_bin's rounding
                out_m = out_m && dm <= tol;
                out_s0 = out_s0 && ds - s0 * dm <= tol;
                out_s1 = out_s1 && s1 * dm - ds <= tol;
                out_t0 = out_t0 && dt - t0 * dm <= tol;
                out_t1 = out_t1 && t1 * dm - dt <= tol;
            }
            if (!(out_m || out_s0 || out_s1 || out_t0 || out_t1)) {
                if (fp) mp[r] |= 1u;
                if (fm) mm[r] |= 1u;
            }
        }
    }
    // word w of a side = bins 32 w .. 32 w + 31 = bit of round w from every lane
    unsigned *out = esc + (size_t)g * (2 * ESC_WORDS);
#pragma unroll
    for (int r = 0; r < ROUNDS; ++r) {
        const unsigned wp = __ballot_sync(FULLW, mp[r] != 0u), wm = __ballot_sync(FULLW, mm[r] != 0u);
        if (lane == 0 && r < ESC_WORDS) { out[r] = wp; out[ESC_WORDS + r] = wm; }
    }
}

} // namespace

cudaError_t srp_launch_escape_masks(const DesignsDev &dz, long long maxT, unsigned *esc, cudaStream_t stream)
{
    if (dz.D > 65535) return cudaErrorInvalidValue;                 // grid.y; the caller builds no masks then
    const dim3 grid((unsigned)((maxT + 127) / 128), (unsigned)dz.D);
    escape_mask_kernel<<<grid, 128, 0, stream>>>(dz, esc);
    return cudaGetLastError();
}

cudaError_t srp_launch_escape_masks_small(const DesignsDev &dz, long long sumT, unsigned *esc, cudaStream_t stream)
{
    escape_mask_small_kernel<<<(unsigned)((sumT + 3) / 4), 128, 0, stream>>>(dz, sumT, esc);
    return cudaGetLastError();
}
