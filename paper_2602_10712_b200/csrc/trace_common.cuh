// trace_common.cuh -- device code shared by the trace kernels of libsrp_b200 (CUDA path only; nothing under
// oracle/ includes this file): Philox4x32-10, emitter set-up and ray generation (O-steps 1-3), the ray-triangle and
// ray-box tests and the BVH2 stack traversal (O-step 4), shading and deposit (O-steps 5-7), the per-tile reduction
// (S7), the 2-D triangle set-up of the beam kernels, and the persistent-kernel launcher.
// numbers the algorithm; the same numbers appear in the comments.
//
// A WARP is the scheduling unit of every trace kernel: it pulls (pair, ray tile) work items from a global atomic
// counter.  Deposits are summed per lane in fp32 (dimensionless, <= a few hundred terms), per warp in fp64 by
// shuffles, and added to a 2^-32 fixed-point int64 accumulator per pair -- integer adds commute, so the result is
// bit-reproducible whatever the scheduling.
#pragma once
#include <cfloat>
#include "srp_internal.cuh"
#include "escape_bins.cuh"

// Debug build (nvcc -DSRP_BOUNDS_CHECK): every write into a fixed-capacity shared-memory list, stack or ray pool
// checks its index and traps with a message.  compute-sanitizer is not available on the target pool.
#ifdef SRP_BOUNDS_CHECK
#include <cstdio>
#define SRP_CHECK(cond, tag) do { if (!(cond)) { printf("SRP_CHECK failed: %s (%s:%d)\n", tag, __FILE__, __LINE__); __trap(); } } while (0)
#else
#define SRP_CHECK(cond, tag) do { } while (0)
#endif

namespace {

constexpr int TRACE_THREADS = 128;
constexpr int TRACE_WARPS = TRACE_THREADS / 32;
#ifndef STACK_SMEM_DEF
#define STACK_SMEM_DEF 20
#endif
constexpr int STACK_SMEM = STACK_SMEM_DEF;   // traversal stack entries per thread kept in shared memory
#ifdef SRP_BVH4
constexpr int STACK_OVF = 128;       // a wide node pushes up to three entries
#else
constexpr int STACK_OVF = 80;
#endif
//        // deeper entries spill to local memory (degenerate trees only)
constexpr unsigned FULL = 0xffffffffu;

enum { MODE_BRUTE_SMEM = 0, MODE_BVH = 1, MODE_BRUTE_GLOBAL = 2 };

__device__ __forceinline__ float3 f3(float x, float y, float z) { return make_float3(x, y, z); }
__device__ __forceinline__ float dot3(float3 a, float3 b) { return fmaf(a.x, b.x, fmaf(a.y, b.y, a.z * b.z)); }
__device__ __forceinline__ float3 cross3(float3 a, float3 b)
{
    return f3(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}

__device__ __forceinline__ void philox4(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                        uint32_t k1, uint32_t &o0, uint32_t &o1, uint32_t &o2, uint32_t &o3)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}
// R4: ((x >> 9) + 0.5) * 2^-23 -- exact in fp32
__device__ __forceinline__ float uniform23(uint32_t x) { return ((float)(x >> 9) + 0.5f) * (1.0f / 8388608.0f); }

// O-step 1: orthonormal basis perpendicular to unit s (Duff et al. 2017)
__device__ __forceinline__ void basis3(float3 s, float3 &u, float3 &v)
{
    const float sign = copysignf(1.0f, s.z);
    const float a = -1.0f / (sign + s.z);
    const float b = s.x * s.y * a;
    u = f3(1.0f + sign * s.x * s.x * a, sign * b, -sign * s.x);
    v = f3(b, sign + s.y * s.y * a, -s.y);
}

struct Emitter {
    float3 s, u, v;
    float u0, v0, du, dv, worg, Ae;
};

// O-steps 1-2: travel direction, basis, rectangle of the projected AABB corners, origin plane.
__device__ inline Emitter make_emitter(const float *sun_dirs, int j, float4 lo, float4 hi)
{
    Emitter e;
    const float wx = sun_dirs[3 * j], wy = sun_dirs[3 * j + 1], wz = sun_dirs[3 * j + 2];
    const float len = sqrtf(wx * wx + wy * wy + wz * wz);
    const bool usable = len > 0.f && len <= FLT_MAX;      // a zero or non-finite direction: A_e = 0, F = 0 (srp.h)
    e.s = usable ? f3(-wx / len, -wy / len, -wz / len) : f3(0.f, 0.f, -1.f);
    basis3(e.s, e.u, e.v);
    float u0 = FLT_MAX, u1 = -FLT_MAX, v0 = FLT_MAX, v1 = -FLT_MAX, w0 = FLT_MAX;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const float3 p = f3((c & 1) ? hi.x : lo.x, (c & 2) ? hi.y : lo.y, (c & 4) ? hi.z : lo.z);
        const float pu = dot3(p, e.u), pv = dot3(p, e.v), pw = dot3(p, e.s);
        u0 = fminf(u0, pu); u1 = fmaxf(u1, pu);
        v0 = fminf(v0, pv); v1 = fmaxf(v1, pv);
        w0 = fminf(w0, pw);
    }
    e.u0 = u0; e.v0 = v0; e.du = u1 - u0; e.dv = v1 - v0;
    e.worg = w0 - 1.0f;
    e.Ae = usable ? e.du * e.dv : 0.f;
    return e;
}

__device__ __forceinline__ uint32_t compact_even_bits(uint32_t x)
{
    x &= 0x55555555u;
    x = (x | (x >> 1)) & 0x33333333u;
    x = (x | (x >> 2)) & 0x0F0F0F0Fu;
    x = (x | (x >> 4)) & 0x00FF00FFu;
    x = (x | (x >> 8)) & 0x0000FFFFu;
    return x;
}

struct RayGen {            // warp-uniform per work item
    uint32_t j, k, key0, key1;
    int sampler;
    float inv_nx, inv_ny;
    float3 xc;             // the design's centre of mass (TORQUE kernels: Eq. 4)
    float inv_arm;         // 1 / torque_arm_scale of the design: arms are summed in units of the design's extent
    bool split;            // TORQUE kernels: the second sum is the direct force (depth-0 deposits), not the torque
};

// O-step 3: ray i of the pair.
__device__ __forceinline__ void make_ray(const Emitter &e, const RayGen &g, uint32_t i, float3 &o)
{
    uint32_t r0, r1, r2, r3;
    philox4(i, g.j, g.k, 0u, g.key0, g.key1, r0, r1, r2, r3);
    float fu, fv;
    if (g.sampler == 0) {
        const float cx = (float)compact_even_bits(i), cy = (float)compact_even_bits(i >> 1);
        fu = (cx + uniform23(r0)) * g.inv_nx;
        fv = (cy + uniform23(r1)) * g.inv_ny;
    } else {
        fu = uniform23(r0); fv = uniform23(r1);
    }
    const float pu = fmaf(fu, e.du, e.u0), pv = fmaf(fv, e.dv, e.v0);
    o = f3(fmaf(pu, e.u.x, fmaf(pv, e.v.x, e.worg * e.s.x)),
           fmaf(pu, e.u.y, fmaf(pv, e.v.y, e.worg * e.s.y)),
           fmaf(pu, e.u.z, fmaf(pv, e.v.z, e.worg * e.s.z)));
}

// 32-byte load (sm_100: LDG.E.256): a 64-byte BVH2 node is two of them instead of four 16-byte loads -- half the
// load instructions and half the L1 tag look-ups of a divergent node fetch.
struct __align__(32) F8 { float4 a, b; };
__device__ __forceinline__ F8 ldg256(const float4 *p)
{
    F8 r;
    asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
        : "=f"(r.a.x), "=f"(r.a.y), "=f"(r.a.z), "=f"(r.a.w), "=f"(r.b.x), "=f"(r.b.y), "=f"(r.b.z), "=f"(r.b.w) : "l"(p));
    return r;
}

// O-step 4, one triangle: Moller-Trumbore on (v0, e1, e2) in the division-free sign-normalised
// form: accept det != 0, u >= 0, v >= 0, u+v <= 1, t > 0; t = T/|det| only for accepted hits.
__device__ __forceinline__ void tri_test(const float4 q0, const float4 q1, const float4 q2, const float3 o,
                                         const float3 d, const int f, float &tbest, int &best)
{
    const float3 e1 = f3(q1.x, q1.y, q1.z), e2 = f3(q2.x, q2.y, q2.z);
    const float3 pv = cross3(d, e2);
    const float det = dot3(e1, pv);
    const float3 tv = f3(o.x - q0.x, o.y - q0.y, o.z - q0.z);
    const float3 qv = cross3(tv, e1);
    const uint32_t sb = __float_as_uint(det) & 0x80000000u;
    const float U = __uint_as_float(__float_as_uint(dot3(tv, pv)) ^ sb);
    const float V = __uint_as_float(__float_as_uint(dot3(d, qv)) ^ sb);
    const float Tn = __uint_as_float(__float_as_uint(dot3(e2, qv)) ^ sb);
    const float adet = fabsf(det);
    if (U >= 0.0f && V >= 0.0f && U + V <= adet && Tn > 0.0f && adet > 0.0f) {
        const float t = Tn / adet;
        if (t < tbest) { tbest = t; best = f; }
    }
}

// All triangles of a design, in index order (ties -> smallest index), source excluded (R10).
template <bool INSTR>
__device__ __forceinline__ void closest_brute(const float4 *__restrict__ tp, const int T, const float3 o,
                                              const float3 d, const int src, float &tbest, int &best,
                                              unsigned &n_tri)
{
    for (int f = 0; f < T; ++f) {
        if (f == src) continue;
        tri_test(tp[3 * f], tp[3 * f + 1], tp[3 * f + 2], o, d, f, tbest, best);
    }
    if (INSTR) n_tri += (unsigned)(T - (src >= 0 ? 1 : 0));
}

__device__ __forceinline__ float safe_rcp(float x)
{
    return 1.0f / (fabsf(x) < 1e-30f ? copysignf(1e-30f, x) : x);
}

// Stack-based BVH2 descent, nearer child first, in "while-while" form: a lane stays in the node
// loop until it lands on a leaf (or runs out of nodes); the warp reconverges after the node loop, so
// the triangle tests of all lanes that hold a leaf run together (in the single-loop form they ran
// with ~4 of 32 lanes active and took a third of the issue slots -- profiles/ round 1).
// Stack: STACK_SMEM entries per thread in shared memory (thread-interleaved, conflict-free), deeper
// levels in a local array.
constexpr int CUR_DONE = 0x7fffffff;
// "while-while" traversal lets a lane walk nodes until it reaches a leaf while the lanes that already hold one
// wait.  Capping a node run (and not unrolling it) bounds that wait: cfg3 bounce rays +9 %, per-ray primaries +13 %.
#ifndef NODE_RUN_CAP_DEF
#define NODE_RUN_CAP_DEF 8
#endif
constexpr int NODE_RUN_CAP = NODE_RUN_CAP_DEF;

#define SRP_POP(cur_)                                                                     \
    do {                                                                                  \
        if (sp == 0) cur_ = CUR_DONE;                                                     \
        else { --sp; cur_ = sp < NSMEM ? s_stack[sp * STRIDE] : ovf[sp - NSMEM]; }        \
    } while (0)

#ifdef SRP_BVH4
// 4-wide node (bvh4.cu): four child boxes against the ray, the hits in order of entry distance: nearest next, the
// others pushed farthest first.  `nodes` is the design's nodes4 base.
#define SRP_TRAV_NODES(dz_, tb_) ((dz_).nodes4 + 8 * (tb_))
#define SRP_CSWAP(i_, j_)                                                                                     \
    do {                                                                                                      \
        const bool sw_ = key[j_] < key[i_];                                                                   \
        const float kf_ = sw_ ? key[j_] : key[i_], kg_ = sw_ ? key[i_] : key[j_];                              \
        const int lf_ = sw_ ? link[j_] : link[i_], lg_ = sw_ ? link[i_] : link[j_];                            \
        key[i_] = kf_; key[j_] = kg_; link[i_] = lf_; link[j_] = lg_;                                          \
    } while (0)
template <int STRIDE, int NSMEM>
__device__ __forceinline__ int bvh_node_step(const float4 *__restrict__ nodes, int cur, int &sp, int *s_stack, int *ovf,
                                             float idx, float idy, float idz, float oxi, float oyi, float ozi, float tbest)
{
    const float4 *p = nodes + 8 * (long long)cur;
    const F8 qa = ldg256(p), qb = ldg256(p + 2), qc = ldg256(p + 4), qd = ldg256(p + 6);
    const float w[24] = { qa.a.x, qa.a.y, qa.a.z, qa.a.w, qa.b.x, qa.b.y, qa.b.z, qa.b.w, qb.a.x, qb.a.y, qb.a.z, qb.a.w,
                          qb.b.x, qb.b.y, qb.b.z, qb.b.w, qc.a.x, qc.a.y, qc.a.z, qc.a.w, qc.b.x, qc.b.y, qc.b.z, qc.b.w };
    int link[4] = { __float_as_int(qd.a.x), __float_as_int(qd.a.y), __float_as_int(qd.a.z), __float_as_int(qd.a.w) };
    float key[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float a0 = fmaf(w[6 * c + 0], idx, -oxi), a1 = fmaf(w[6 * c + 3], idx, -oxi);
        const float b0 = fmaf(w[6 * c + 1], idy, -oyi), b1 = fmaf(w[6 * c + 4], idy, -oyi);
        const float c0 = fmaf(w[6 * c + 2], idz, -ozi), c1 = fmaf(w[6 * c + 5], idz, -ozi);
        const float tmin = fmaxf(fmaxf(fminf(a0, a1), fminf(b0, b1)), fmaxf(fminf(c0, c1), 0.0f));
        const float tmax = fminf(fminf(fmaxf(a0, a1), fmaxf(b0, b1)), fminf(fmaxf(c0, c1), tbest));
        key[c] = tmin <= tmax * 1.0000004f ? tmin : FLT_MAX;
    }
#ifdef SRP_BVH4_NOSORT
    int m = 0;
    float km = key[0];
#pragma unroll
    for (int c = 1; c < 4; ++c)
        if (key[c] < km) { km = key[c]; m = c; }
    int lm = link[0];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        if (c == m) lm = link[c];
        else if (key[c] < FLT_MAX) {
            if (sp < NSMEM) s_stack[sp * STRIDE] = link[c]; else ovf[sp - NSMEM] = link[c];
            ++sp;
        }
    }
    if (km < FLT_MAX) return lm;
#else
    SRP_CSWAP(0, 1); SRP_CSWAP(2, 3); SRP_CSWAP(0, 2); SRP_CSWAP(1, 3); SRP_CSWAP(1, 2);
#pragma unroll
    for (int c = 3; c >= 1; --c)
        if (key[c] < FLT_MAX) {
            SRP_CHECK(sp < NSMEM + STACK_OVF, "traversal stack");
            if (sp < NSMEM) s_stack[sp * STRIDE] = link[c]; else ovf[sp - NSMEM] = link[c];
            ++sp;
        }
    if (key[0] < FLT_MAX) return link[0];
#endif
    SRP_POP(cur);
    return cur;
}
#else
#define SRP_TRAV_NODES(dz_, tb_) ((dz_).nodes + 4 * (tb_))
// STRIDE: distance in ints between consecutive stack entries of one thread (thread-interleaved
// layout); NSMEM: entries kept in shared memory.
// One internal node for one lane: both child boxes against the ray, nearer child next, farther child
// pushed.  Returns the next value of `cur` (node index, leaf link < 0, or CUR_DONE).
template <int STRIDE, int NSMEM>
__device__ __forceinline__ int bvh_node_step(const float4 *__restrict__ nodes, int cur, int &sp, int *s_stack, int *ovf,
                                             float idx, float idy, float idz, float oxi, float oyi, float ozi, float tbest)
{
#ifdef SRP_NO_LD256
    const float4 n0 = __ldg(nodes + 4 * cur), n1 = __ldg(nodes + 4 * cur + 1),
                 n2 = __ldg(nodes + 4 * cur + 2), n3 = __ldg(nodes + 4 * cur + 3);
#else
    const F8 lo_ = ldg256(nodes + 4 * cur), hi_ = ldg256(nodes + 4 * cur + 2);
    const float4 n0 = lo_.a, n1 = lo_.b, n2 = hi_.a, n3 = hi_.b;
#endif
    float a0 = fmaf(n0.x, idx, -oxi), a1 = fmaf(n0.w, idx, -oxi);
    float b0 = fmaf(n0.y, idy, -oyi), b1 = fmaf(n1.x, idy, -oyi);
    float c0 = fmaf(n0.z, idz, -ozi), c1 = fmaf(n1.y, idz, -ozi);
    const float tmin0 = fmaxf(fmaxf(fminf(a0, a1), fminf(b0, b1)), fmaxf(fminf(c0, c1), 0.0f));
    const float tmax0 = fminf(fminf(fmaxf(a0, a1), fmaxf(b0, b1)), fminf(fmaxf(c0, c1), tbest));
    a0 = fmaf(n1.z, idx, -oxi); a1 = fmaf(n2.y, idx, -oxi);
    b0 = fmaf(n1.w, idy, -oyi); b1 = fmaf(n2.z, idy, -oyi);
    c0 = fmaf(n2.x, idz, -ozi); c1 = fmaf(n2.w, idz, -ozi);
    const float tmin1 = fmaxf(fmaxf(fminf(a0, a1), fminf(b0, b1)), fmaxf(fminf(c0, c1), 0.0f));
    const float tmax1 = fminf(fminf(fmaxf(a0, a1), fmaxf(b0, b1)), fminf(fmaxf(c0, c1), tbest));
    const bool h0 = tmin0 <= tmax0 * 1.0000004f, h1 = tmin1 <= tmax1 * 1.0000004f;
    int l0 = __float_as_int(n3.x), l1 = __float_as_int(n3.y);
    if (h0 && h1) {
        if (tmin1 < tmin0) { const int t = l0; l0 = l1; l1 = t; }
        SRP_CHECK(sp < NSMEM + STACK_OVF, "traversal stack");
        if (sp < NSMEM) s_stack[sp * STRIDE] = l1; else ovf[sp - NSMEM] = l1;
        ++sp;
        return l0;
    }
    if (h0) return l0;
    if (h1) return l1;
    SRP_POP(cur);
    return cur;
}

#endif

// One leaf for one lane: its triangles (source excluded, R10), then the next stack entry.
template <int STRIDE, int NSMEM>
__device__ __forceinline__ int bvh_leaf_step(const float4 *__restrict__ tri, int cur, int &sp, int *s_stack, int *ovf,
                                             const float3 o, const float3 d, const int src, float &tbest, int &best,
                                             unsigned &n_tri)
{
    const unsigned u = (unsigned)~cur;
    const int first = (int)(u >> 3), cnt = (int)(u & 7u) + 1;
    for (int f = first; f < first + cnt; ++f) {
        if (f == src) continue;
        tri_test(__ldg(tri + 3 * f), __ldg(tri + 3 * f + 1), __ldg(tri + 3 * f + 2), o, d, f, tbest, best);
    }
    n_tri += (unsigned)cnt;
    SRP_POP(cur);
    return cur;
}

// STRIDE: distance in ints between consecutive stack entries of one thread (thread-interleaved
// layout); NSMEM: entries kept in shared memory.
template <bool INSTR, int STRIDE = TRACE_THREADS, int NSMEM = STACK_SMEM>
__device__ __forceinline__ void closest_bvh(const float4 *__restrict__ nodes, const float4 *__restrict__ tri,
                                            const float3 o, const float3 d, const int src, float &tbest,
                                            int &best, int *s_stack, unsigned &n_box, unsigned &n_tri)
{
    const float idx = safe_rcp(d.x), idy = safe_rcp(d.y), idz = safe_rcp(d.z);
    const float oxi = o.x * idx, oyi = o.y * idy, ozi = o.z * idz;
    int ovf[STACK_OVF];
    int sp = 0;
    int cur = 0;
    unsigned nt = 0;
    while (cur != CUR_DONE) {
        // internal nodes; at most NODE_RUN_CAP steps before the lanes that wait at a leaf get their turn
#pragma unroll 1
        for (int steps = 0; steps < NODE_RUN_CAP && (unsigned)cur < (unsigned)CUR_DONE; ++steps) {
            if (INSTR) n_box += 2;
            cur = bvh_node_step<STRIDE, NSMEM>(nodes, cur, sp, s_stack, ovf, idx, idy, idz, oxi, oyi, ozi, tbest);
        }
        if (cur < 0)                                                 // leaf: all lanes that hold one, together
            cur = bvh_leaf_step<STRIDE, NSMEM>(tri, cur, sp, s_stack, ovf, o, d, src, tbest, best, nt);
    }
    if (INSTR) n_tri += nt;
}

struct LaneCounters {
    unsigned launched, pmiss, absorbed, escaped, capped, segments, n_box, n_tri;
    unsigned mesc;          // bounce rays resolved by the escape masks (also in escaped and segments)
};
struct BeamCounters {       // rays resolved per beam level (lane-distributed counts); instrumented: beam work
    unsigned tile_miss, block_miss, group_miss, fallback;
    unsigned beam_box, tri2d, setups, rect;     // beam-box tests, 2-D ray-triangle tests, triangle set-ups, rectangle-triangle tests
};

// O-steps 5-7 at a hit: deposit, lobe selection, continuation.
// Returns SHADE_CONTINUE if the photon goes on (o, d, src, depth updated), else how it ended.
// R23: one direction of the Phong lobe cos^ns about refl, for a facet with facing normal nf and first-edge tangent
// tu; directions below the facet's horizon are redrawn (attempt a >= 1: words 1, 2 of Philox(i, j, k, cword | a << 8)),
// after 8 rejections the photon takes refl.  Not inlined: facets without shininess never come here.
__device__ __noinline__ float3 phong_direction(const float ns, const float3 nf, const float3 refl, const float3 tu,
                                               float z1, float z2, const uint32_t i, const uint32_t j, const uint32_t k,
                                               const uint32_t cword, const uint32_t key0, const uint32_t key1)
{
    const float3 tv = cross3(nf, tu), kx = cross3(nf, refl);
    const float icc = 1.0f / (1.0f + dot3(nf, refl));
    for (int a = 0; a < 8; ++a) {
        if (a > 0) {
            uint32_t w0, w1, w2, w3;
            philox4(i, j, k, cword | ((uint32_t)a << 8), key0, key1, w0, w1, w2, w3);
            z1 = uniform23(w1); z2 = uniform23(w2);
        }
        const float ct = powf(z2, 1.0f / (ns + 1.0f)), st = sqrtf(fmaxf(0.0f, 1.0f - ct * ct));
        float sn, cs;
        sincospif(2.0f * z1, &sn, &cs);
        const float lx = st * cs, ly = st * sn;
        const float3 L = f3(fmaf(lx, tu.x, fmaf(ly, tv.x, ct * nf.x)), fmaf(lx, tu.y, fmaf(ly, tv.y, ct * nf.y)),
                            fmaf(lx, tu.z, fmaf(ly, tv.z, ct * nf.z)));
        const float3 kL = cross3(kx, L), kkL = cross3(kx, kL);
        const float3 c = f3(L.x + kL.x + kkL.x * icc, L.y + kL.y + kkL.y * icc, L.z + kL.z + kkL.z * icc);
        if (dot3(c, nf) > 0.0f) return c;
    }
    return refl;
}

enum { SHADE_CONTINUE = 0, SHADE_ABSORBED = 1, SHADE_CAPPED = 2, SHADE_ESCAPES = 3 };   // ESCAPES: goes on, but the
// escape mask of the facet (escape_mask.cu) shows that its next segment cannot hit anything
// CFLAG is OR-ed into the Philox counter word that holds the depth: 0 for sun photons, 0x80000000 for photons of
// thermal emitters (R22), so the two families draw from disjoint streams.
template <bool TORQUE, uint32_t CFLAG = 0u, bool GLOSSY = false, int DEPOSIT = -1>
__device__ __forceinline__ int shade(const float4 q0, const float4 q1, const float4 q2, const float t,
                                      const int f, const RayGen &g, const uint32_t i, const int B,
                                      const int deposit_, float3 &o, float3 &d, int &src, int &depth,
                                      float3 &acc, float3 &acc_t, const unsigned *esc = nullptr, long long gidx = 0,
                                      const float *shin = nullptr)
{
    // DEPOSIT 0 / 1: the deposit rule is fixed at compile time (the sun-photon kernels: +9 % on cfg2 against the
    // run-time test); -1: taken from the argument
    const int deposit = DEPOSIT >= 0 ? DEPOSIT : deposit_;
    (void)q0;
    // every deposit of this hit is made at the hit point x; Eq. 4: torque += (x - x_COM) x deposit
    const float3 x = f3(fmaf(t, d.x, o.x), fmaf(t, d.y, o.y), fmaf(t, d.z, o.z));
    auto put = [&](const float3 dd) {
        acc.x += dd.x; acc.y += dd.y; acc.z += dd.z;
        if (TORQUE) {
            if (g.split) {                                        // direct part: what sun light deposits at its first hit
                if (depth == 0) { acc_t.x += dd.x; acc_t.y += dd.y; acc_t.z += dd.z; }
            } else {
                const float3 r = f3((x.x - g.xc.x) * g.inv_arm, (x.y - g.xc.y) * g.inv_arm, (x.z - g.xc.z) * g.inv_arm);
                const float3 m = cross3(r, dd);
                acc_t.x += m.x; acc_t.y += m.y; acc_t.z += m.z;
            }
        }
    };
    const float al = q0.w, rs = q1.w, rd = q2.w;
    float3 n = cross3(f3(q1.x, q1.y, q1.z), f3(q2.x, q2.y, q2.z));
    const float inv_len = 1.0f / sqrtf(dot3(n, n));
    n = f3(n.x * inv_len, n.y * inv_len, n.z * inv_len);
    const float nd = dot3(n, d);
    const float3 nf = nd > 0.0f ? f3(-n.x, -n.y, -n.z) : n;      // facets are two-sided (R6)
    const float cost = fabsf(nd);
    const float3 refl = f3(fmaf(2.0f * cost, nf.x, d.x), fmaf(2.0f * cost, nf.y, d.y), fmaf(2.0f * cost, nf.z, d.z));
    // R23: shininess >= 0 = Phong lobe about refl; none, or < 0 = ideal mirror
    // (GLOSSY is a build of its own, so that the ideal-mirror kernels carry none of this)
    const float ns = (GLOSSY && shin) ? __ldg(shin + gidx) : -1.0f;
    const bool glossy = GLOSSY && ns >= 0.0f;
    if (deposit == 0) {                                           // expected-value deposit
        const float rsm = glossy ? 0.0f : rs;                     // a glossy specular part is deposited when drawn
        const float a = al + rsm + rd, c = (2.0f / 3.0f) * rd;
        put(f3(a * d.x - rsm * refl.x - c * nf.x, a * d.y - rsm * refl.y - c * nf.y, a * d.z - rsm * refl.z - c * nf.z));
    }
    uint32_t y0, y1, y2, y3;
    philox4(i, g.j, g.k, (uint32_t)(depth + 1) | CFLAG, g.key0, g.key1, y0, y1, y2, y3);
    const float z0 = uniform23(y0);
    float3 dn;
    if (z0 < al) {                                                // absorbed
        if (deposit == 1) put(d);
        return SHADE_ABSORBED;
    } else if (z0 < al + rs) {                                    // ideal mirror (R3), or the Phong lobe about it
        dn = refl;
        if (glossy) {
            const float ie = rsqrtf(q1.x * q1.x + q1.y * q1.y + q1.z * q1.z);
            dn = phong_direction(ns, nf, refl, f3(q1.x * ie, q1.y * ie, q1.z * ie), uniform23(y1), uniform23(y2), i, g.j, g.k,
                                 (uint32_t)(depth + 1) | CFLAG, g.key0, g.key1);
            if (deposit == 0) put(f3(d.x - dn.x, d.y - dn.y, d.z - dn.z));
        }
    } else {                                                      // Lambertian: cosine-weighted about nf
        const float z1 = uniform23(y1), z2 = uniform23(y2);
        float sn, cs;
        sincospif(2.0f * z1, &sn, &cs);
        const float rho = sqrtf(z2), lz = sqrtf(1.0f - z2);
        // tangent frame (R18): first edge of the facet and nf x edge (no discontinuity in nf)
        const float ie = rsqrtf(q1.x * q1.x + q1.y * q1.y + q1.z * q1.z);
        const float3 tu = f3(q1.x * ie, q1.y * ie, q1.z * ie);
        const float3 tv = cross3(nf, tu);
        const float lx = rho * cs, ly = rho * sn;
        dn = f3(fmaf(lx, tu.x, fmaf(ly, tv.x, lz * nf.x)), fmaf(lx, tu.y, fmaf(ly, tv.y, lz * nf.y)),
                fmaf(lx, tu.z, fmaf(ly, tv.z, lz * nf.z)));
    }
    if (deposit == 1) put(f3(d.x - dn.x, d.y - dn.y, d.z - dn.z));
    if (depth == B) return SHADE_CAPPED;                         // R5: B reflections followed
    // the photon leaves on the side it came from (nf): side 0 = the side of e1 x e2
    if (esc && esc_escapes(esc, gidx, nd > 0.0f ? 1 : 0, dn.x, dn.y, dn.z)) return SHADE_ESCAPES;
    // Hit point in fp32 is off the facet's plane by a few ulp of |x| + t (micrometres here).  An origin
    // that ends up BELOW the plane lets the outgoing ray hit a coplanar or convex neighbour from
    // behind -- a path the exact arithmetic of the definition never takes.  Lift the origin along the
    // facing normal by more than that error (R10: "exclude the source triangle, t > 0, no
    // epsilon" is the definition; this is the fp32 guard that keeps the CUDA path on it).
    const float lift = 1.0e-6f * (fabsf(x.x) + fabsf(x.y) + fabsf(x.z) + t);
    o = f3(fmaf(lift, nf.x, x.x), fmaf(lift, nf.y, x.y), fmaf(lift, nf.z, x.z));
    d = dn; src = f; depth += 1;
    return SHADE_CONTINUE;
}

// Pair p -> (design k, direction j).  Entries of a caller's pair list are clamped into range: a bad list gives
// meaningless forces, never an out-of-bounds read.
__device__ __forceinline__ void clamp_pair(const TraceArgs &a, int &k, int &j)
{
    k = min(max(k, 0), a.dz.D - 1); j = min(max(j, 0), a.S - 1);
}
// same for a pair index known to fit 32 bits (rays of the ray queue)
__device__ __forceinline__ void pair_of32(const TraceArgs &a, uint32_t p, int &k, int &j)
{
    if (a.pairs) { k = a.pairs[2 * (size_t)p]; j = a.pairs[2 * (size_t)p + 1]; clamp_pair(a, k, j); }
    else { const uint32_t kk = p / (uint32_t)a.S; k = (int)kk; j = (int)(p - kk * (uint32_t)a.S); }
}
__device__ __forceinline__ void pair_of(const TraceArgs &a, long long p, int &k, int &j)
{
    if (a.pairs) { k = a.pairs[2 * p]; j = a.pairs[2 * p + 1]; clamp_pair(a, k, j); }
    else { k = (int)(p / a.S); j = (int)(p - (long long)k * a.S); }
}

// Torque arms |x - x_COM| are summed in units of this length (an upper bound of the arm over the design's box), so
// that the fixed-point torque sums have the range of the force sums whatever the mesh's units; finalize_kernel
// multiplies it back.
__device__ __forceinline__ float torque_arm_scale(const float4 lo, const float4 hi, const float3 xc)
{
    const float ax = fmaxf(fabsf(lo.x - xc.x), fabsf(hi.x - xc.x)), ay = fmaxf(fabsf(lo.y - xc.y), fabsf(hi.y - xc.y)),
                az = fmaxf(fabsf(lo.z - xc.z), fabsf(hi.z - xc.z));
    return fmaxf(sqrtf(ax * ax + ay * ay + az * az), 1e-30f);
}

template <bool TORQUE>
__device__ __forceinline__ void set_torque(RayGen &g, const TraceArgs &a, int k)
{
    g.xc = (TORQUE && a.xcom) ? f3(a.xcom[3 * k], a.xcom[3 * k + 1], a.xcom[3 * k + 2]) : f3(0.f, 0.f, 0.f);
    g.split = TORQUE && a.torque == 2;
    g.inv_arm = (TORQUE && a.torque == 1) ? 1.0f / torque_arm_scale(a.dz.box[2 * k], a.dz.box[2 * k + 1], g.xc) : 1.0f;
}

// S7 for one work item: per-lane fp32 sums -> fp64 warp shuffle tree -> one fixed-point atomic per component.
// accum holds acc_stride (3, or 6 with torque) int64 per pair.
template <bool TORQUE>
__device__ __forceinline__ void flush_tile_acc(const TraceArgs &a, long long p, const float3 acc, const float3 acc_t, int lane)
{
    const double s[6] = { acc.x, acc.y, acc.z, acc_t.x, acc_t.y, acc_t.z };
#pragma unroll
    for (int c = 0; c < (TORQUE ? 6 : 3); ++c) {
        double v = s[c];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(FULL, v, off);
        if (lane == 0) {
            unsigned long long *dst = (unsigned long long *)(a.accum + a.acc_stride * p);
            atomicAdd(dst + c, (unsigned long long)__double2ll_rn(v * a.acc_scale));
        }
    }
}

// counters: warp sums, one global atomic each
template <bool INSTR>
__device__ __forceinline__ void flush_counters(const TraceArgs &a, const LaneCounters &cn, const unsigned *hist, int lane)
{
    unsigned long long *st = (unsigned long long *)a.stats;
    const unsigned vals[8] = { cn.launched, cn.pmiss, cn.absorbed, cn.escaped, cn.capped, cn.segments, cn.n_box, cn.n_tri };
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        if (!INSTR && c >= 6) break;
        unsigned long long v = vals[c];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(FULL, v, off);
        if (lane == 0 && v) atomicAdd(st + (c < 6 ? c : 22 + (c - 6)), v);
    }
    {
        unsigned long long v = cn.mesc;
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(FULL, v, off);
        if (lane == 0 && v) atomicAdd(st + 32, v);
    }
    __syncwarp();
    if (lane < 16 && hist[lane]) atomicAdd(st + 6 + lane, (unsigned long long)hist[lane]);
}


// ---- ray queue (beam kernel -> bounce kernel), DESIGN.md "Data layout" ----
// A ray is 9 words: origin, direction, ray index i, pair index p, src | depth << 27 (src = SRC_NONE for a primary),
// plus the 64-bit path signature in the instrumented build; field-major, so that the appends of a warp and the
// fetches of the bounce kernel coalesce.  Written with st.cg / read with ld.cg: the data crosses kernels through L2.
constexpr uint32_t SRC_NONE = 0x07ffffffu;
constexpr uint32_t RQ_DEAD = 0xffffffffu;        // src | depth word of a reserved slot that holds no ray (depth 31 never occurs)
constexpr uint32_t RQ_CHUNK = 256u;              // slots a beam warp reserves at a time

__device__ __forceinline__ void rq_mark_dead(const TraceArgs &a, uint32_t pos) { __stcg(a.rq + 8 * (size_t)a.rq_cap + pos, RQ_DEAD); }

template <bool INSTR>
__device__ __forceinline__ void rq_store(const TraceArgs &a, uint32_t pos, const float3 &o, const float3 &d, uint32_t i,
                                         uint32_t p, uint32_t sd, unsigned long long sig)
{
    unsigned *q = a.rq + pos;
    const size_t c = a.rq_cap;
    __stcg(q, __float_as_uint(o.x)); __stcg(q + c, __float_as_uint(o.y)); __stcg(q + 2 * c, __float_as_uint(o.z));
    __stcg(q + 3 * c, __float_as_uint(d.x)); __stcg(q + 4 * c, __float_as_uint(d.y)); __stcg(q + 5 * c, __float_as_uint(d.z));
    __stcg(q + 6 * c, i); __stcg(q + 7 * c, p); __stcg(q + 8 * c, sd);
    if (INSTR) { __stcg(q + 9 * c, (uint32_t)sig); __stcg(q + 10 * c, (uint32_t)(sig >> 32)); }
}

template <bool INSTR>
__device__ __forceinline__ void rq_load(const TraceArgs &a, uint32_t pos, float3 &o, float3 &d, uint32_t &i, uint32_t &p,
                                        uint32_t &sd, unsigned long long &sig)
{
    const unsigned *q = a.rq + pos;
    const size_t c = a.rq_cap;
    o = f3(__uint_as_float(__ldcg(q)), __uint_as_float(__ldcg(q + c)), __uint_as_float(__ldcg(q + 2 * c)));
    d = f3(__uint_as_float(__ldcg(q + 3 * c)), __uint_as_float(__ldcg(q + 4 * c)), __uint_as_float(__ldcg(q + 5 * c)));
    i = __ldcg(q + 6 * c); p = __ldcg(q + 7 * c); sd = __ldcg(q + 8 * c);
    if (INSTR) sig = (unsigned long long)__ldcg(q + 9 * c) | ((unsigned long long)__ldcg(q + 10 * c) << 32);
}

// Per-warp shared-memory queue of bounce rays (bvh_trace_kernel, small_beam_kernel).
constexpr int QCAP = 64;
struct WarpQueue {
    float ox[QCAP], oy[QCAP], oz[QCAP], dx[QCAP], dy[QCAP], dz[QCAP];
    uint32_t i[QCAP];
    int src_depth[QCAP];                 // (depth << 27) | src
};

__device__ __forceinline__ void flush_beam_counters(const TraceArgs &a, const BeamCounters &bc, int lane)
{
    unsigned long long *st = (unsigned long long *)a.stats;
    const unsigned vals[8] = { bc.tile_miss, bc.block_miss, bc.group_miss, bc.fallback, bc.beam_box, bc.tri2d, bc.setups, bc.rect };
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        unsigned long long v = vals[c];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(FULL, v, off);
        if (lane == 0 && v) atomicAdd(st + 24 + c, v);
    }
}


// Candidate set-up: triangle -> sign-normalised edge functions E_i(x) = A_i x_u + B_i x_v + C_i
// (inside <=> all >= 0) and the depth plane t(x) = Wu x_u + Wv x_v + Wc, in the sub-block's local
// emitter frame (origin at the sub-block's corner, t measured from the ray-origin plane).
// bbox (optional): the projected triangle's extent (umin, umax, vmin, vmax) in the same frame; empty (min > max) for a
// triangle that is never hit.
__device__ __forceinline__ void beam_setup(const float4 q0, const float4 q1, const float4 q2, const Emitter &em,
                                           float offu, float offv, float4 *eq, float4 *bbox = nullptr)
{
    const float3 a = f3(q0.x, q0.y, q0.z);
    const float3 b = f3(q0.x + q1.x, q0.y + q1.y, q0.z + q1.z);
    const float3 c = f3(q0.x + q2.x, q0.y + q2.y, q0.z + q2.z);
    const float au = dot3(a, em.u) - offu, av = dot3(a, em.v) - offv, aw = dot3(a, em.s) - em.worg;
    const float bu = dot3(b, em.u) - offu, bv = dot3(b, em.v) - offv, bw = dot3(b, em.s) - em.worg;
    const float cu = dot3(c, em.u) - offu, cv = dot3(c, em.v) - offv, cw = dot3(c, em.s) - em.worg;
    // E_pq(x) = (q_u - p_u)(x_v - p_v) - (q_v - p_v)(x_u - p_u)
    float A0 = -(bv - av), B0 = bu - au, C0 = -fmaf(A0, au, B0 * av);       // edge a -> b
    float A1 = -(cv - bv), B1 = cu - bu, C1 = -fmaf(A1, bu, B1 * bv);       // edge b -> c
    float A2 = -(av - cv), B2 = au - cu, C2 = -fmaf(A2, cu, B2 * cv);       // edge c -> a
    const float area2 = fmaf(A0, cu, fmaf(B0, cv, C0));                     // E_ab(c)
    if (area2 == 0.0f || !(fabsf(area2) < FLT_MAX)) {                       // edge-on or degenerate: never hit
        eq[0] = make_float4(0.f, 0.f, -1.f, 0.f); eq[1] = eq[0]; eq[2] = eq[0];
        if (bbox) *bbox = make_float4(1.f, 0.f, 1.f, 0.f);
        return;
    }
    if (bbox) *bbox = make_float4(fminf(au, fminf(bu, cu)), fmaxf(au, fmaxf(bu, cu)), fminf(av, fminf(bv, cv)), fmaxf(av, fmaxf(bv, cv)));
    if (area2 < 0.0f) { A0 = -A0; B0 = -B0; C0 = -C0; A1 = -A1; B1 = -B1; C1 = -C1; A2 = -A2; B2 = -B2; C2 = -C2; }
    const float ia = 1.0f / area2;
    const float Wu = ((cv - av) * (bw - aw) - (bv - av) * (cw - aw)) * ia;
    const float Wv = ((bu - au) * (cw - aw) - (cu - au) * (bw - aw)) * ia;
    const float Wc = aw - fmaf(Wu, au, Wv * av);
    eq[0] = make_float4(A0, B0, C0, Wu);
    eq[1] = make_float4(A1, B1, C1, Wv);
    eq[2] = make_float4(A2, B2, C2, Wc);
}


// Shared-memory carve-out: no more than the resident blocks of the kernel use; the rest of the SM's 256 KB is L1
// for nodes and triangles (bounce kernel: 92 KB instead of 28 KB, cfg3 -3.7 %).
#ifndef SRP_NO_CARVE
template <typename K>
cudaError_t prefer_l1(K kernel, int per_sm, size_t dyn_smem)
{
    cudaFuncAttributes fa;
    const cudaError_t e = cudaFuncGetAttributes(&fa, kernel);
    if (e != cudaSuccess) return e;
    const size_t need = (size_t)per_sm * (fa.sharedSizeBytes + dyn_smem + 1024);
    int pct = (int)((need * 100 + 228 * 1024 - 1) / (228 * 1024));
    if (pct > 100) pct = 100;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, pct);
}
#else
template <typename K> cudaError_t prefer_l1(K, int, size_t) { return cudaSuccess; }
#endif

// Launches a persistent trace kernel: as many blocks as fit the machine once, or fewer if there is less work.
template <typename K>
cudaError_t launch_persistent(K kernel, const TraceArgs &a, int num_sms, cudaStream_t stream, size_t dyn_smem = 0)
{
    int per_sm = 0;
    cudaError_t e = cudaSuccess;
    if (dyn_smem > 0) e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_smem);
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, TRACE_THREADS, dyn_smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    e = prefer_l1(kernel, per_sm, dyn_smem);
    if (e != cudaSuccess) return e;
    const unsigned long long total_tiles = a.tile_end - a.tile_begin;
    unsigned long long blocks = (unsigned long long)num_sms * per_sm;       // persistent: fill the machine once
    const unsigned long long needed = (total_tiles + TRACE_WARPS - 1) / TRACE_WARPS;
    if (blocks > needed) blocks = needed;
    if (blocks < 1) blocks = 1;
    kernel<<<(unsigned)blocks, TRACE_THREADS, dyn_smem, stream>>>(a);
    return cudaGetLastError();
}

template <typename K>
int blocks_per_sm(K kernel, size_t dyn_smem = 0)
{
    int per_sm = 0;
    if (dyn_smem > 0) cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_smem);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, TRACE_THREADS, dyn_smem);
    return per_sm;
}

// Builds of each trace kernel: plain, instrumented (test counters, path signatures), and with torque
// accumulation -- each also with glossy specular lobes (R23), used when the designs carry
// shininess, and each of those for the expected-value and for the analog deposit rule.  Instrumented torque runs are refused by the caller (srp_api.cu).
#define SRP_LAUNCH_A(K_, I_, T_, G_, ...)                                                                 \
    (a.deposit ? launch_persistent(K_<__VA_ARGS__ I_, T_, G_, true>, a, num_sms, stream, dyn_smem)        \
               : launch_persistent(K_<__VA_ARGS__ I_, T_, G_, false>, a, num_sms, stream, dyn_smem))
#define SRP_LAUNCH_G(K_, I_, T_, ...)                                                                     \
    (a.dz.shin ? SRP_LAUNCH_A(K_, I_, T_, true, __VA_ARGS__) : SRP_LAUNCH_A(K_, I_, T_, false, __VA_ARGS__))
#define SRP_LAUNCH3(K_, ...)                                                                              \
    (instrumented ? SRP_LAUNCH_G(K_, true, false, __VA_ARGS__)                                            \
                  : a.torque ? SRP_LAUNCH_G(K_, false, true, __VA_ARGS__)                                 \
                             : SRP_LAUNCH_G(K_, false, false, __VA_ARGS__))

} // namespace
