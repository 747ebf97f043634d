// trace_sample.cu -- sample_design_kernel: the paper's own workload shape ("not ... for a specific light
// direction and a specific design parameter vector in one thread, but for many of these in a batch"; "each
// ray effectively intersects a different world ... each of these rays, for each bounce, is tested against all
// triangles in parallel"; "100 k light directions and/or designs x 1000 samples, ~1 k faces").
// Every record m has its own design theta_m AND its own light direction omega_m, and only ~10^3 photons: a hierarchy
// would never be repaid, so -- as in the paper -- there is none.  One thread block per record: the record's packed
// triangles (generated just before by mesh_gen.cu for this chunk of records) are staged in shared memory once --
// rotated into the record's emitter frame (u, v, s), so that a primary ray is (p_u, p_v, w_org) + t (0, 0, 1) and its
// Moller-Trumbore test collapses to two 2-D edge functions (R19: the same inequalities; 16 instead of 44 flop), the
// depth being computed only for a ray inside the triangle -- the block's warps trace the record's photons against
// ALL of them (S3-S6, operands broadcast from shared memory, lanes refilled as photons end; bounce rays take the
// general test in the same frame), and the block reduces the deposits in a fixed order and rotates them back (S7).
#include "trace_common.cuh"

namespace {

constexpr int SAMPLE_THREADS = 512;
constexpr int SAMPLE_WARPS = SAMPLE_THREADS / 32;
// Primaries of the stratified sampler sit one per cell of the emitter grid, so the closest primary hits of a record
// are found triangle by triangle: a triangle is tested against the rays of the cells its bounding rectangle touches
// (a few) instead of every ray against every triangle -- the same test on the same operands, ~100 x fewer of them.
constexpr int SAMPLE_CLUSTER = 32;                    // triangles per cluster box (bounce rays)
constexpr int RASTER_MIN_TRIS = 1;                    // (a threshold below which all triangles would be tested per ray: none)
constexpr int RASTER_MAX_RAYS = 8192;                 // 16 bytes of shared memory per ray, if they fit beside the triangles
constexpr int RASTER_BIG = 32, RASTER_BIGCAP = 128;   // a triangle over more cells goes to a warp (the first 128 of them)

// O-step 4 for a primary in the emitter frame: origin (pu, pv, worg), direction (0, 0, 1), all triangles.
__device__ __forceinline__ void closest_primary(const float4 *__restrict__ tp, const int T, const float pu, const float pv,
                                                const float worg, float &tbest, int &best)
{
#pragma unroll 4
    for (int f = 0; f < T; ++f) {
        const float4 q0 = tp[3 * f], q1 = tp[3 * f + 1], q2 = tp[3 * f + 2];
        // d x e2 = (-e2.y, e2.x, 0); det = e1 . (d x e2); U = tv . (d x e2); V = d . (tv x e1) = (tv x e1).z
        const float det = fmaf(q1.y, q2.x, -q1.x * q2.y);
        const float tx = pu - q0.x, ty = pv - q0.y;
        const uint32_t sb = __float_as_uint(det) & 0x80000000u;
        const float U = __uint_as_float(__float_as_uint(fmaf(ty, q2.x, -tx * q2.y)) ^ sb);
        const float V = __uint_as_float(__float_as_uint(fmaf(tx, q1.y, -ty * q1.x)) ^ sb);
        const float adet = fabsf(det);
        if (U >= 0.0f && V >= 0.0f && U + V <= adet && adet > 0.0f) {
            const float tz = worg - q0.z;
            const float3 qv = f3(fmaf(ty, q1.z, -tz * q1.y), fmaf(tz, q1.x, -tx * q1.z), fmaf(tx, q1.y, -ty * q1.x));
            const float Tn = __uint_as_float(__float_as_uint(fmaf(q2.x, qv.x, fmaf(q2.y, qv.y, q2.z * qv.z))) ^ sb);
            if (Tn > 0.0f) {
                const float t = Tn / adet;
                if (t < tbest) { tbest = t; best = f; }
            }
        }
    }
}

// The same test for ONE triangle and the primary of ONE cell of the emitter grid (rasterised primaries, below): the
// hit goes into the cell's key -- depth in the high word, triangle in the low word, so that a 64-bit minimum keeps the
// smallest t and, among equal t, the smallest index (the definition's tie rule).
__device__ __forceinline__ void raster_test(const float4 q0, const float4 q1, const float4 q2, const int f, const float2 p,
                                            const float worg, unsigned long long *key)
{
    const float det = fmaf(q1.y, q2.x, -q1.x * q2.y);
    const float tx = p.x - q0.x, ty = p.y - q0.y;
    const uint32_t sb = __float_as_uint(det) & 0x80000000u;
    const float U = __uint_as_float(__float_as_uint(fmaf(ty, q2.x, -tx * q2.y)) ^ sb);
    const float V = __uint_as_float(__float_as_uint(fmaf(tx, q1.y, -ty * q1.x)) ^ sb);
    const float adet = fabsf(det);
    if (U >= 0.0f && V >= 0.0f && U + V <= adet && adet > 0.0f) {
        const float tz = worg - q0.z;
        const float3 qv = f3(fmaf(ty, q1.z, -tz * q1.y), fmaf(tz, q1.x, -tx * q1.z), fmaf(tx, q1.y, -ty * q1.x));
        const float Tn = __uint_as_float(__float_as_uint(fmaf(q2.x, qv.x, fmaf(q2.y, qv.y, q2.z * qv.z))) ^ sb);
        if (Tn > 0.0f) {
            const float t = Tn / adet;
            atomicMin(key, ((unsigned long long)__float_as_uint(t) << 32) | (unsigned long long)(unsigned)f);
        }
    }
}

__device__ __forceinline__ uint32_t spread_even_bits(uint32_t x)     // inverse of compact_even_bits, 16 bits
{
    x &= 0x0000FFFFu;
    x = (x | (x << 8)) & 0x00FF00FFu;
    x = (x | (x << 4)) & 0x0F0F0F0Fu;
    x = (x | (x << 2)) & 0x33333333u;
    x = (x | (x << 1)) & 0x55555555u;
    return x;
}

// The cells of the nx x ny emitter grid that a triangle's bounding rectangle touches (widened by `marg`, the bound of
// the fp32 projection error: a ray outside them fails the test above).  false: none.
__device__ __forceinline__ bool raster_cells(const float4 q0, const float4 q1, const float4 q2, const Emitter &em, const float sx,
                                             const float sy, const float marg, const int nx, const int ny, int &cx0, int &cx1, int &cy0, int &cy1)
{
    const float ua = q0.x, ub = q0.x + q1.x, uc = q0.x + q2.x, va = q0.y, vb = q0.y + q1.y, vc = q0.y + q2.y;
    const float x0 = floorf((fminf(ua, fminf(ub, uc)) - em.u0 - marg) * sx), x1 = floorf((fmaxf(ua, fmaxf(ub, uc)) - em.u0 + marg) * sx);
    const float y0 = floorf((fminf(va, fminf(vb, vc)) - em.v0 - marg) * sy), y1 = floorf((fmaxf(va, fmaxf(vb, vc)) - em.v0 + marg) * sy);
    if (!(x1 >= 0.f && y1 >= 0.f && x0 <= (float)(nx - 1) && y0 <= (float)(ny - 1))) return false;      // also NaN
    cx0 = (int)fmaxf(x0, 0.f); cx1 = (int)fminf(x1, (float)(nx - 1)); cy0 = (int)fmaxf(y0, 0.f); cy1 = (int)fminf(y1, (float)(ny - 1));
    return true;
}

// O-step 4 for the bounce rays of a pass.  n <= 32 rays wait in the warp's queue; with fewer than 17 the lanes are
// shared out: g = 32 / n' lanes per ray (n' = n rounded up to a power of two).  The triangles sit in clusters of 32
// consecutive ones (neighbours on their patch) behind a box each.  The lanes of a ray test its boxes, every g-th each;
// for every box that a ray meets the WHOLE warp then tests the cluster's 32 triangles against that ray, a lane per
// triangle, and reduces to the closest (smallest t, ties to the smallest index as in the definition) -- so both
// steps run with full warps however few photons the deep bounces of a record with ~10^3 photons have left.
__device__ __forceinline__ void closest_shared(const float4 *__restrict__ tp, const float4 *__restrict__ cl, const int T, const bool has_ray,
                                               const float3 o, const float3 d, const int src, const int g, const int sub, float &tbest,
                                               int &best, unsigned &n_tri, unsigned &n_box)
{
    const int lane = threadIdx.x & 31;
    const float idx = safe_rcp(d.x), idy = safe_rcp(d.y), idz = safe_rcp(d.z);
    const float oxi = o.x * idx, oyi = o.y * idy, ozi = o.z * idz;
    const int ncl = (T + SAMPLE_CLUSTER - 1) / SAMPLE_CLUSTER;
    const int iters = (ncl + g - 1) / g;                                   // warp-uniform
    for (int k = 0; k < iters; ++k) {
        const int c = sub + k * g;
        bool hit = false;
        if (has_ray && c < ncl) {
            const float4 lo = cl[2 * c], hi = cl[2 * c + 1];
            const float a0 = fmaf(lo.x, idx, -oxi), a1 = fmaf(hi.x, idx, -oxi);
            const float b0 = fmaf(lo.y, idy, -oyi), b1 = fmaf(hi.y, idy, -oyi);
            const float c0 = fmaf(lo.z, idz, -ozi), c1 = fmaf(hi.z, idz, -ozi);
            const float tmin = fmaxf(fmaxf(fminf(a0, a1), fminf(b0, b1)), fmaxf(fminf(c0, c1), 0.0f));
            const float tmax = fminf(fminf(fmaxf(a0, a1), fmaxf(b0, b1)), fminf(fmaxf(c0, c1), tbest));
            ++n_box;
            hit = tmin <= tmax * 1.0000004f;
        }
        unsigned m = __ballot_sync(FULL, hit);
        while (m != 0u) {                                                  // one (ray, cluster) pair at a time, all lanes
            const int L = __ffs(m) - 1;
            m &= m - 1u;
            const float3 ro = f3(__shfl_sync(FULL, o.x, L), __shfl_sync(FULL, o.y, L), __shfl_sync(FULL, o.z, L));
            const float3 rd = f3(__shfl_sync(FULL, d.x, L), __shfl_sync(FULL, d.y, L), __shfl_sync(FULL, d.z, L));
            const int rsrc = __shfl_sync(FULL, src, L);
            const int f = __shfl_sync(FULL, c, L) * SAMPLE_CLUSTER + lane;
            float tt = FLT_MAX;
            int bb = -1;
            if (f < T && f != rsrc) {
                tri_test(tp[3 * f], tp[3 * f + 1], tp[3 * f + 2], ro, rd, f, tt, bb);
                ++n_tri;
            }
            // closest of the 32: t > 0, so its bits order like the value; among equal t the lowest lane has the smallest index
            const unsigned tmin = __reduce_min_sync(FULL, __float_as_uint(tt));
            const unsigned who = __ballot_sync(FULL, bb >= 0 && __float_as_uint(tt) == tmin);
            tt = __uint_as_float(tmin);
            bb = who != 0u ? f - lane + (__ffs(who) - 1) : -1;
            // every lane of the ray's group keeps the result, so that its later boxes are tested against it
            if (lane / g == L / g && bb >= 0 && (best < 0 || tt < tbest || (tt == tbest && bb < best))) { tbest = tt; best = bb; }
        }
    }
}

template <bool ANALOG>
__global__ void __launch_bounds__(SAMPLE_THREADS, 2)
sample_design_kernel(const TraceArgs a, const float *__restrict__ verts, const float *__restrict__ mats, float *__restrict__ out,
                     const uint32_t k_offset, const uint32_t raster_n)
{
    extern __shared__ float4 s_tri[];                 // 3 x float4 per triangle of the record being traced
    // rasterised primaries (raster_n = N, else 0): per cell of the emitter grid the ray's position and its closest hit
    float4 *s_cl = s_tri + 3 * a.max_tris;            // 2 x float4 per cluster of 32 triangles: its box (lo, hi)
    float2 *s_puv = reinterpret_cast<float2 *>(s_cl + 2 * ((a.max_tris + SAMPLE_CLUSTER - 1) / SAMPLE_CLUSTER));
    unsigned long long *s_key = reinterpret_cast<unsigned long long *>(s_puv + raster_n);
    __shared__ int s_big[RASTER_BIGCAP];              // triangles over many cells: rasterised by a warp, not a thread
    __shared__ int s_nbig;
    __shared__ WarpQueue s_q[SAMPLE_WARPS];           // photons that go on, per warp
    __shared__ double s_part[SAMPLE_WARPS][3];
    __shared__ unsigned s_hist[SAMPLE_WARPS][16];
    __shared__ unsigned s_next;                       // next ray of the record: all warps of the block draw from it

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    if (lane < 16) s_hist[warp][lane] = 0;
    WarpQueue &Q = s_q[warp];
    LaneCounters cn = { 0, 0, 0, 0, 0, 0, 0, 0 };
    unsigned long long n_tri64 = 0, n_2d64 = 0, n_cl64 = 0;
    unsigned n_cl = 0;                                // cluster-box tests of the record       // every test is counted (32-bit lane counters are folded in per record)

    for (long long m = blockIdx.x; m < a.n_pairs; m += gridDim.x) {
        const long long tbase = a.dz.tri_off[m];
        const int T = (int)(a.dz.tri_off[m + 1] - tbase);
        __syncthreads();                              // the previous record's photons are done with s_tri / s_part
        if (threadIdx.x == 0) s_next = 0u;
        // S1 for a record without a hierarchy, on the way into shared memory: the generator's vertices (verts: 9 floats per
        // triangle, mats: 3) become (v0, alpha) (e1, rho_s) (e2, rho_d), and the block finds the design's box
        float blo[3] = { FLT_MAX, FLT_MAX, FLT_MAX }, bhi[3] = { -FLT_MAX, -FLT_MAX, -FLT_MAX };
        for (int f = threadIdx.x; f < T; f += SAMPLE_THREADS) {
            const float *v = verts + 9 * (tbase + f), *mt = mats + 3 * (tbase + f);
            float p[9];
#pragma unroll
            for (int x = 0; x < 9; ++x) p[x] = __ldg(v + x);
            s_tri[3 * f] = make_float4(p[0], p[1], p[2], __ldg(mt));
            s_tri[3 * f + 1] = make_float4(p[3] - p[0], p[4] - p[1], p[5] - p[2], __ldg(mt + 1));
            s_tri[3 * f + 2] = make_float4(p[6] - p[0], p[7] - p[1], p[8] - p[2], __ldg(mt + 2));
#pragma unroll
            for (int x = 0; x < 9; ++x) { blo[x % 3] = fminf(blo[x % 3], p[x]); bhi[x % 3] = fmaxf(bhi[x % 3], p[x]); }
        }
        float *s_box = reinterpret_cast<float *>(&s_part[0][0]);          // [warp][6]: free until the record's reduction
#pragma unroll
        for (int x = 0; x < 3; ++x) {
            for (int off = 16; off > 0; off >>= 1) {
                blo[x] = fminf(blo[x], __shfl_xor_sync(FULL, blo[x], off)); bhi[x] = fmaxf(bhi[x], __shfl_xor_sync(FULL, bhi[x], off));
            }
            if (lane == 0) { s_box[6 * warp + x] = blo[x]; s_box[6 * warp + 3 + x] = bhi[x]; }
        }
        __syncthreads();
        for (int w = 0; w < SAMPLE_WARPS; ++w)
#pragma unroll
            for (int x = 0; x < 3; ++x) { blo[x] = fminf(blo[x], s_box[6 * w + x]); bhi[x] = fmaxf(bhi[x], s_box[6 * w + 3 + x]); }
        const Emitter em = make_emitter(a.sun_dirs, (int)m, make_float4(blo[0], blo[1], blo[2], 0.f), make_float4(bhi[0], bhi[1], bhi[2], 0.f));
        for (int x = threadIdx.x; x < 3 * T; x += SAMPLE_THREADS) {      // into the emitter frame; materials ride along
            const float4 q = s_tri[x];
            const float3 p = f3(q.x, q.y, q.z);
            s_tri[x] = make_float4(dot3(p, em.u), dot3(p, em.v), dot3(p, em.s), q.w);
        }
        __syncthreads();
        for (int c = warp; c < (T + SAMPLE_CLUSTER - 1) / SAMPLE_CLUSTER; c += SAMPLE_WARPS) {      // cluster boxes: a lane per triangle
            const int f = c * SAMPLE_CLUSTER + lane;
            float lo[3] = { FLT_MAX, FLT_MAX, FLT_MAX }, hi[3] = { -FLT_MAX, -FLT_MAX, -FLT_MAX };
            if (f < T) {
                const float4 q0 = s_tri[3 * f], q1 = s_tri[3 * f + 1], q2 = s_tri[3 * f + 2];
                const float v[3][3] = { { q0.x, q0.x + q1.x, q0.x + q2.x }, { q0.y, q0.y + q1.y, q0.y + q2.y }, { q0.z, q0.z + q1.z, q0.z + q2.z } };
#pragma unroll
                for (int x = 0; x < 3; ++x) { lo[x] = fminf(v[x][0], fminf(v[x][1], v[x][2])); hi[x] = fmaxf(v[x][0], fmaxf(v[x][1], v[x][2])); }
            }
#pragma unroll
            for (int x = 0; x < 3; ++x)
                for (int off = 16; off > 0; off >>= 1) {
                    lo[x] = fminf(lo[x], __shfl_xor_sync(FULL, lo[x], off)); hi[x] = fmaxf(hi[x], __shfl_xor_sync(FULL, hi[x], off));
                }
            if (lane == 0) {
                // widened by the rounding of the vertex sums (the test works on v0, e1, e2)
                const float m = 1.0e-6f * (fabsf(lo[0]) + fabsf(hi[0]) + fabsf(lo[1]) + fabsf(hi[1]) + fabsf(lo[2]) + fabsf(hi[2]));
                s_cl[2 * c] = make_float4(lo[0] - m, lo[1] - m, lo[2] - m, 0.f);
                s_cl[2 * c + 1] = make_float4(hi[0] + m, hi[1] + m, hi[2] + m, 0.f);
            }
        }
        __syncthreads();
        float3 acc = f3(0, 0, 0), acc_t = f3(0, 0, 0);
        if (em.Ae > 0.0f) {                           // else: edge-on flat design, F = 0, nothing launched
            RayGen g;
            g.j = 0u; g.k = (uint32_t)m + k_offset; g.key0 = a.key0; g.key1 = a.key1; g.sampler = a.sampler;
            g.xc = f3(0.f, 0.f, 0.f); g.inv_arm = 1.0f; g.split = false;
            g.inv_nx = 1.0f / (float)(1u << ((a.log2N + 1) >> 1));
            g.inv_ny = 1.0f / (float)(1u << (a.log2N >> 1));
            const uint32_t end = (uint32_t)a.N;
            const float3 sdir = f3(0.f, 0.f, 1.f);    // the photons' travel direction in the emitter frame
            const bool raster = raster_n != 0u && T >= RASTER_MIN_TRIS;          // block-uniform
            if (raster) {
                for (uint32_t i = threadIdx.x; i < end; i += SAMPLE_THREADS) {   // O-step 3 for every ray of the record
                    uint32_t r0, r1, r2, r3;
                    philox4(i, g.j, g.k, 0u, g.key0, g.key1, r0, r1, r2, r3);
                    const float fu = ((float)compact_even_bits(i) + uniform23(r0)) * g.inv_nx;
                    const float fv = ((float)compact_even_bits(i >> 1) + uniform23(r1)) * g.inv_ny;
                    s_puv[i] = make_float2(fmaf(fu, em.du, em.u0), fmaf(fv, em.dv, em.v0));
                    s_key[i] = ~0ULL;
                }
                if (threadIdx.x == 0) s_nbig = 0;
                __syncthreads();
                const int nx = 1 << ((a.log2N + 1) >> 1), ny = 1 << (a.log2N >> 1);
                const float sx = (float)nx / em.du, sy = (float)ny / em.dv;
                const float marg = 1.0e-5f * (fabsf(em.u0) + fabsf(em.v0) + em.du + em.dv);
                for (int f = threadIdx.x; f < T; f += SAMPLE_THREADS) {
                    const float4 q0 = s_tri[3 * f], q1 = s_tri[3 * f + 1], q2 = s_tri[3 * f + 2];
                    int cx0, cx1, cy0, cy1;
                    if (!raster_cells(q0, q1, q2, em, sx, sy, marg, nx, ny, cx0, cx1, cy0, cy1)) continue;
                    if ((cx1 - cx0 + 1) * (cy1 - cy0 + 1) > RASTER_BIG) {
                        const int slot = atomicAdd(&s_nbig, 1);
                        if (slot < RASTER_BIGCAP) { s_big[slot] = f; continue; }
                    }
                    for (int cy = cy0; cy <= cy1; ++cy)
                        for (int cx = cx0; cx <= cx1; ++cx) {
                            const uint32_t i = spread_even_bits((uint32_t)cx) | (spread_even_bits((uint32_t)cy) << 1);
                            raster_test(q0, q1, q2, f, s_puv[i], em.worg, s_key + i);
                            ++n_2d64;
                        }
                }
                __syncthreads();
                const int nbig = s_nbig < RASTER_BIGCAP ? s_nbig : RASTER_BIGCAP;
                for (int b = warp; b < nbig; b += SAMPLE_WARPS) {
                    const int f = s_big[b];
                    const float4 q0 = s_tri[3 * f], q1 = s_tri[3 * f + 1], q2 = s_tri[3 * f + 2];
                    int cx0 = 0, cx1 = -1, cy0 = 0, cy1 = -1;
                    raster_cells(q0, q1, q2, em, sx, sy, marg, nx, ny, cx0, cx1, cy0, cy1);
                    const int w = cx1 - cx0 + 1, n = w * (cy1 - cy0 + 1);
                    for (int x = lane; x < n; x += 32) {
                        const uint32_t i = spread_even_bits((uint32_t)(cx0 + x % w)) | (spread_even_bits((uint32_t)(cy0 + x / w)) << 1);
                        raster_test(q0, q1, q2, f, s_puv[i], em.worg, s_key + i);
                        ++n_2d64;
                    }
                }
                __syncthreads();
            }
            bool more = true;                         // the record still has rays nobody has taken
            int qcount = 0;                           // warp-uniform
            for (;;) {
                bool alive = false;
                uint32_t i = 0;
                float3 o = f3(0, 0, 0), d = sdir;
                int src = -1, depth = 0, share = 1;
                float tbest = FLT_MAX; int best = -1;
                if (qcount >= 32 || (!more && qcount > 0)) {              // a pass of bounce rays
                    const int take = qcount < 32 ? qcount : 32;
                    int np2 = 1;
                    while (np2 < take) np2 <<= 1;
                    share = 32 / np2;                                     // lanes per ray
                    const int r = lane / share;
                    if (r < take) {
                        const int e = qcount - take + r;
                        o = f3(Q.ox[e], Q.oy[e], Q.oz[e]); d = f3(Q.dx[e], Q.dy[e], Q.dz[e]);
                        i = Q.i[e]; src = Q.src_depth[e] & 0x07ffffff; depth = (int)((unsigned)Q.src_depth[e] >> 27);
                        alive = true;
                    }
                    qcount -= take;
                    __syncwarp();
                    closest_shared(s_tri, s_cl, T, alive, o, d, src, share, lane % share, tbest, best, cn.n_tri, n_cl);   // all lanes: it shuffles
                    alive = alive && (lane % share) == 0;                 // one lane per ray goes on to shade
                    if (alive) cn.segments++;
                } else if (more) {                                        // a pass of primaries (O-step 3 in the emitter frame)
                    uint32_t next = 0;
                    if (lane == 0) next = atomicAdd(&s_next, 32u);
                    next = __shfl_sync(FULL, next, 0);
                    more = next + 32u < end;
                    // rasterised: a warp's 32 rays are spread over the grid, so that the warps share the hits evenly
                    i = raster ? (uint32_t)lane * (end >> 5) + (next >> 5) : next + (uint32_t)lane;
                    if (raster && next < end) {
                        const float2 p = s_puv[i];
                        const unsigned long long key = s_key[i];
                        o = f3(p.x, p.y, em.worg);
                        alive = true;
                        cn.launched++; cn.segments++;
                        if (key != ~0ULL) { tbest = __uint_as_float((uint32_t)(key >> 32)); best = (int)(uint32_t)key; }
                    } else if (!raster && i < end) {
                        uint32_t r0, r1, r2, r3;
                        philox4(i, g.j, g.k, 0u, g.key0, g.key1, r0, r1, r2, r3);
                        float fu, fv;
                        if (g.sampler == 0) {
                            fu = ((float)compact_even_bits(i) + uniform23(r0)) * g.inv_nx;
                            fv = ((float)compact_even_bits(i >> 1) + uniform23(r1)) * g.inv_ny;
                        } else { fu = uniform23(r0); fv = uniform23(r1); }
                        o = f3(fmaf(fu, em.du, em.u0), fmaf(fv, em.dv, em.v0), em.worg);
                        alive = true;
                        cn.launched++; cn.segments++;
                        closest_primary(s_tri, T, o.x, o.y, o.z, tbest, best);
                        cn.n_box += (unsigned)T;
                    }
                } else break;                                             // no rays left, queue empty
                int fate = -1;
                if (alive) {
                    if (best < 0) {
                        if (depth == 0) cn.pmiss++; else cn.escaped++;
                    } else {
                        atomicAdd(&s_hist[warp][depth], 1u);
                        const float4 *tp = s_tri + 3 * best;
                        fate = shade<false, 0u, false, ANALOG ? 1 : 0>(tp[0], tp[1], tp[2], tbest, best, g, i, a.B, a.deposit,
                                                                         o, d, src, depth, acc, acc_t);
                        if (fate == SHADE_ABSORBED) cn.absorbed++;
                        if (fate == SHADE_CAPPED) cn.capped++;
                    }
                }
                const unsigned cont = __ballot_sync(FULL, fate == SHADE_CONTINUE);
                SRP_CHECK(qcount + __popc(cont) <= QCAP, "photon queue");
                if (fate == SHADE_CONTINUE) {
                    const int e = qcount + __popc(cont & lt_mask);
                    Q.ox[e] = o.x; Q.oy[e] = o.y; Q.oz[e] = o.z; Q.dx[e] = d.x; Q.dy[e] = d.y; Q.dz[e] = d.z;
                    Q.i[e] = i; Q.src_depth[e] = (depth << 27) | src;
                }
                qcount += __popc(cont);
                __syncwarp();
            }
        }
        n_tri64 += cn.n_tri; cn.n_tri = 0; n_2d64 += cn.n_box; cn.n_box = 0; n_cl64 += n_cl; n_cl = 0;
        // S7: lane fp32 sums -> fp64 warp shuffle tree -> the block's warps in index order -> back to the body frame
        double s[3] = { acc.x, acc.y, acc.z };
#pragma unroll
        for (int c = 0; c < 3; ++c) {
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) s[c] += __shfl_xor_sync(FULL, s[c], off);
            if (lane == 0) s_part[warp][c] = s[c];
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double f[3] = { 0.0, 0.0, 0.0 };
            for (int w = 0; w < SAMPLE_WARPS; ++w)
                for (int c = 0; c < 3; ++c) f[c] += s_part[w][c];
            const double wph = em.Ae > 0.0f ? a.P * (double)em.Ae / (double)a.N : 0.0;
            out[3 * m + 0] = (float)(wph * (f[0] * (double)em.u.x + f[1] * (double)em.v.x + f[2] * (double)em.s.x));
            out[3 * m + 1] = (float)(wph * (f[0] * (double)em.u.y + f[1] * (double)em.v.y + f[2] * (double)em.s.y));
            out[3 * m + 2] = (float)(wph * (f[0] * (double)em.u.z + f[1] * (double)em.v.z + f[2] * (double)em.s.z));
        }
    }
    __syncwarp();
    // primaries' emitter-frame tests are reported as tri2d_tests, bounce rays' Moller-Trumbore tests as tri_tests
    unsigned long long n2d = n_2d64;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        n_tri64 += __shfl_xor_sync(FULL, n_tri64, off); n2d += __shfl_xor_sync(FULL, n2d, off);
        n_cl64 += __shfl_xor_sync(FULL, n_cl64, off);
    }
    if (lane == 0) {
        atomicAdd((unsigned long long *)&a.stats->box_tests, n_cl64);
        atomicAdd((unsigned long long *)&a.stats->tri_tests, n_tri64);
        atomicAdd((unsigned long long *)&a.stats->tri2d_tests, n2d);
    }
    flush_counters<false>(a, cn, s_hist[warp], lane);
}

} // namespace

// records the kernel can take: the triangles of one record must fit the block's shared memory
long long srp_sample_max_tris()
{
    return (190 * 1024) / 49;                    // 48 bytes per triangle and 32 per cluster of 32, beside 36 KB of queues
}

// a.n_pairs records; record m = the triangles [a.dz.tri_off[m], a.dz.tri_off[m + 1]) of verts / mats (the mesh generator's
// output: no box, no packing, no hierarchy) lit from a.sun_dirs[m]; out DEVICE float[n_pairs,3].
cudaError_t srp_launch_sample(const TraceArgs &a, const float *verts, const float *mats, float *out, unsigned k_offset, int num_sms,
                              cudaStream_t stream)
{
    size_t smem = (size_t)a.max_tris * 48 + 32 * (size_t)((a.max_tris + SAMPLE_CLUSTER - 1) / SAMPLE_CLUSTER);
    uint32_t raster_n = 0;                       // rasterised primaries: stratified sampler, a grid of 32 .. 2048 cells that fits
    if (a.sampler == 0 && a.N >= 32 && a.N <= RASTER_MAX_RAYS && a.max_tris >= RASTER_MIN_TRIS && smem + 16 * (size_t)a.N <= 190 * 1024) {
        raster_n = (uint32_t)a.N;
        smem += 16 * (size_t)a.N;
    }
    auto kernel = a.deposit ? sample_design_kernel<true> : sample_design_kernel<false>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, SAMPLE_THREADS, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    long long blocks = (long long)num_sms * per_sm;
    if (blocks > a.n_pairs) blocks = a.n_pairs;
    kernel<<<(unsigned)blocks, SAMPLE_THREADS, smem, stream>>>(a, verts, mats, out, k_offset, raster_n);
    return cudaGetLastError();
}
