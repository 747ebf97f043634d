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

// O-step 4 for the bounce rays of a pass.  n <= 32 rays wait in the warp's queue; with fewer than 17 the lanes are
// shared out: g = 32 / n' lanes per ray (n' = n rounded up to a power of two), each testing every g-th triangle,
// then a minimum over the group (smallest t, ties to the smallest index as in the definition) -- so that the few
// photons of the deep bounces, of which a record with ~10^3 photons has only a handful, still fill the warp.
__device__ __forceinline__ void closest_shared(const float4 *__restrict__ tp, const int T, const float3 o, const float3 d,
                                               const int src, const int g, const int sub, float &tbest, int &best, unsigned &n_tri)
{
    for (int f = sub; f < T; f += g) {
        if (f == src) continue;
        tri_test(tp[3 * f], tp[3 * f + 1], tp[3 * f + 2], o, d, f, tbest, best);
    }
    n_tri += (unsigned)((T - sub + g - 1) / g);
    for (int off = 1; off < g; off <<= 1) {           // the g lanes of a ray are consecutive
        const float t2 = __shfl_xor_sync(FULL, tbest, off);
        const int b2 = __shfl_xor_sync(FULL, best, off);
        if (b2 >= 0 && (t2 < tbest || (t2 == tbest && b2 < best) || best < 0)) { tbest = t2; best = b2; }
    }
}

template <bool ANALOG>
__global__ void __launch_bounds__(SAMPLE_THREADS, 2)
sample_design_kernel(const TraceArgs a, float *__restrict__ out, const uint32_t k_offset)
{
    extern __shared__ float4 s_tri[];                 // 3 x float4 per triangle of the record being traced
    __shared__ WarpQueue s_q[SAMPLE_WARPS];           // photons that go on, per warp
    __shared__ double s_part[SAMPLE_WARPS][3];
    __shared__ unsigned s_hist[SAMPLE_WARPS][16];
    __shared__ unsigned s_next;                       // next ray of the record: all warps of the block draw from it

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    if (lane < 16) s_hist[warp][lane] = 0;
    WarpQueue &Q = s_q[warp];
    LaneCounters cn = { 0, 0, 0, 0, 0, 0, 0, 0 };
    unsigned long long n_tri64 = 0, n_2d64 = 0;       // every test is counted (32-bit lane counters are folded in per record)

    for (long long m = blockIdx.x; m < a.n_pairs; m += gridDim.x) {
        const long long tbase = a.dz.tri_off[m];
        const int T = (int)(a.dz.tri_off[m + 1] - tbase);
        const Emitter em = make_emitter(a.sun_dirs, (int)m, a.dz.box[2 * m], a.dz.box[2 * m + 1]);
        __syncthreads();                              // the previous record's photons are done with s_tri / s_part
        if (threadIdx.x == 0) s_next = 0u;
        for (int x = threadIdx.x; x < 3 * T; x += SAMPLE_THREADS) {      // into the emitter frame; materials ride along
            const float4 q = __ldg(a.dz.tri + 3 * tbase + x);
            const float3 p = f3(q.x, q.y, q.z);
            s_tri[x] = make_float4(dot3(p, em.u), dot3(p, em.v), dot3(p, em.s), q.w);
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
                    closest_shared(s_tri, alive ? T : 0, o, d, src, share, lane % share, tbest, best, cn.n_tri);   // all lanes: it shuffles
                    alive = alive && (lane % share) == 0;                 // one lane per ray goes on to shade
                    if (alive) cn.segments++;
                } else if (more) {                                        // a pass of primaries (O-step 3 in the emitter frame)
                    uint32_t next = 0;
                    if (lane == 0) next = atomicAdd(&s_next, 32u);
                    next = __shfl_sync(FULL, next, 0);
                    more = next + 32u < end;
                    i = next + (uint32_t)lane;
                    if (i < end) {
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
        n_tri64 += cn.n_tri; cn.n_tri = 0; n_2d64 += cn.n_box; cn.n_box = 0;
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
    }
    if (lane == 0) {
        atomicAdd((unsigned long long *)&a.stats->tri_tests, n_tri64);
        atomicAdd((unsigned long long *)&a.stats->tri2d_tests, n2d);
    }
    flush_counters<false>(a, cn, s_hist[warp], lane);
}

} // namespace

// records the kernel can take: the triangles of one record must fit the block's shared memory
long long srp_sample_max_tris()
{
    return (200 * 1024) / 48;
}

// a.n_pairs records; record m = design m of a.dz (no hierarchy) lit from a.sun_dirs[m]; out DEVICE float[n_pairs,3].
cudaError_t srp_launch_sample(const TraceArgs &a, float *out, unsigned k_offset, int num_sms, cudaStream_t stream)
{
    const size_t smem = (size_t)a.max_tris * 48;
    auto kernel = a.deposit ? sample_design_kernel<true> : sample_design_kernel<false>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, SAMPLE_THREADS, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    long long blocks = (long long)num_sms * per_sm;
    if (blocks > a.n_pairs) blocks = a.n_pairs;
    kernel<<<(unsigned)blocks, SAMPLE_THREADS, smem, stream>>>(a, out, k_offset);
    return cudaGetLastError();
}
