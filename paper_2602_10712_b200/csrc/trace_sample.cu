// trace_sample.cu -- sample_design_kernel: the paper's own workload shape ("not ... for a specific light
// direction and a specific design parameter vector in one thread, but for many of these in a batch"; "each
// ray effectively intersects a different world ... each of these rays, for each bounce, is tested against all
// triangles in parallel"; "100 k light directions and/or designs x 1000 samples, ~1 k faces").
// Every record m has its own design theta_m AND its own light direction omega_m, and only ~10^3 photons: a hierarchy
// would never be repaid, so -- as in the paper -- there is none.  One thread block per record: the record's packed
// triangles (generated just before by mesh_gen.cu for this chunk of records) are staged in shared memory once, the
// block's warps trace the record's photons against ALL of them (S3-S6, Moller-Trumbore, operands broadcast from
// shared memory, lanes refilled as photons end), and the block reduces the deposits in a fixed order (S7).
#include "trace_common.cuh"

namespace {

constexpr int SAMPLE_THREADS = 256;
constexpr int SAMPLE_WARPS = SAMPLE_THREADS / 32;

template <bool ANALOG>
__global__ void __launch_bounds__(SAMPLE_THREADS)
sample_design_kernel(const TraceArgs a, float *__restrict__ out, const uint32_t k_offset)
{
    extern __shared__ float4 s_tri[];                 // 3 x float4 per triangle of the record being traced
    __shared__ double s_part[SAMPLE_WARPS][3];
    __shared__ unsigned s_hist[SAMPLE_WARPS][16];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    if (lane < 16) s_hist[warp][lane] = 0;
    LaneCounters cn = { 0, 0, 0, 0, 0, 0, 0, 0 };
    // rays of a record are split over the warps in contiguous runs (a multiple of 32, so that a warp's first pass is full)
    const uint32_t per_warp = (uint32_t)((((a.N + SAMPLE_WARPS - 1) / SAMPLE_WARPS) + 31) / 32 * 32);

    for (long long m = blockIdx.x; m < a.n_pairs; m += gridDim.x) {
        const long long tbase = a.dz.tri_off[m];
        const int T = (int)(a.dz.tri_off[m + 1] - tbase);
        __syncthreads();                              // the previous record's photons are done with s_tri / s_part
        for (int x = threadIdx.x; x < 3 * T; x += SAMPLE_THREADS) s_tri[x] = __ldg(a.dz.tri + 3 * tbase + x);
        __syncthreads();
        const Emitter em = make_emitter(a.sun_dirs, (int)m, a.dz.box[2 * m], a.dz.box[2 * m + 1]);
        float3 acc = f3(0, 0, 0), acc_t = f3(0, 0, 0);
        if (em.Ae > 0.0f) {                           // else: edge-on flat design, F = 0, nothing launched
            RayGen g;
            g.j = 0u; g.k = (uint32_t)m + k_offset; g.key0 = a.key0; g.key1 = a.key1; g.sampler = a.sampler;
            g.xc = f3(0.f, 0.f, 0.f); g.inv_arm = 1.0f; g.split = false;
            g.inv_nx = 1.0f / (float)(1u << ((a.log2N + 1) >> 1));
            g.inv_ny = 1.0f / (float)(1u << (a.log2N >> 1));
            uint32_t next = min((uint32_t)a.N, (uint32_t)warp * per_warp);
            const uint32_t end = min((uint32_t)a.N, next + per_warp);
            bool alive = false;
            uint32_t i = 0;
            float3 o = f3(0, 0, 0), d = em.s;
            int src = -1, depth = 0;
            for (;;) {
                // S6: lanes whose photon ended take the next rays of the warp's run
                const unsigned need = __ballot_sync(FULL, !alive);
                if (need) {
                    const uint32_t mine = next + __popc(need & lt_mask);
                    if (!alive && mine < end) {
                        i = mine; make_ray(em, g, i, o); d = em.s; src = -1; depth = 0; alive = true;
                        cn.launched++;
                    }
                    const uint32_t room = end - next, want = __popc(need);
                    next += want < room ? want : room;
                }
                if (!__any_sync(FULL, alive)) break;
                if (alive) {
                    float tbest = FLT_MAX; int best = -1;
                    cn.segments++;
                    closest_brute<false>(s_tri, T, o, d, src, tbest, best, cn.n_tri);
                    if (best < 0) {
                        if (depth == 0) cn.pmiss++; else cn.escaped++;
                        alive = false;
                    } else {
                        atomicAdd(&s_hist[warp][depth], 1u);
                        const float4 *tp = s_tri + 3 * best;
                        const int fate = shade<false, 0u, false, ANALOG ? 1 : 0>(tp[0], tp[1], tp[2], tbest, best, g, i, a.B, a.deposit,
                                                                                   o, d, src, depth, acc, acc_t);
                        if (fate == SHADE_ABSORBED) cn.absorbed++;
                        if (fate == SHADE_CAPPED) cn.capped++;
                        alive = fate == SHADE_CONTINUE;
                    }
                }
            }
        }
        // S7: lane fp32 sums -> fp64 warp shuffle tree -> the block's warps in index order
        double s[3] = { acc.x, acc.y, acc.z };
#pragma unroll
        for (int c = 0; c < 3; ++c) {
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) s[c] += __shfl_xor_sync(FULL, s[c], off);
            if (lane == 0) s_part[warp][c] = s[c];
        }
        __syncthreads();
        if (threadIdx.x < 3) {
            double f = 0.0;
            for (int w = 0; w < SAMPLE_WARPS; ++w) f += s_part[w][threadIdx.x];
            const double wph = em.Ae > 0.0f ? a.P * (double)em.Ae / (double)a.N : 0.0;
            out[3 * m + threadIdx.x] = (float)(f * wph);
        }
    }
    __syncwarp();
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
