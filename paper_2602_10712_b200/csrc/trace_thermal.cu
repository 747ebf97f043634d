// trace_thermal.cu -- thermal (local Lambertian) facet emitters, PAPER.md:606-612 (Sec. 5.9): "our simulation
// easily handles local sources in the same way it does handle distant sun light"; reading R22.
// Facet f of design k radiates |W_f| watts from the side of n = normalize(e1 x e2) (W_f > 0) or of -n (W_f < 0):
// N photons of weight |W_f| / (c N), origin uniform on the triangle, direction cosine-weighted about the emitting
// normal, recoil -(2/3) w n_e at emission, then O-steps 4-7 like any other photon.  The rays are
// incoherent from the start, so this is the per-ray kernel's structure: a warp owns (facet, tile of rays) items,
// traces 32 emitted or 32 queued bounce rays per pass, and keeps the survivors in its shared-memory queue.
#include "trace_common.cuh"

namespace {

constexpr uint32_t THERMAL_FLAG = 0x80000000u;
constexpr double C_LIGHT = 299792458.0;

struct ThermalArgs {
    const float *power;          // [sumT] watts, signed, ORIGINAL triangle order
    const int *emit_list;        // global SORTED triangle positions with non-zero power
    const int *n_emit;           // device: how many
    const float *design_power;   // [D]: sum of |W_f|
};

__device__ inline int find_design_of(const long long *off, int D, long long g)
{
    int lo = 0, hi = D;            // off[lo] <= g < off[hi]
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (off[mid] <= g) lo = mid; else hi = mid;
    }
    return lo;
}

// P_k = sum of |W_f| over design k: one block per design
__global__ void __launch_bounds__(256) thermal_power_kernel(const float *power, const long long *off, float *design_power)
{
    const int k = blockIdx.x;
    double s = 0.0;
    for (long long g = off[k] + threadIdx.x; g < off[k + 1]; g += blockDim.x) s += fabs((double)power[g]);
    __shared__ double sh[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(FULL, s, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) sh[0] += sh[w];
        design_power[k] = (float)sh[0];
    }
}

// sorted positions of the emitting facets (order does not matter: the sums are integer)
__global__ void __launch_bounds__(256) thermal_list_kernel(const float *power, const DesignsDev dz, long long sumT, int *emit_list, int *n_emit)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= sumT) return;
    const int k = find_design_of(dz.tri_off, dz.D, g);
    const long long base = dz.tri_off[k];
    if (power[base + dz.perm[g]] != 0.0f) emit_list[atomicAdd(n_emit, 1)] = (int)g;
}

#ifndef THERMAL_BLOCKS_PER_SM
#define THERMAL_BLOCKS_PER_SM 8
#endif
template <bool BVH, bool GLOSSY>
__global__ void __launch_bounds__(TRACE_THREADS, THERMAL_BLOCKS_PER_SM)
thermal_trace_kernel(const TraceArgs a, const ThermalArgs h)
{
    __shared__ int s_stack[BVH ? STACK_SMEM * TRACE_THREADS : 1];
    __shared__ WarpQueue s_q[TRACE_WARPS];
    __shared__ unsigned s_hist[TRACE_WARPS][16];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    if (lane < 16) s_hist[warp][lane] = 0;
    __syncwarp();
    WarpQueue &Q = s_q[warp];
    LaneCounters cn = { 0, 0, 0, 0, 0, 0, 0, 0 };
    const unsigned long long total_tiles = (unsigned long long)(*h.n_emit) * a.tiles_per_pair;

    for (;;) {
        unsigned long long tile = 0;
        if (lane == 0) tile = atomicAdd(a.work_counter, 1ULL);
        tile = __shfl_sync(FULL, tile, 0);
        if (tile >= total_tiles) break;
        const long long e = (long long)(tile / a.tiles_per_pair);
        const long long q = (long long)(tile - (unsigned long long)e * a.tiles_per_pair);
        const long long gpos = h.emit_list[e];                       // global sorted position of the facet
        const int k = find_design_of(a.dz.tri_off, a.dz.D, gpos);
        const long long tbase = a.dz.tri_off[k];
        const int T = (int)(a.dz.tri_off[k + 1] - tbase);
        const int fs = (int)(gpos - tbase);                          // sorted position within the design
        const int f = a.dz.perm[gpos];                               // original facet index (Philox counter, R22)
        const float W = h.power[tbase + f];
        const float Pk = h.design_power[k];
        const float4 *gtri = a.dz.tri + 3 * tbase;
        const float4 *gnodes = SRP_TRAV_NODES(a.dz, tbase);
        const float4 q0 = __ldg(gtri + 3 * fs), q1 = __ldg(gtri + 3 * fs + 1), q2 = __ldg(gtri + 3 * fs + 2);
        float3 n = cross3(f3(q1.x, q1.y, q1.z), f3(q2.x, q2.y, q2.z));
        const float il = 1.0f / sqrtf(dot3(n, n));
        const float sgn = W > 0.0f ? il : -il;
        const float3 ne = f3(n.x * sgn, n.y * sgn, n.z * sgn);       // emitting normal
        const float ie = rsqrtf(q1.x * q1.x + q1.y * q1.y + q1.z * q1.z);
        const float3 tu = f3(q1.x * ie, q1.y * ie, q1.z * ie), tv = cross3(ne, tu);     // R18 frame
        RayGen g;
        g.j = (uint32_t)f; g.k = (uint32_t)k; g.key0 = a.key0; g.key1 = a.key1; g.sampler = 0;
        g.inv_nx = g.inv_ny = 0.f; g.xc = f3(0.f, 0.f, 0.f);
        uint32_t next = (uint32_t)(q * a.tile_rays);
        const uint32_t end = (uint32_t)min((long long)a.N, (q + 1) * (long long)a.tile_rays);
        int qcount = 0;                                   // warp-uniform
        float3 acc = f3(0, 0, 0), acc_t = f3(0, 0, 0);

        for (;;) {
            bool alive = false;
            uint32_t i = 0;
            float3 o = f3(0, 0, 0), d = ne;
            int src = fs, depth = 0;
            if (qcount >= 32 || (next >= end && qcount > 0)) {          // a pass of bounce rays
                const int take = qcount < 32 ? qcount : 32;
                if (lane < take) {
                    const int x = qcount - take + lane;
                    o = f3(Q.ox[x], Q.oy[x], Q.oz[x]); d = f3(Q.dx[x], Q.dy[x], Q.dz[x]);
                    i = Q.i[x]; src = Q.src_depth[x] & 0x07ffffff; depth = (int)((unsigned)Q.src_depth[x] >> 27);
                    alive = true;
                }
                qcount -= take;
            } else if (next < end) {                                     // a pass of emitted photons
                const uint32_t mine = next + lane;
                if (mine < end) {
                    i = mine;
                    uint32_t r0, r1, r2, r3;
                    philox4(i, g.j, g.k, THERMAL_FLAG, g.key0, g.key1, r0, r1, r2, r3);
                    const float x0 = uniform23(r0), x1 = uniform23(r1), x2 = uniform23(r2), x3 = uniform23(r3);
                    const float su = sqrtf(x0), b1 = su * (1.0f - x1), b2 = su * x1;
                    const float3 x = f3(fmaf(b1, q1.x, fmaf(b2, q2.x, q0.x)), fmaf(b1, q1.y, fmaf(b2, q2.y, q0.y)),
                                        fmaf(b1, q1.z, fmaf(b2, q2.z, q0.z)));
                    float sn, cs;
                    sincospif(2.0f * x2, &sn, &cs);
                    const float rho = sqrtf(x3), lz = sqrtf(1.0f - x3), lx = rho * cs, ly = rho * sn;
                    d = f3(fmaf(lx, tu.x, fmaf(ly, tv.x, lz * ne.x)), fmaf(lx, tu.y, fmaf(ly, tv.y, lz * ne.y)),
                           fmaf(lx, tu.z, fmaf(ly, tv.z, lz * ne.z)));
                    // recoil at emission (2/3 of a collimated beam), expected value or analog
                    if (a.deposit == 0) { acc.x -= (2.0f / 3.0f) * ne.x; acc.y -= (2.0f / 3.0f) * ne.y; acc.z -= (2.0f / 3.0f) * ne.z; }
                    else { acc.x -= d.x; acc.y -= d.y; acc.z -= d.z; }
                    // same fp32 guard as for bounce rays (R10): start just above the facet
                    const float lift = 1.0e-6f * (fabsf(x.x) + fabsf(x.y) + fabsf(x.z));
                    o = f3(fmaf(lift, ne.x, x.x), fmaf(lift, ne.y, x.y), fmaf(lift, ne.z, x.z));
                    alive = true; cn.launched++;
                    if (a.dz.esc && esc_escapes(a.dz.esc, gpos, W > 0.0f ? 0 : 1, d.x, d.y, d.z)) {
                        alive = false; cn.segments++; cn.pmiss++; cn.mesc++;      // nothing in that direction
                    }
                }
                next = (end - next) < 32u ? end : next + 32u;
            } else break;
            __syncwarp();
            int fate = -1;
            if (alive) {
                float tbest = FLT_MAX; int best = -1;
                cn.segments++;
                if (BVH) closest_bvh<false>(gnodes, gtri, o, d, src, tbest, best, s_stack + threadIdx.x, cn.n_box, cn.n_tri);
                else closest_brute<false>(gtri, T, o, d, src, tbest, best, cn.n_tri);
                if (best < 0) {
                    if (depth == 0) cn.pmiss++; else cn.escaped++;
                } else {
                    atomicAdd(&s_hist[warp][depth], 1u);
                    fate = shade<false, THERMAL_FLAG, GLOSSY>(__ldg(gtri + 3 * best), __ldg(gtri + 3 * best + 1), __ldg(gtri + 3 * best + 2),
                                                      tbest, best, g, i, a.B, a.deposit, o, d, src, depth, acc, acc_t, a.dz.esc, tbase + best, a.dz.shin);
                    if (fate == SHADE_ESCAPES) { cn.segments++; cn.escaped++; cn.mesc++; }
                    if (fate == SHADE_ABSORBED) cn.absorbed++;
                    if (fate == SHADE_CAPPED) cn.capped++;
                }
            }
            const unsigned cont = __ballot_sync(FULL, fate == SHADE_CONTINUE);
            if (fate == SHADE_CONTINUE) {
                const int x = qcount + __popc(cont & lt_mask);
                Q.ox[x] = o.x; Q.oy[x] = o.y; Q.oz[x] = o.z; Q.dx[x] = d.x; Q.dy[x] = d.y; Q.dz[x] = d.z;
                Q.i[x] = i; Q.src_depth[x] = (depth << 27) | src;
            }
            qcount += __popc(cont);
            __syncwarp();
        }
        // S7: this facet's photons all weigh |W_f| / P_k of the design's accumulator
        const float wrel = fabsf(W) / Pk;
        flush_tile_acc<false>(a, (long long)k, f3(acc.x * wrel, acc.y * wrel, acc.z * wrel), acc_t, lane);
    }
    flush_counters<false>(a, cn, s_hist[warp], lane);
}

// F[k] = accum[k] * 2^-32 * P_k / (c N)
__global__ void __launch_bounds__(256) thermal_finalize_kernel(const TraceArgs a, const float *design_power, float *out)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= a.dz.D) return;
    const double w = (double)design_power[k] / (C_LIGHT * (double)a.N) / a.acc_scale;
#pragma unroll
    for (int c = 0; c < 3; ++c) out[3 * k + c] = (float)((double)a.accum[3 * k + c] * w);
}

} // namespace

// scratch: emit_list int[sumT], n_emit int[1], design_power float[D] (all device); a.n_pairs is unused,
// a.tiles_per_pair = tiles per emitting facet, a.accum = int64[D*3] zeroed, a.acc_stride = 3.
cudaError_t srp_launch_thermal(const TraceArgs &a, const float *facet_power, long long sumT, int *emit_list, int *n_emit,
                               float *design_power, float *out_forces, int num_sms, cudaStream_t stream)
{
    cudaError_t e = cudaMemsetAsync(n_emit, 0, sizeof(int), stream);
    if (e != cudaSuccess) return e;
    thermal_power_kernel<<<a.dz.D, 256, 0, stream>>>(facet_power, a.dz.tri_off, design_power);
    thermal_list_kernel<<<(unsigned)((sumT + 255) / 256), 256, 0, stream>>>(facet_power, a.dz, sumT, emit_list, n_emit);
    ThermalArgs h;
    h.power = facet_power; h.emit_list = emit_list; h.n_emit = n_emit; h.design_power = design_power;
    const bool gl = a.dz.shin != nullptr;
    int per_sm = a.dz.has_bvh ? (gl ? blocks_per_sm(thermal_trace_kernel<true, true>) : blocks_per_sm(thermal_trace_kernel<true, false>))
                              : (gl ? blocks_per_sm(thermal_trace_kernel<false, true>) : blocks_per_sm(thermal_trace_kernel<false, false>));
    if (per_sm < 1) per_sm = 1;
    const unsigned blocks = (unsigned)(num_sms * per_sm);             // persistent; the item count lives on the device
    if (a.dz.has_bvh) {
        if (gl) thermal_trace_kernel<true, true><<<blocks, TRACE_THREADS, 0, stream>>>(a, h);
        else thermal_trace_kernel<true, false><<<blocks, TRACE_THREADS, 0, stream>>>(a, h);
    } else {
        if (gl) thermal_trace_kernel<false, true><<<blocks, TRACE_THREADS, 0, stream>>>(a, h);
        else thermal_trace_kernel<false, false><<<blocks, TRACE_THREADS, 0, stream>>>(a, h);
    }
    thermal_finalize_kernel<<<(a.dz.D + 255) / 256, 256, 0, stream>>>(a, design_power, out_forces);
    return cudaGetLastError();
}
