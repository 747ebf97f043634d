// trace_perray.cu -- the per-ray trace kernels (S2-S7): every segment finds its closest hit on its own, by BVH2
// stack traversal (bvh_trace_kernel: dense meshes with about one ray per triangle, i.i.d. sampler) or by testing all
// triangles (trace_kernel: designs without a hierarchy under the i.i.d. sampler; force_brute).
// Also finalize_kernel (S7) and the first-hit debug kernel.
#include "trace_common.cuh"

namespace {

// ---- the persistent trace kernel ----
template <int MODE, bool INSTR, bool TORQUE, bool GLOSSY, bool ANALOG>
__global__ void __launch_bounds__(TRACE_THREADS, MODE == MODE_BVH ? 4 : 5)
trace_kernel(const TraceArgs a)
{
    __shared__ int s_stack[MODE == MODE_BVH ? STACK_SMEM * TRACE_THREADS : 1];
    __shared__ float4 s_tri[MODE == MODE_BRUTE_SMEM ? TRACE_WARPS * SRP_BRUTE_MAX_TRIS * 3 : 1];
    __shared__ unsigned s_hist[TRACE_WARPS][16];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    if (lane < 16) s_hist[warp][lane] = 0;
    __syncwarp();
    LaneCounters cn = { 0, 0, 0, 0, 0, 0, 0, 0 };
    const unsigned long long total_tiles = (unsigned long long)a.n_pairs * a.tiles_per_pair;
    int loaded_k = -1;
    float4 *my_tri = s_tri + (MODE == MODE_BRUTE_SMEM ? warp * SRP_BRUTE_MAX_TRIS * 3 : 0);

    for (;;) {
        unsigned long long tile = 0;
        if (lane == 0) tile = atomicAdd(a.work_counter, 1ULL);
        tile = __shfl_sync(FULL, tile, 0);
        if (tile >= total_tiles) break;
        const long long p = (long long)(tile / a.tiles_per_pair);
        const long long q = (long long)(tile - (unsigned long long)p * a.tiles_per_pair);
        int k, j;
        pair_of(a, p, k, j);
        const Emitter em = make_emitter(a.sun_dirs, j, a.dz.box[2 * k], a.dz.box[2 * k + 1]);
        if (!(em.Ae > 0.0f)) continue;                      // edge-on flat design: F = 0, nothing launched
        const long long tbase = a.dz.tri_off[k];
        const int T = (int)(a.dz.tri_off[k + 1] - tbase);
        const float4 *gtri = a.dz.tri + 3 * tbase;
        const float4 *gnodes = SRP_TRAV_NODES(a.dz, tbase);
        if (MODE == MODE_BRUTE_SMEM && loaded_k != k) {
            __syncwarp();
            for (int x = lane; x < 3 * T; x += 32) my_tri[x] = gtri[x];
            __syncwarp();
            loaded_k = k;
        }
        RayGen g;
        g.j = (uint32_t)j; g.k = (uint32_t)k; g.key0 = a.key0; g.key1 = a.key1; g.sampler = a.sampler; set_torque<TORQUE>(g, a, k);
        g.inv_nx = 1.0f / (float)(1u << ((a.log2N + 1) >> 1));
        g.inv_ny = 1.0f / (float)(1u << (a.log2N >> 1));
        uint32_t next = (uint32_t)(q * a.tile_rays);
        const uint32_t end = (uint32_t)min((long long)a.N, (q + 1) * (long long)a.tile_rays);

        bool alive = false;
        uint32_t i = 0;
        unsigned long long sig = 0;                         // debug: hash of the hit-triangle sequence
        float3 o = f3(0, 0, 0), d = em.s, acc = f3(0, 0, 0), acc_t = f3(0, 0, 0);
        int src = -1, depth = 0;
        for (;;) {
            // S6: lanes whose photon ended take the next rays of the tile
            const unsigned need = __ballot_sync(FULL, !alive);
            if (need) {
                const uint32_t mine = next + __popc(need & lt_mask);
                if (!alive && mine < end) {
                    i = mine; make_ray(em, g, i, o); d = em.s; src = -1; depth = 0; alive = true;
                    cn.launched++;
                    if (INSTR) sig = 0;
                }
                const uint32_t room = end - next, want = __popc(need);
                next += want < room ? want : room;
            }
            if (!__any_sync(FULL, alive)) break;
            if (alive) {
                float tbest = FLT_MAX; int best = -1;
                cn.segments++;
                if (MODE == MODE_BVH)
                    closest_bvh<INSTR>(gnodes, gtri, o, d, src, tbest, best, s_stack + threadIdx.x, cn.n_box, cn.n_tri);
                else if (MODE == MODE_BRUTE_SMEM)
                    closest_brute<INSTR>(my_tri, T, o, d, src, tbest, best, cn.n_tri);
                else
                    closest_brute<INSTR>(gtri, T, o, d, src, tbest, best, cn.n_tri);
                if (best < 0) {
                    if (depth == 0) cn.pmiss++; else cn.escaped++;
                    alive = false;
                } else {
                    atomicAdd(&s_hist[warp][depth], 1u);
                    const float4 *tp = (MODE == MODE_BRUTE_SMEM) ? my_tri + 3 * best : gtri + 3 * best;
                    if (INSTR) sig = sig * 1000003ULL + (unsigned long long)(a.dz.perm[tbase + best] + 1);
                    const int fate = shade<TORQUE, 0u, GLOSSY, ANALOG ? 1 : 0>(tp[0], tp[1], tp[2], tbest, best, g, i, a.B, a.deposit, o, d, src, depth, acc, acc_t,
                                                   nullptr, tbase + best, a.dz.shin);
                    if (fate == SHADE_ABSORBED) cn.absorbed++;
                    if (fate == SHADE_CAPPED) cn.capped++;
                    alive = fate == SHADE_CONTINUE;
                }
                if (INSTR && !alive && a.sig_out) a.sig_out[p * a.N + i] = sig;
            }
        }
        // S7: warp reduction in fp64, then one fixed-point atomic per component
        flush_tile_acc<TORQUE>(a, p, acc, acc_t, lane);
    }
    flush_counters<INSTR>(a, cn, s_hist[warp], lane);
}

// ---- the BVH trace kernel: persistent warps with a per-warp queue of bounce rays ----
// A warp traces 32 rays of ONE kind per pass: either 32 fresh primaries of its tile (parallel, in
// Morton order, so they walk the same part of the tree) or 32 queued secondary rays (incoherent, and
// mostly gone after a few nodes).  Photons that survive shading are pushed to the warp's queue in
// shared memory (ballot + prefix popcount, so the order is deterministic) and popped 32 at a time.
// Mixing the two kinds in one pass left the short secondaries waiting for the long primaries
// (14 of 32 lanes active, profiles/ round 1); this is S6's "compaction between bounces".

// MASKS: the designs carry escape masks (a build of its own: the lookup's branch costs the sail 2.8 % when it is
// only a run-time null test -- 603.9 against 620.9 ms, profiles/r1d_escape_masks.md).
#ifndef PERRAY_BLOCKS_PER_SM
#define PERRAY_BLOCKS_PER_SM 10
#endif
template <bool MASKS, bool INSTR, bool TORQUE, bool GLOSSY, bool ANALOG>
__global__ void __launch_bounds__(TRACE_THREADS, PERRAY_BLOCKS_PER_SM)
bvh_trace_kernel(const TraceArgs a)
{
    __shared__ int s_stack[STACK_SMEM * TRACE_THREADS];
    __shared__ WarpQueue s_q[TRACE_WARPS];
    __shared__ unsigned long long s_qsig[INSTR ? TRACE_WARPS * QCAP : 1];
    __shared__ unsigned s_hist[TRACE_WARPS][16];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    if (lane < 16) s_hist[warp][lane] = 0;
    __syncwarp();
    WarpQueue &Q = s_q[warp];
    unsigned long long *qsig = s_qsig + (INSTR ? warp * QCAP : 0);
    LaneCounters cn = { 0, 0, 0, 0, 0, 0, 0, 0 };
    const unsigned long long total_tiles = (unsigned long long)a.n_pairs * a.tiles_per_pair;

    for (;;) {
        unsigned long long tile = 0;
        if (lane == 0) tile = atomicAdd(a.work_counter, 1ULL);
        tile = __shfl_sync(FULL, tile, 0);
        if (tile >= total_tiles) break;
        const long long p = (long long)(tile / a.tiles_per_pair);
        const long long q = (long long)(tile - (unsigned long long)p * a.tiles_per_pair);
        int k, j;
        pair_of(a, p, k, j);
        const Emitter em = make_emitter(a.sun_dirs, j, a.dz.box[2 * k], a.dz.box[2 * k + 1]);
        if (!(em.Ae > 0.0f)) continue;
        const long long tbase = a.dz.tri_off[k];
        const float4 *gtri = a.dz.tri + 3 * tbase;
        const float4 *gnodes = SRP_TRAV_NODES(a.dz, tbase);
        RayGen g;
        g.j = (uint32_t)j; g.k = (uint32_t)k; g.key0 = a.key0; g.key1 = a.key1; g.sampler = a.sampler; set_torque<TORQUE>(g, a, k);
        g.inv_nx = 1.0f / (float)(1u << ((a.log2N + 1) >> 1));
        g.inv_ny = 1.0f / (float)(1u << (a.log2N >> 1));
        uint32_t next = (uint32_t)(q * a.tile_rays);
        const uint32_t end = (uint32_t)min((long long)a.N, (q + 1) * (long long)a.tile_rays);
        int qcount = 0;                                   // warp-uniform
        float3 acc = f3(0, 0, 0), acc_t = f3(0, 0, 0);

        for (;;) {
            bool alive = false;
            uint32_t i = 0;
            float3 o = f3(0, 0, 0), d = em.s;
            int src = -1, depth = 0;
            unsigned long long sig = 0;
            if (qcount >= 32 || (next >= end && qcount > 0)) {          // a pass of secondary rays
                const int take = qcount < 32 ? qcount : 32;
                if (lane < take) {
                    const int e = qcount - take + lane;
                    o = f3(Q.ox[e], Q.oy[e], Q.oz[e]); d = f3(Q.dx[e], Q.dy[e], Q.dz[e]);
                    i = Q.i[e]; src = Q.src_depth[e] & 0x07ffffff; depth = (int)((unsigned)Q.src_depth[e] >> 27);
                    if (INSTR) sig = qsig[e];
                    alive = true;
                }
                qcount -= take;
            } else if (next < end) {                                     // a pass of primaries
                const uint32_t mine = next + lane;
                if (mine < end) { i = mine; make_ray(em, g, i, o); alive = true; cn.launched++; }
                next = (end - next) < 32u ? end : next + 32u;
            } else break;                                                // tile exhausted, queue empty
            __syncwarp();
            int fate = -1;                                               // -1: no hit / no photon
            if (alive) {
                float tbest = FLT_MAX; int best = -1;
                cn.segments++;
                closest_bvh<INSTR>(gnodes, gtri, o, d, src, tbest, best, s_stack + threadIdx.x, cn.n_box, cn.n_tri);
                if (best < 0) {
                    if (depth == 0) cn.pmiss++; else cn.escaped++;
                } else {
                    atomicAdd(&s_hist[warp][depth], 1u);
                    if (INSTR) sig = sig * 1000003ULL + (unsigned long long)(a.dz.perm[tbase + best] + 1);
                    fate = shade<TORQUE, 0u, GLOSSY, ANALOG ? 1 : 0>(__ldg(gtri + 3 * best), __ldg(gtri + 3 * best + 1), __ldg(gtri + 3 * best + 2), tbest,
                                 best, g, i, a.B, a.deposit, o, d, src, depth, acc, acc_t, MASKS ? a.dz.esc : nullptr, tbase + best, a.dz.shin);
                    if (fate == SHADE_ESCAPES) { cn.segments++; cn.escaped++; cn.mesc++; }
                    if (fate == SHADE_ABSORBED) cn.absorbed++;
                    if (fate == SHADE_CAPPED) cn.capped++;
                }
                if (INSTR && fate != SHADE_CONTINUE && a.sig_out) a.sig_out[p * a.N + i] = sig;
            }
            const unsigned cont = __ballot_sync(FULL, fate == SHADE_CONTINUE);
            if (fate == SHADE_CONTINUE) {
                const int e = qcount + __popc(cont & lt_mask);
                Q.ox[e] = o.x; Q.oy[e] = o.y; Q.oz[e] = o.z; Q.dx[e] = d.x; Q.dy[e] = d.y; Q.dz[e] = d.z;
                Q.i[e] = i; Q.src_depth[e] = (depth << 27) | src;
                if (INSTR) qsig[e] = sig;
            }
            qcount += __popc(cont);
            __syncwarp();
        }
        // S7: warp reduction in fp64, then one fixed-point atomic per component
        flush_tile_acc<TORQUE>(a, p, acc, acc_t, lane);
    }
    flush_counters<INSTR>(a, cn, s_hist[warp], lane);
}


// F[p] = accum[p] * 2^-32 * P * A_e / N
__global__ void __launch_bounds__(256) finalize_kernel(const TraceArgs a, float *out, float *out_torque)
{
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= a.n_pairs) return;
    int k, j;
    pair_of(a, p, k, j);
    const Emitter em = make_emitter(a.sun_dirs, j, a.dz.box[2 * k], a.dz.box[2 * k + 1]);
    const double w = em.Ae > 0.0f ? a.P * (double)em.Ae / (double)a.N / a.acc_scale : 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) out[3 * p + c] = (float)((double)a.accum[a.acc_stride * p + c] * w);
    if (a.torque && out_torque) {
        // second output: torque (arms were summed in units of torque_arm_scale), or the direct part of the force
        double w2 = w;
        if (a.torque == 1) {
            const float3 xc = a.xcom ? f3(a.xcom[3 * k], a.xcom[3 * k + 1], a.xcom[3 * k + 2]) : f3(0.f, 0.f, 0.f);
            w2 *= (double)torque_arm_scale(a.dz.box[2 * k], a.dz.box[2 * k + 1], xc);
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) out_torque[3 * p + c] = (float)((double)a.accum[a.acc_stride * p + 3 + c] * w2);
    }
}

// debug: primary-hit triangle (original index) of every ray of the listed pairs
template <int MODE>
__global__ void __launch_bounds__(TRACE_THREADS) first_hit_kernel(const TraceArgs a, int *out_prim)
{
    __shared__ int s_stack[MODE == MODE_BVH ? STACK_SMEM * TRACE_THREADS : 1];
    const long long total = a.n_pairs * a.N;
    for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < total;
         r += (long long)gridDim.x * blockDim.x) {
        const long long p = r / a.N;
        const uint32_t i = (uint32_t)(r - p * a.N);
        int k, j;
        pair_of(a, p, k, j);
        const Emitter em = make_emitter(a.sun_dirs, j, a.dz.box[2 * k], a.dz.box[2 * k + 1]);
        int best = -1;
        if (em.Ae > 0.0f) {
            const long long tbase = a.dz.tri_off[k];
            const int T = (int)(a.dz.tri_off[k + 1] - tbase);
            RayGen g;
            g.j = (uint32_t)j; g.k = (uint32_t)k; g.key0 = a.key0; g.key1 = a.key1; g.sampler = a.sampler; g.xc = f3(0.f, 0.f, 0.f);
            g.inv_nx = 1.0f / (float)(1u << ((a.log2N + 1) >> 1));
            g.inv_ny = 1.0f / (float)(1u << (a.log2N >> 1));
            float3 o;
            make_ray(em, g, i, o);
            float tbest = FLT_MAX;
            unsigned nb = 0, nt = 0;
            if (MODE == MODE_BVH)
                closest_bvh<false>(SRP_TRAV_NODES(a.dz, tbase), a.dz.tri + 3 * tbase, o, em.s, -1, tbest, best,
                                   s_stack + threadIdx.x, nb, nt);
            else
                closest_brute<false>(a.dz.tri + 3 * tbase, T, o, em.s, -1, tbest, best, nt);
            if (best >= 0) best = a.dz.perm[tbase + best];
        }
        out_prim[r] = best;
    }
}


} // namespace

int srp_perray_blocks_per_sm(bool brute)
{
    return brute ? blocks_per_sm(trace_kernel<MODE_BRUTE_SMEM, false, false, false, false>) : blocks_per_sm(bvh_trace_kernel<false, false, false, false, false>);
}

// mode: MODE_BVH (0 is BRUTE_SMEM, 1 BVH, 2 BRUTE_GLOBAL -- the enum of trace_common.cuh)
cudaError_t srp_launch_perray(const TraceArgs &a, int mode, bool instrumented, int num_sms, cudaStream_t stream)
{
    const size_t dyn_smem = 0;
    if (mode == MODE_BRUTE_GLOBAL) return SRP_LAUNCH3(trace_kernel, MODE_BRUTE_GLOBAL,);
    if (mode == MODE_BRUTE_SMEM) return SRP_LAUNCH3(trace_kernel, MODE_BRUTE_SMEM,);
    return a.dz.esc ? SRP_LAUNCH3(bvh_trace_kernel, true,) : SRP_LAUNCH3(bvh_trace_kernel, false,);
}

cudaError_t srp_launch_finalize(const TraceArgs &a, float *out_forces, float *out_torques, cudaStream_t stream)
{
    finalize_kernel<<<(unsigned)((a.n_pairs + 255) / 256), 256, 0, stream>>>(a, out_forces, out_torques);
    return cudaGetLastError();
}

cudaError_t srp_launch_first_hits(const TraceArgs &a, int method, int *out_prim, cudaStream_t stream)
{
    const long long total = a.n_pairs * a.N;
    long long blocks = (total + TRACE_THREADS - 1) / TRACE_THREADS;
    if (blocks > 148 * 64) blocks = 148 * 64;
    if (method == 0 && a.dz.has_bvh)
        first_hit_kernel<MODE_BVH><<<(unsigned)blocks, TRACE_THREADS, 0, stream>>>(a, out_prim);
    else
        first_hit_kernel<MODE_BRUTE_GLOBAL><<<(unsigned)blocks, TRACE_THREADS, 0, stream>>>(a, out_prim);
    return cudaGetLastError();
}
