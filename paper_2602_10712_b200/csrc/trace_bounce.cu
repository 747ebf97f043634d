// trace_bounce.cu -- bounce_trace_kernel (S4-S7 for everything the beam kernel could not resolve as a beam):
// per-ray BVH traversal of the rays in the ray queue -- bounce rays, and the primaries of groups whose beam lists
// overflowed -- shading of their hits, and the photons that go on from there (all depths share one loop).
// A kernel of its own (it was a phase of the beam kernel in round 1) so that it has its own register budget,
// occupancy and instruction-cache footprint: incoherent traversal hides its load latency with resident warps,
// the beam kernel needs registers and shared memory for its lists instead (profiles/r2_*).
#include "trace_common.cuh"

namespace {

#ifndef BOUNCE_BLOCKS_PER_SM
#define BOUNCE_BLOCKS_PER_SM 8
#endif
#ifndef BOUNCE_STACK_DEF
#define BOUNCE_STACK_DEF 12
#endif
constexpr int BOUNCE_STACK = BOUNCE_STACK_DEF;   // per-thread stack entries in shared memory; deeper ones in local memory
constexpr int HITQ = 64;                 // queued hits per warp (shaded 32 at a time, converged) and photons that go on after
                                         // such a hit, waiting for a free lane, in one array: hits from the front, photons
                                         // from the back (a warp holds <= 63 photons in lanes and queues together)
#ifndef BOUNCE_BATCH_DEF
#define BOUNCE_BATCH_DEF 256
#endif
constexpr uint32_t BOUNCE_BATCH = BOUNCE_BATCH_DEF;      // rays a warp claims from the queue at a time
#ifndef DRAIN_ACTIVE_MIN_DEF
#define DRAIN_ACTIVE_MIN_DEF 24
#endif
constexpr int DRAIN_ACTIVE_MIN = DRAIN_ACTIVE_MIN_DEF;   // leave the traversal loop to refill when fewer lanes are busy

template <bool INSTR>
struct BounceSmem {                 // per warp
    int stack[BOUNCE_STACK * 32];   // per-thread traversal stacks, thread-interleaved
    uint32_t hq[11][HITQ];          // queued hits [0, nhit): o, d, i, p, sd, triangle, t; photons that go on
                                    // [HITQ - nlq, HITQ), last one first: o, d, i, p, sd.  Less shared memory = more L1
                                    // for the nodes: 8 blocks leave 92 KB instead of 28 KB
    unsigned long long hsig[INSTR ? HITQ : 1];
};

template <bool INSTR, bool TORQUE, bool GLOSSY, bool ANALOG>
__global__ void __launch_bounds__(TRACE_THREADS, BOUNCE_BLOCKS_PER_SM)
bounce_trace_kernel(const TraceArgs a)
{
    __shared__ BounceSmem<INSTR> s_w[TRACE_WARPS];
    __shared__ unsigned s_hist[TRACE_WARPS][16];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    if (lane < 16) s_hist[warp][lane] = 0;
    __syncwarp();
    BounceSmem<INSTR> &W = s_w[warp];
    LaneCounters cn = { 0, 0, 0, 0, 0, 0, 0, 0 };
    const float inv_nx = 1.0f / (float)(1u << ((a.log2N + 1) >> 1)), inv_ny = 1.0f / (float)(1u << (a.log2N >> 1));
    const uint32_t n_queued = *(volatile unsigned *)a.rq_ctr;          // the beam kernel has finished: stable

    int nhit = 0, nlq = 0;                                             // warp-uniform
    uint32_t gb_next = 0, gb_end = 0;                                  // the warp's claimed slice of the queue
    bool g_more = n_queued != 0u;

    // ---- S5-S7 for <= 32 queued hits, converged; photons that go on wait in lq for a free lane ----
    auto shade_batch = [&]() {
        const int take = nhit < 32 ? nhit : 32;
        int fate = -1, src = -1, depth = 0;
        float3 o = f3(0, 0, 0), d = f3(0, 0, 1);
        uint32_t i = 0, p = 0;
        unsigned long long sig = 0;
        if (lane < take) {
            const int e = nhit - take + lane;
            o = f3(__uint_as_float(W.hq[0][e]), __uint_as_float(W.hq[1][e]), __uint_as_float(W.hq[2][e]));
            d = f3(__uint_as_float(W.hq[3][e]), __uint_as_float(W.hq[4][e]), __uint_as_float(W.hq[5][e]));
            i = W.hq[6][e]; p = W.hq[7][e];
            depth = (int)(W.hq[8][e] >> 27);
            const int best = (int)W.hq[9][e];
            const float t = __uint_as_float(W.hq[10][e]);
            int k, j;
            pair_of32(a, p, k, j);
            const long long tb = a.dz.tri_off[k];
            const float4 *lt = a.dz.tri + 3 * tb;
            RayGen g;
            g.j = (uint32_t)j; g.k = (uint32_t)k; g.key0 = a.key0; g.key1 = a.key1; g.sampler = 0; set_torque<TORQUE>(g, a, k);
            g.inv_nx = inv_nx; g.inv_ny = inv_ny;
            atomicAdd(&s_hist[warp][depth], 1u);
            if (INSTR) sig = W.hsig[e] * 1000003ULL + (unsigned long long)(a.dz.perm[tb + best] + 1);
            float3 dep = f3(0, 0, 0), dep_t = f3(0, 0, 0);
            fate = shade<TORQUE, 0u, GLOSSY, ANALOG ? 1 : 0>(__ldg(lt + 3 * best), __ldg(lt + 3 * best + 1), __ldg(lt + 3 * best + 2), t, best, g, i, a.B,
                         a.deposit, o, d, src, depth, dep, dep_t, a.dz.esc, tb + best, a.dz.shin);
            if (fate == SHADE_ESCAPES) { cn.segments++; cn.escaped++; cn.mesc++; }
            if (fate == SHADE_ABSORBED) cn.absorbed++;
            if (fate == SHADE_CAPPED) cn.capped++;
            // S7: these hits are ~1 % of the segments; one fixed-point atomic per component and hit
            unsigned long long *dst = (unsigned long long *)(a.accum + a.acc_stride * (long long)p);
            if (dep.x != 0.0f) atomicAdd(dst + 0, (unsigned long long)__double2ll_rn((double)dep.x * a.acc_scale));
            if (dep.y != 0.0f) atomicAdd(dst + 1, (unsigned long long)__double2ll_rn((double)dep.y * a.acc_scale));
            if (dep.z != 0.0f) atomicAdd(dst + 2, (unsigned long long)__double2ll_rn((double)dep.z * a.acc_scale));
            if (TORQUE) {
                if (dep_t.x != 0.0f) atomicAdd(dst + 3, (unsigned long long)__double2ll_rn((double)dep_t.x * a.acc_scale));
                if (dep_t.y != 0.0f) atomicAdd(dst + 4, (unsigned long long)__double2ll_rn((double)dep_t.y * a.acc_scale));
                if (dep_t.z != 0.0f) atomicAdd(dst + 5, (unsigned long long)__double2ll_rn((double)dep_t.z * a.acc_scale));
            }
            if (INSTR && fate != SHADE_CONTINUE && a.sig_out) a.sig_out[(long long)p * a.N + i] = sig;
        }
        nhit -= take;
        const unsigned mc = __ballot_sync(FULL, fate == SHADE_CONTINUE);
        SRP_CHECK(nhit + nlq + __popc(mc) <= HITQ, "photon queue");
        __syncwarp();                                                // the hits of this batch have been read: their slots are free
        if (fate == SHADE_CONTINUE) {
            const int e = HITQ - 1 - (nlq + __popc(mc & lt_mask));
            W.hq[0][e] = __float_as_uint(o.x); W.hq[1][e] = __float_as_uint(o.y); W.hq[2][e] = __float_as_uint(o.z);
            W.hq[3][e] = __float_as_uint(d.x); W.hq[4][e] = __float_as_uint(d.y); W.hq[5][e] = __float_as_uint(d.z);
            W.hq[6][e] = i; W.hq[7][e] = p; W.hq[8][e] = ((uint32_t)depth << 27) | (uint32_t)src;
            if (INSTR) W.hsig[e] = sig;
        }
        nlq += __popc(mc);
        __syncwarp();
    };

    // ---- per-ray traversal (S4 for incoherent rays, S6): a lane whose ray has ended takes the next ray at once ----
    constexpr int STRIDE = 32, NSMEM = BOUNCE_STACK;
    int *s_stack = W.stack + lane;
    int ovf[STACK_OVF];
    bool has = false;
    int cur = CUR_DONE, sp = 0, best = -1, src = -1;
    float tbest = FLT_MAX;
    float3 o = f3(0, 0, 0), d = f3(0, 0, 1);
    float idx = 0.f, idy = 0.f, idz = 0.f, oxi = 0.f, oyi = 0.f, ozi = 0.f;
    uint32_t ri = 0, rp = 0, rsd = 0;
    unsigned long long rsig = 0;
    const float4 *ln = a.dz.nodes, *lt = a.dz.tri;
    unsigned nt = 0;
    auto start_ray = [&]() {
        int k, j;
        pair_of32(a, rp, k, j);
        const long long tb = a.dz.tri_off[k];
        ln = SRP_TRAV_NODES(a.dz, tb); lt = a.dz.tri + 3 * tb;
        const uint32_t s27 = rsd & SRC_NONE;
        src = s27 == SRC_NONE ? -1 : (int)s27;
        idx = safe_rcp(d.x); idy = safe_rcp(d.y); idz = safe_rcp(d.z);
        oxi = o.x * idx; oyi = o.y * idy; ozi = o.z * idz;
        has = true; cur = 0; sp = 0; tbest = FLT_MAX; best = -1;
        if ((rsd >> 27) != 0u) cn.segments++;                    // primaries were counted when generated
    };
    for (;;) {
        // lanes without a ray: first the photons waiting in lq, then the warp's slice of the queue
        unsigned idle = __ballot_sync(FULL, !has);
        if (idle != 0u && nlq > 0) {
            const int nidle = __popc(idle), take = nidle < nlq ? nidle : nlq;
            const int rank = __popc(idle & lt_mask);
            if (!has && rank < take) {
                const int e = HITQ - 1 - (nlq - take + rank);
                o = f3(__uint_as_float(W.hq[0][e]), __uint_as_float(W.hq[1][e]), __uint_as_float(W.hq[2][e]));
                d = f3(__uint_as_float(W.hq[3][e]), __uint_as_float(W.hq[4][e]), __uint_as_float(W.hq[5][e]));
                ri = W.hq[6][e]; rp = W.hq[7][e]; rsd = W.hq[8][e];
                if (INSTR) rsig = W.hsig[e];
                start_ray();
            }
            nlq -= take;
            __syncwarp();
            idle = __ballot_sync(FULL, !has);
        }
        if (idle != 0u && (gb_next != gb_end || g_more)) {
            if (gb_next == gb_end) {                                 // claim the next slice
                uint32_t b = 0;
                if (lane == 0) b = atomicAdd(a.rq_ctr + 1, BOUNCE_BATCH);
                b = __shfl_sync(FULL, b, 0);
                if (b >= n_queued) g_more = false;
                else { gb_next = b; gb_end = b + BOUNCE_BATCH < n_queued ? b + BOUNCE_BATCH : n_queued; }
            }
            const uint32_t navail = gb_end - gb_next;
            if (navail != 0u) {
                const uint32_t rank = (uint32_t)__popc(idle & lt_mask);
                if (!has && rank < navail) {
                    rq_load<INSTR>(a, gb_next + rank, o, d, ri, rp, rsd, rsig);
                    if (rsd != RQ_DEAD) start_ray();                 // a slot a beam warp reserved and did not fill
                }
                const uint32_t want = (uint32_t)__popc(idle);
                gb_next += want < navail ? want : navail;
            }
        }
        const bool waiting = nlq > 0 || gb_next != gb_end || g_more;     // rays a free lane could take
        if (!__any_sync(FULL, has)) {
            if (nhit > 0) { shade_batch(); continue; }                  // shading may put photons into lq
            if (waiting) continue;
            break;
        }
        // traverse until every lane is done, or enough lanes are free and rays are waiting
        for (;;) {
#pragma unroll 1
            for (int steps = 0; steps < NODE_RUN_CAP && (unsigned)cur < (unsigned)CUR_DONE; ++steps) {
                if (INSTR) cn.n_box += 2;
                cur = bvh_node_step<STRIDE, NSMEM>(ln, cur, sp, s_stack, ovf, idx, idy, idz, oxi, oyi, ozi, tbest);
            }
            if (cur < 0) cur = bvh_leaf_step<STRIDE, NSMEM>(lt, cur, sp, s_stack, ovf, o, d, src, tbest, best, nt);
            const unsigned act = __ballot_sync(FULL, cur != CUR_DONE);
            if (act == 0u || (waiting && __popc(act) < DRAIN_ACTIVE_MIN)) break;
        }
        // retire the rays that ended
        const bool fin = has && cur == CUR_DONE;
        const bool hit = fin && best >= 0;
        if (fin && !hit) {
            if ((rsd >> 27) == 0u) cn.pmiss++; else cn.escaped++;
            if (INSTR && a.sig_out) a.sig_out[(long long)rp * a.N + ri] = rsig;
        }
        const unsigned mh = __ballot_sync(FULL, hit);
        SRP_CHECK(nhit + nlq + __popc(mh) <= HITQ, "hit queue");
        if (hit) {
            const int e = nhit + __popc(mh & lt_mask);
            W.hq[0][e] = __float_as_uint(o.x); W.hq[1][e] = __float_as_uint(o.y); W.hq[2][e] = __float_as_uint(o.z);
            W.hq[3][e] = __float_as_uint(d.x); W.hq[4][e] = __float_as_uint(d.y); W.hq[5][e] = __float_as_uint(d.z);
            W.hq[6][e] = ri; W.hq[7][e] = rp; W.hq[8][e] = rsd;
            W.hq[9][e] = (uint32_t)best; W.hq[10][e] = __float_as_uint(tbest);
            if (INSTR) W.hsig[e] = rsig;
        }
        nhit += __popc(mh);
        if (fin) has = false;
        __syncwarp();
        // A warp holds at most 63 photons (new ones enter only into free lanes, with no photon waiting and < 32 hits
        // queued), so the two ends of the queue cannot meet.
        if (nhit >= 32) shade_batch();
    }
    if (INSTR) cn.n_tri += nt;
    flush_counters<INSTR>(a, cn, s_hist[warp], lane);
    // the last warp to finish empties the queue for the next launch of the beam kernel
    __syncwarp();
    if (lane == 0) {
        __threadfence();
        if (atomicAdd(a.rq_ctr + 2, 1u) == gridDim.x * TRACE_WARPS - 1u) {
            if (n_queued != 0u) {                                   // atomics: the pipelines' bounce kernels may run side by side
                atomicAdd((unsigned long long *)&a.stats->queued_rays, (unsigned long long)n_queued);
                atomicAdd((unsigned long long *)&a.stats->loop_rounds, 1ULL);
                atomicAdd(a.rounds_total, 1ULL);
            }
            a.rq_ctr[0] = 0u; a.rq_ctr[1] = 0u; a.rq_ctr[2] = 0u;
            __threadfence();
        }
    }
}

// Loop condition of the beam / bounce loop (a conditional WHILE node of a CUDA graph): go round again while tiles
// are left.  Runs after the bounce kernel, which has emptied the queue.
__global__ void loop_cond_kernel(cudaGraphConditionalHandle handle, const unsigned long long *work_counter,
                                 unsigned long long n_tiles)
{
    cudaGraphSetConditional(handle, *work_counter < n_tiles ? 1u : 0u);
}

template <typename K>
cudaError_t launch_bounce(K kernel, const TraceArgs &a, int num_sms, cudaStream_t stream)
{
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, TRACE_THREADS, 0);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    e = prefer_l1(kernel, per_sm, 0);
    if (e != cudaSuccess) return e;
    kernel<<<(unsigned)(num_sms * per_sm), TRACE_THREADS, 0, stream>>>(a);
    return cudaGetLastError();
}

#define SRP_BOUNCE_A(I_, T_, G_) (a.deposit ? launch_bounce(bounce_trace_kernel<I_, T_, G_, true>, a, num_sms, stream) \
                                            : launch_bounce(bounce_trace_kernel<I_, T_, G_, false>, a, num_sms, stream))
#define SRP_BOUNCE_G(I_, T_) (a.dz.shin ? SRP_BOUNCE_A(I_, T_, true) : SRP_BOUNCE_A(I_, T_, false))

} // namespace

cudaError_t srp_launch_loop_cond(cudaGraphConditionalHandle handle, const TraceArgs &a, cudaStream_t stream)
{
    loop_cond_kernel<<<1, 1, 0, stream>>>(handle, a.work_counter, a.tile_end - a.tile_begin);
    return cudaGetLastError();
}

cudaError_t srp_launch_bounce(const TraceArgs &a, bool instrumented, int num_sms, cudaStream_t stream)
{
    return instrumented ? SRP_BOUNCE_G(true, false) : a.torque ? SRP_BOUNCE_G(false, true) : SRP_BOUNCE_G(false, false);
}
