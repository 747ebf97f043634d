// trace_beam.cu -- beam_trace_kernel (S2-S7 for designs with a BVH, stratified sampler): the primaries of a tile
// are traced as beams, everything else through a per-warp ray pool.
#include "trace_common.cuh"

namespace {

// ---- the beam trace kernel: coherent primaries as beams, bounce rays one by one ----
// The primaries of a pair are parallel and, in the stratified sampler, ray i sits in cell
// Morton(i) of the emitter grid, so every aligned block of 2^b consecutive rays is a rectangle of
// cells -- a BEAM with a rectangular cross-section.  A warp walks the BVH once per beam instead of
// once per ray (BVH "packet"/beam traversal; the tree and the hit definition are unchanged):
//   tile      (<= 8192 rays): frontier descent from the root, all lanes testing different nodes
//             against the tile's rectangle, until the frontier holds > 32 nodes -> entry list.
//             Nothing overlaps: the whole tile is primary misses, no ray is generated.
//   sub-block (256 rays, 16 x 16 cells): descent from the entry list to the leaves -> candidate
//             triangles (<= BEAM_CMAX), each set up ONCE as three 2-D edge functions and a depth
//             plane in the emitter frame (the ray-triangle test of a ray parallel to the frame's
//             axis: inside <=> the three edge functions are >= 0, same inclusive rule as O-step 4).
//   group     (32 rays, 8 x 4 cells, one per lane): the candidates whose edge functions admit the
//             group's rectangle are listed; an empty list resolves 32 misses without Philox;
//             otherwise every lane tests ITS ray against the same short list, all 32 lanes
//             converged, operands broadcast from shared memory.
// Bounce rays are incoherent: they go to the warp's ray pool and through per-ray stack traversal
// (drain(), below).  A sub-block whose lists overflow is halved; a single group that still
// overflows (a beam along an edge-on panel, a bundle of thin facets) sends its 32 primaries to the
// pool as well, so any input is handled.
#ifndef BEAM_BLOCKS_PER_SM
#define BEAM_BLOCKS_PER_SM 5
#endif
#ifndef BEAM_SB_DEF
#define BEAM_SB_DEF 256
#endif
constexpr int BEAM_SB = BEAM_SB_DEF;        // rays per sub-block
#ifndef BEAM_CMAX_DEF
#define BEAM_CMAX_DEF 160
#endif
constexpr int BEAM_CMAX = BEAM_CMAX_DEF;      // candidate triangles per sub-block
#ifndef BEAM_QN_DEF
#define BEAM_QN_DEF 192
#endif
constexpr int BEAM_QN = BEAM_QN_DEF;        // node queue of the sub-block descent
constexpr int BEAM_EN = 64;         // tile entry list: internal nodes
constexpr int BEAM_EL = 96;         // tile entry list: leaf links (<= 32 when a level starts, + 2 x 32 in that level)
constexpr int BEAM_STACK = 16;      // per-thread stack entries in shared memory (bounce rays)

struct BeamFrame {                  // warp-uniform per pair
    float3 uh, vh, auh, avh;        // u/2, v/2 and their absolute values
    float csu, csv;                 // cell size along u and v
    float margin;                   // bound of the fp32 projection error of a box
};

// Does the box's projection on the emitter plane meet the rectangle [0,wu] x [0,wv] of the local
// frame whose origin projects to (offu, offv)?  NaN (the empty-box sentinel) compares false.
__device__ __forceinline__ bool beam_box(const BeamFrame &f, float offu, float offv, float wu, float wv,
                                         float lox, float loy, float loz, float hix, float hiy, float hiz)
{
    const float sx = lox + hix, sy = loy + hiy, sz = loz + hiz;
    const float dx = hix - lox, dy = hiy - loy, dz = hiz - loz;
    const float pu = fmaf(sx, f.uh.x, fmaf(sy, f.uh.y, sz * f.uh.z)) - offu;
    const float pv = fmaf(sx, f.vh.x, fmaf(sy, f.vh.y, sz * f.vh.z)) - offv;
    const float ru = fmaf(dx, f.auh.x, fmaf(dy, f.auh.y, dz * f.auh.z)) + f.margin;
    const float rv = fmaf(dx, f.avh.x, fmaf(dy, f.avh.y, dz * f.avh.z)) + f.margin;
    return (pu + ru >= 0.0f) && (pu - ru <= wu) && (pv + rv >= 0.0f) && (pv - rv <= wv);
}

// One node against a beam: which children overlap, and their links.
template <bool INSTR>
__device__ __forceinline__ void beam_node(const float4 *__restrict__ nodes, int node, const BeamFrame &f, float offu,
                                          float offv, float wu, float wv, bool &h0, bool &h1, int &l0, int &l1,
                                          unsigned &n_box)
{
    h0 = h1 = false; l0 = l1 = 0;
    if (node < 0) return;
    const float4 n0 = __ldg(nodes + 4 * node), n1 = __ldg(nodes + 4 * node + 1), n2 = __ldg(nodes + 4 * node + 2),
                 n3 = __ldg(nodes + 4 * node + 3);
    h0 = beam_box(f, offu, offv, wu, wv, n0.x, n0.y, n0.z, n0.w, n1.x, n1.y);
    h1 = beam_box(f, offu, offv, wu, wv, n1.z, n1.w, n2.x, n2.y, n2.z, n2.w);
    l0 = __float_as_int(n3.x); l1 = __float_as_int(n3.y);
    if (INSTR) n_box += 2;
}

// Appends the triangles of up to two leaves per lane to the candidate list (warp scan of the
// counts, so the order is deterministic).  Returns false if the list would overflow.
__device__ __forceinline__ bool beam_push_tris(int *cid, int &ncand, int first0, int cnt0, int first1, int cnt1,
                                               int lane)
{
    const int c = cnt0 + cnt1;
    int incl = c;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const int t = __shfl_up_sync(FULL, incl, off);
        if (lane >= off) incl += t;
    }
    const int total = __shfl_sync(FULL, incl, 31);
    if (ncand + total > BEAM_CMAX) return false;
    int pos = ncand + incl - c;
    for (int t = 0; t < cnt0; ++t) cid[pos++] = first0 + t;
    for (int t = 0; t < cnt1; ++t) cid[pos++] = first1 + t;
    ncand += total;
    return true;
}


// ---- per-warp ray pool (global memory ring) ----
// Rays that are not resolved by a beam -- bounce rays, and primaries of a group whose lists
// overflowed -- are appended to the warp's private ring in global memory (L2-resident) and traced
// later, many tiles' worth at a time, by the per-ray traversal loop of drain(): a lane whose ray
// has ended takes the next ray of the pool at once, so lanes stay busy although path lengths
// differ widely (persistent "while-while" traversal with dynamic fetch).  Hits are not shaded where
// they are found: they are queued in shared memory and shaded 32 at a time, converged.
// Entry = 9 words (origin, direction, ray index i, pair index p, src | depth << 27), plus the
// 64-bit path signature in the instrumented build; field-major so appends and fetches coalesce.
constexpr int POOL_FIELDS = 9;
constexpr int POOL_FIELDS_INSTR = 11;
#ifndef POOL_HIGH_DEF
#define POOL_HIGH_DEF 4096
#endif
constexpr int POOL_HIGH = POOL_HIGH_DEF;          // drain when the pool holds at least this many rays
constexpr int HITQ = 64;                 // queued hits per warp
#ifndef DRAIN_ACTIVE_MIN_DEF
#define DRAIN_ACTIVE_MIN_DEF 24
#endif
constexpr int DRAIN_ACTIVE_MIN = DRAIN_ACTIVE_MIN_DEF;     // leave the traversal loop to refill when fewer lanes are busy
constexpr uint32_t SRC_NONE = 0x07ffffffu;

struct Pool {
    unsigned *base;
    uint32_t cap, mask, head, tail;      // head/tail count rays; position = counter & mask
};
__device__ __forceinline__ void pool_st(const Pool &q, int field, uint32_t pos, uint32_t v)
{
    __stcg(q.base + (size_t)field * q.cap + (pos & q.mask), v);
}
__device__ __forceinline__ uint32_t pool_ld(const Pool &q, int field, uint32_t pos)
{
    return __ldcg(q.base + (size_t)field * q.cap + (pos & q.mask));
}

struct BeamSmem {                   // per warp; beam structures and drain structures are never live together
    union {
        struct {
            float4 eq[3 * BEAM_CMAX];       // (A0,B0,C0,Wu) (A1,B1,C1,Wv) (A2,B2,C2,Wc) per candidate
            int cid[BEAM_CMAX];             // candidate -> sorted triangle index
            int enode[BEAM_EN];
            int eleaf[BEAM_EL];
            int nq[BEAM_QN];
            unsigned char glist[BEAM_CMAX];
        } b;
        struct {
            int stack[BEAM_STACK * 32];     // per-thread traversal stacks, thread-interleaved
            uint32_t hq[11][HITQ];          // queued hits: o, d, i, p, sd, triangle, t
        } s;
    } u;
};

template <bool INSTR, bool TORQUE, bool GLOSSY, bool ANALOG>
__global__ void __launch_bounds__(TRACE_THREADS, BEAM_BLOCKS_PER_SM)
beam_trace_kernel(const TraceArgs a)
{
    __shared__ BeamSmem s_w[TRACE_WARPS];
    __shared__ unsigned long long s_hsig[INSTR ? TRACE_WARPS * HITQ : 1];
    __shared__ unsigned s_hist[TRACE_WARPS][16];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    if (lane < 16) s_hist[warp][lane] = 0;
    __syncwarp();
    BeamSmem &W = s_w[warp];
    unsigned long long *hsig = s_hsig + (INSTR ? warp * HITQ : 0);
    LaneCounters cn = { 0, 0, 0, 0, 0, 0, 0, 0 };
    BeamCounters bc = { 0, 0, 0, 0, 0, 0, 0, 0 };
    const unsigned long long total_tiles = (unsigned long long)a.n_pairs * a.tiles_per_pair;
    const uint32_t ldx = compact_even_bits((uint32_t)lane), ldy = compact_even_bits((uint32_t)lane >> 1);
    const float inv_nx = 1.0f / (float)(1u << ((a.log2N + 1) >> 1)), inv_ny = 1.0f / (float)(1u << (a.log2N >> 1));
    Pool pool;
    pool.cap = (uint32_t)a.pool_cap; pool.mask = pool.cap - 1u; pool.head = pool.tail = 0u;
    pool.base = a.pool + (size_t)(blockIdx.x * TRACE_WARPS + warp) * (size_t)(INSTR ? POOL_FIELDS_INSTR : POOL_FIELDS) * pool.cap;

    // Appends this lane's ray (if `push`) to the pool; warp-wide call.
    auto pool_push = [&](bool push, const float3 &o, const float3 &d, uint32_t i, uint32_t p, uint32_t sd,
                         unsigned long long sig) {
        const unsigned m = __ballot_sync(FULL, push);
        if (push) {
            const uint32_t pos = pool.tail + (uint32_t)__popc(m & lt_mask);
            pool_st(pool, 0, pos, __float_as_uint(o.x)); pool_st(pool, 1, pos, __float_as_uint(o.y));
            pool_st(pool, 2, pos, __float_as_uint(o.z)); pool_st(pool, 3, pos, __float_as_uint(d.x));
            pool_st(pool, 4, pos, __float_as_uint(d.y)); pool_st(pool, 5, pos, __float_as_uint(d.z));
            pool_st(pool, 6, pos, i); pool_st(pool, 7, pos, p); pool_st(pool, 8, pos, sd);
            if (INSTR) { pool_st(pool, 9, pos, (uint32_t)sig); pool_st(pool, 10, pos, (uint32_t)(sig >> 32)); }
        }
        pool.tail += (uint32_t)__popc(m);
        SRP_CHECK(pool.tail - pool.head <= pool.cap, "ray pool");
    };

    // ---- S5-S7 for <= 32 queued hits, converged; survivors go back to the pool ----
    int nhit = 0;                                                  // warp-uniform
    auto shade_batch = [&]() {
        const int take = nhit < 32 ? nhit : 32;
        int fate = -1, src = -1, depth = 0;
        float3 o = f3(0, 0, 0), d = f3(0, 0, 1);
        uint32_t i = 0, p = 0;
        unsigned long long sig = 0;
        if (lane < take) {
            const int e = nhit - take + lane;
            o = f3(__uint_as_float(W.u.s.hq[0][e]), __uint_as_float(W.u.s.hq[1][e]), __uint_as_float(W.u.s.hq[2][e]));
            d = f3(__uint_as_float(W.u.s.hq[3][e]), __uint_as_float(W.u.s.hq[4][e]), __uint_as_float(W.u.s.hq[5][e]));
            i = W.u.s.hq[6][e]; p = W.u.s.hq[7][e];
            depth = (int)(W.u.s.hq[8][e] >> 27);
            const int best = (int)W.u.s.hq[9][e];
            const float t = __uint_as_float(W.u.s.hq[10][e]);
            int k, j;
            pair_of32(a, p, k, j);
            const long long tb = a.dz.tri_off[k];
            const float4 *lt = a.dz.tri + 3 * tb;
            RayGen g;
            g.j = (uint32_t)j; g.k = (uint32_t)k; g.key0 = a.key0; g.key1 = a.key1; g.sampler = 0; set_torque<TORQUE>(g, a, k);
            g.inv_nx = inv_nx; g.inv_ny = inv_ny;
            atomicAdd(&s_hist[warp][depth], 1u);
            if (INSTR) sig = hsig[e] * 1000003ULL + (unsigned long long)(a.dz.perm[tb + best] + 1);
            float3 dep = f3(0, 0, 0), dep_t = f3(0, 0, 0);
            fate = shade<TORQUE, 0u, GLOSSY, ANALOG ? 1 : 0>(__ldg(lt + 3 * best), __ldg(lt + 3 * best + 1), __ldg(lt + 3 * best + 2), t, best, g, i, a.B,
                         a.deposit, o, d, src, depth, dep, dep_t, a.dz.esc, tb + best, a.dz.shin);
            if (fate == SHADE_ESCAPES) { cn.segments++; cn.escaped++; cn.mesc++; }
            if (fate == SHADE_ABSORBED) cn.absorbed++;
            if (fate == SHADE_CAPPED) cn.capped++;
            unsigned long long *dst = (unsigned long long *)(a.accum + a.acc_stride * (long long)p);
            if (dep.x != 0.0f) atomicAdd(dst + 0, (unsigned long long)__double2ll_rn((double)dep.x * SRP_ACC_SCALE));
            if (dep.y != 0.0f) atomicAdd(dst + 1, (unsigned long long)__double2ll_rn((double)dep.y * SRP_ACC_SCALE));
            if (dep.z != 0.0f) atomicAdd(dst + 2, (unsigned long long)__double2ll_rn((double)dep.z * SRP_ACC_SCALE));
            if (TORQUE) {
                if (dep_t.x != 0.0f) atomicAdd(dst + 3, (unsigned long long)__double2ll_rn((double)dep_t.x * SRP_ACC_SCALE));
                if (dep_t.y != 0.0f) atomicAdd(dst + 4, (unsigned long long)__double2ll_rn((double)dep_t.y * SRP_ACC_SCALE));
                if (dep_t.z != 0.0f) atomicAdd(dst + 5, (unsigned long long)__double2ll_rn((double)dep_t.z * SRP_ACC_SCALE));
            }
            if (INSTR && fate != SHADE_CONTINUE && a.sig_out) a.sig_out[(long long)p * a.N + i] = sig;
        }
        nhit -= take;
        __syncwarp();
        pool_push(fate == SHADE_CONTINUE, o, d, i, p, ((uint32_t)depth << 27) | (uint32_t)src, sig);
    };

    // ---- per-ray traversal of everything in the pool (S4 for incoherent rays, S6) ----
    auto drain = [&]() {
        constexpr int STRIDE = 32, NSMEM = BEAM_STACK;
        int *s_stack = W.u.s.stack + lane;
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
        for (;;) {
            // lanes without a ray take the next rays of the pool
            const unsigned idle = __ballot_sync(FULL, !has);
            uint32_t navail = pool.tail - pool.head;
            if (idle != 0u && navail != 0u) {
                const uint32_t rank = (uint32_t)__popc(idle & lt_mask);
                if (!has && rank < navail) {
                    const uint32_t pos = pool.head + rank;
                    o = f3(__uint_as_float(pool_ld(pool, 0, pos)), __uint_as_float(pool_ld(pool, 1, pos)),
                           __uint_as_float(pool_ld(pool, 2, pos)));
                    d = f3(__uint_as_float(pool_ld(pool, 3, pos)), __uint_as_float(pool_ld(pool, 4, pos)),
                           __uint_as_float(pool_ld(pool, 5, pos)));
                    ri = pool_ld(pool, 6, pos); rp = pool_ld(pool, 7, pos); rsd = pool_ld(pool, 8, pos);
                    if (INSTR) rsig = (unsigned long long)pool_ld(pool, 9, pos) | ((unsigned long long)pool_ld(pool, 10, pos) << 32);
                    int k, j;
                    pair_of32(a, rp, k, j);
                    const long long tb = a.dz.tri_off[k];
                    ln = a.dz.nodes + 4 * tb; lt = a.dz.tri + 3 * tb;
                    const uint32_t s27 = rsd & SRC_NONE;
                    src = s27 == SRC_NONE ? -1 : (int)s27;
                    idx = safe_rcp(d.x); idy = safe_rcp(d.y); idz = safe_rcp(d.z);
                    oxi = o.x * idx; oyi = o.y * idy; ozi = o.z * idz;
                    has = true; cur = 0; sp = 0; tbest = FLT_MAX; best = -1;
                    if ((rsd >> 27) != 0u) cn.segments++;            // primaries were counted when generated
                }
                const uint32_t want = (uint32_t)__popc(idle);
                pool.head += want < navail ? want : navail;
                navail = pool.tail - pool.head;
            }
            if (!__any_sync(FULL, has)) {
                if (nhit > 0) { shade_batch(); continue; }          // shading may put rays back
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
                if (act == 0u || (navail != 0u && __popc(act) < DRAIN_ACTIVE_MIN)) break;
            }
            // retire the rays that ended
            const bool fin = has && cur == CUR_DONE;
            const bool hit = fin && best >= 0;
            if (fin && !hit) {
                if ((rsd >> 27) == 0u) cn.pmiss++; else cn.escaped++;
                if (INSTR && a.sig_out) a.sig_out[(long long)rp * a.N + ri] = rsig;
            }
            const unsigned mh = __ballot_sync(FULL, hit);
            SRP_CHECK(nhit + __popc(mh) <= HITQ, "hit queue");
            if (hit) {
                const int e = nhit + __popc(mh & lt_mask);
                W.u.s.hq[0][e] = __float_as_uint(o.x); W.u.s.hq[1][e] = __float_as_uint(o.y); W.u.s.hq[2][e] = __float_as_uint(o.z);
                W.u.s.hq[3][e] = __float_as_uint(d.x); W.u.s.hq[4][e] = __float_as_uint(d.y); W.u.s.hq[5][e] = __float_as_uint(d.z);
                W.u.s.hq[6][e] = ri; W.u.s.hq[7][e] = rp; W.u.s.hq[8][e] = rsd;
                W.u.s.hq[9][e] = (uint32_t)best; W.u.s.hq[10][e] = __float_as_uint(tbest);
                if (INSTR) hsig[e] = rsig;
            }
            nhit += __popc(mh);
            if (fin) has = false;
            __syncwarp();
            if (nhit >= 32) shade_batch();
        }
        if (INSTR) cn.n_tri += nt;
    };

    // ---- S2-S5 for the primaries of one tile, as beams ----
    auto process_tile = [&](unsigned long long tile) {
        const long long p = (long long)(tile / a.tiles_per_pair);
        const long long q = (long long)(tile - (unsigned long long)p * a.tiles_per_pair);
        int k, j;
        pair_of(a, p, k, j);
        const float4 blo = a.dz.box[2 * k], bhi = a.dz.box[2 * k + 1];
        const Emitter em = make_emitter(a.sun_dirs, j, blo, bhi);
        if (!(em.Ae > 0.0f)) return;                              // edge-on flat design: F = 0, nothing launched
        const long long tbase = a.dz.tri_off[k];
        const float4 *gtri = a.dz.tri + 3 * tbase;
        const float4 *gnodes = a.dz.nodes + 4 * tbase;
        RayGen g;
        g.j = (uint32_t)j; g.k = (uint32_t)k; g.key0 = a.key0; g.key1 = a.key1; g.sampler = 0; set_torque<TORQUE>(g, a, k);
        g.inv_nx = inv_nx; g.inv_ny = inv_ny;
        BeamFrame bf;
        bf.uh = f3(0.5f * em.u.x, 0.5f * em.u.y, 0.5f * em.u.z);
        bf.vh = f3(0.5f * em.v.x, 0.5f * em.v.y, 0.5f * em.v.z);
        bf.auh = f3(fabsf(bf.uh.x), fabsf(bf.uh.y), fabsf(bf.uh.z));
        bf.avh = f3(fabsf(bf.vh.x), fabsf(bf.vh.y), fabsf(bf.vh.z));
        bf.csu = em.du * inv_nx; bf.csv = em.dv * inv_ny;
        {   // fp32 projections of points of this design are off by < 1e-6 of this scale; 10x that
            const float L = fmaxf(fabsf(blo.x), fabsf(bhi.x)) + fmaxf(fabsf(blo.y), fabsf(bhi.y)) +
                            fmaxf(fabsf(blo.z), fabsf(bhi.z));
            bf.margin = 1.0e-5f * L;
        }
        const uint32_t start = (uint32_t)(q * a.tile_rays);
        const uint32_t end = (uint32_t)min((long long)a.N, (q + 1) * (long long)a.tile_rays);
        const uint32_t nt = end - start;                          // a power of two
        const int tbits = 31 - __clz((int)nt);
        float3 acc = f3(0, 0, 0), acc_t = f3(0, 0, 0);

        // tile level: frontier descent to an entry list
        const uint32_t tcx0 = compact_even_bits(start), tcy0 = compact_even_bits(start >> 1);
        const float t_offu = fmaf((float)tcx0 * inv_nx, em.du, em.u0), t_offv = fmaf((float)tcy0 * inv_ny, em.dv, em.v0);
        const float t_wu = (float)(1u << ((tbits + 1) >> 1)) * bf.csu, t_wv = (float)(1u << (tbits >> 1)) * bf.csv;
        int n_en = 1, n_el = 0;
        if (lane == 0) W.u.b.enode[0] = 0;
        __syncwarp();
        for (int lvl = 0; lvl < 24 && n_en > 0 && n_en <= 32 && n_el <= 32; ++lvl) {
            const int node = lane < n_en ? W.u.b.enode[lane] : -1;
            __syncwarp();
            bool h0, h1; int l0, l1;
            beam_node<INSTR>(gnodes, node, bf, t_offu, t_offv, t_wu, t_wv, h0, h1, l0, l1, bc.beam_box);
            const bool p0 = h0 && l0 >= 0, p1 = h1 && l1 >= 0, f0 = h0 && l0 < 0, f1 = h1 && l1 < 0;
            const unsigned mp0 = __ballot_sync(FULL, p0), mp1 = __ballot_sync(FULL, p1);
            const unsigned mf0 = __ballot_sync(FULL, f0), mf1 = __ballot_sync(FULL, f1);
            const int np0 = __popc(mp0), nf0 = __popc(mf0), nf1 = __popc(mf1);
            SRP_CHECK(np0 + __popc(mp1) <= BEAM_EN, "entry nodes"); SRP_CHECK(n_el + nf0 + nf1 <= BEAM_EL, "entry leaves");
            if (p0) W.u.b.enode[__popc(mp0 & lt_mask)] = l0;
            if (p1) W.u.b.enode[np0 + __popc(mp1 & lt_mask)] = l1;
            if (f0) W.u.b.eleaf[n_el + __popc(mf0 & lt_mask)] = l0;
            if (f1) W.u.b.eleaf[n_el + nf0 + __popc(mf1 & lt_mask)] = l1;
            n_en = np0 + __popc(mp1); n_el += nf0 + nf1;
            __syncwarp();
        }
        if (n_en == 0 && n_el == 0) {                             // the tile's beam meets nothing: nt primary misses
            const unsigned c = nt >= 32u ? nt >> 5 : (unsigned)(lane < (int)nt);
            cn.launched += c; cn.pmiss += c; cn.segments += c; bc.tile_miss += c;
            return;
        }

        // Sub-blocks are adaptive: a block whose lists overflow is halved (down to one group of 32 rays, whose
        // rays then go to the pool for per-ray traversal); the size grows back at the next aligned position.
        const uint32_t nb_max = nt < (uint32_t)BEAM_SB ? nt : (uint32_t)BEAM_SB;
        uint32_t nb = nb_max;                                     // rays in the current sub-block
        for (uint32_t sb = start; sb < end;) {
            const int sbits = 31 - __clz((int)nb);
            const uint32_t s_wx = 1u << ((sbits + 1) >> 1), s_wy = 1u << (sbits >> 1);
            const uint32_t g_wx = nb >= 32u ? 8u : s_wx, g_wy = nb >= 32u ? 4u : s_wy;
            const float s_wu = (float)s_wx * bf.csu, s_wv = (float)s_wy * bf.csv;
            const uint32_t scx0 = compact_even_bits(sb), scy0 = compact_even_bits(sb >> 1);
            const float s_offu = fmaf((float)scx0 * inv_nx, em.du, em.u0), s_offv = fmaf((float)scy0 * inv_ny, em.dv, em.v0);
            bool ovf = false;
            int ncand = 0;
            {
                // sub-block level: descent from the entry list to candidate triangles
                for (int x = lane; x < n_en; x += 32) W.u.b.nq[x] = W.u.b.enode[x];
                int qn = n_en;
                for (int base = 0; base < n_el && !ovf; base += 32) {
                    const int x = base + lane;
                    int first = 0, cnt = 0;
                    if (x < n_el) { const unsigned u = (unsigned)~W.u.b.eleaf[x]; first = (int)(u >> 3); cnt = (int)(u & 7u) + 1; }
                    if (!beam_push_tris(W.u.b.cid, ncand, first, cnt, 0, 0, lane)) ovf = true;
                }
                __syncwarp();
                while (qn > 0 && !ovf) {
                    const int take = qn < 32 ? qn : 32;
                    const int node = lane < take ? W.u.b.nq[qn - take + lane] : -1;
                    qn -= take;
                    __syncwarp();
                    bool h0, h1; int l0, l1;
                    beam_node<INSTR>(gnodes, node, bf, s_offu, s_offv, s_wu, s_wv, h0, h1, l0, l1, bc.beam_box);
                    const bool p0 = h0 && l0 >= 0, p1 = h1 && l1 >= 0, f0 = h0 && l0 < 0, f1 = h1 && l1 < 0;
                    const unsigned mp0 = __ballot_sync(FULL, p0), mp1 = __ballot_sync(FULL, p1);
                    const int np0 = __popc(mp0), np1 = __popc(mp1);
                    if (qn + np0 + np1 > BEAM_QN) { ovf = true; break; }
                    if (p0) W.u.b.nq[qn + __popc(mp0 & lt_mask)] = l0;
                    if (p1) W.u.b.nq[qn + np0 + __popc(mp1 & lt_mask)] = l1;
                    qn += np0 + np1;
                    if (__any_sync(FULL, f0 || f1)) {
                        const unsigned u0 = (unsigned)~l0, u1 = (unsigned)~l1;
                        if (!beam_push_tris(W.u.b.cid, ncand, (int)(u0 >> 3), f0 ? (int)(u0 & 7u) + 1 : 0, (int)(u1 >> 3),
                                            f1 ? (int)(u1 & 7u) + 1 : 0, lane))
                            ovf = true;
                    }
                    __syncwarp();
                }
                if (!ovf && ncand == 0) {                        // empty sub-block
                    const unsigned c = nb >= 32u ? nb >> 5 : (unsigned)(lane < (int)nb);
                    cn.launched += c; cn.pmiss += c; cn.segments += c; bc.block_miss += c;
                    sb += nb;
                    if (nb < nb_max && (sb & (2u * nb - 1u)) == 0u) nb <<= 1;
                    continue;
                }
                if (ovf && nb > 32u) { nb >>= 1; continue; }     // retry this position with half the rays
                if (!ovf) {
                    __syncwarp();
                    for (int c = lane; c < ncand; c += 32) {
                        const int f = W.u.b.cid[c];
                        if (INSTR) bc.setups++;
                        beam_setup(__ldg(gtri + 3 * f), __ldg(gtri + 3 * f + 1), __ldg(gtri + 3 * f + 2), em, s_offu, s_offv,
                                   W.u.b.eq + 3 * c);
                    }
                    __syncwarp();
                }
            }

            // groups of 32 rays
            for (uint32_t gs = sb; gs < sb + nb; gs += 32) {
                const uint32_t gcx = compact_even_bits(gs) - scx0, gcy = compact_even_bits(gs >> 1) - scy0;
                int ng = 0;
                if (!ovf) {
                    const float gu0 = (float)gcx * bf.csu, gu1 = (float)(gcx + g_wx) * bf.csu;
                    const float gv0 = (float)gcy * bf.csv, gv1 = (float)(gcy + g_wy) * bf.csv;
                    for (int base = 0; base < ncand; base += 32) {
                        const int c = base + lane;
                        bool keep = false;
                        if (c < ncand) {
                            if (INSTR) bc.rect++;
                            const float4 E0 = W.u.b.eq[3 * c], E1 = W.u.b.eq[3 * c + 1], E2 = W.u.b.eq[3 * c + 2];
                            // largest value of each edge function over the rectangle (monotone in fp32 too)
                            const float m0 = fmaf(E0.x, E0.x >= 0.f ? gu1 : gu0, fmaf(E0.y, E0.y >= 0.f ? gv1 : gv0, E0.z));
                            const float m1 = fmaf(E1.x, E1.x >= 0.f ? gu1 : gu0, fmaf(E1.y, E1.y >= 0.f ? gv1 : gv0, E1.z));
                            const float m2 = fmaf(E2.x, E2.x >= 0.f ? gu1 : gu0, fmaf(E2.y, E2.y >= 0.f ? gv1 : gv0, E2.z));
                            keep = fminf(m0, fminf(m1, m2)) >= 0.0f;
                        }
                        const unsigned m = __ballot_sync(FULL, keep);
                        SRP_CHECK(ng + __popc(m) <= BEAM_CMAX, "group list");
                        if (keep) W.u.b.glist[ng + __popc(m & lt_mask)] = (unsigned char)c;
                        ng += __popc(m);
                    }
                    __syncwarp();
                    if (ng == 0) {                               // 32 primary misses, no ray generated
                        const unsigned c = (unsigned)(lane < (int)nb);
                        cn.launched += c; cn.pmiss += c; cn.segments += c; bc.group_miss += c;
                        continue;
                    }
                }
                // O-step 3 for this lane's ray
                const bool on = lane < (int)nb;
                const uint32_t i = gs + (uint32_t)lane;
                float3 o = f3(0, 0, 0), d = em.s;
                float lu = 0.f, lv = 0.f;
                if (on) {
                    uint32_t r0, r1, r2, r3;
                    philox4(i, g.j, g.k, 0u, g.key0, g.key1, r0, r1, r2, r3);
                    const float xi0 = uniform23(r0), xi1 = uniform23(r1);
                    const uint32_t cx = nb >= 32u ? scx0 + gcx + ldx : compact_even_bits(i);
                    const uint32_t cy = nb >= 32u ? scy0 + gcy + ldy : compact_even_bits(i >> 1);
                    const float fu = ((float)cx + xi0) * inv_nx, fv = ((float)cy + xi1) * inv_ny;
                    const float pu = fmaf(fu, em.du, em.u0), pv = fmaf(fv, em.dv, em.v0);
                    o = f3(fmaf(pu, em.u.x, fmaf(pv, em.v.x, em.worg * em.s.x)),
                           fmaf(pu, em.u.y, fmaf(pv, em.v.y, em.worg * em.s.y)),
                           fmaf(pu, em.u.z, fmaf(pv, em.v.z, em.worg * em.s.z)));
                    lu = ((float)(cx - scx0) + xi0) * bf.csu;
                    lv = ((float)(cy - scy0) + xi1) * bf.csv;
                    cn.launched++; cn.segments++;
                }
                if (ovf) {                                       // too much geometry behind this group: per-ray traversal
                    if (on) bc.fallback++;
                    pool_push(on, o, d, i, (uint32_t)p, SRC_NONE, 0ULL);
                    continue;
                }
                // O-step 4 against the shared list: all lanes converged, operands broadcast
                float tbest = FLT_MAX;
                int best = -1;
                for (int e = 0; e < ng; ++e) {
                    const int c = W.u.b.glist[e];
                    const float4 E0 = W.u.b.eq[3 * c], E1 = W.u.b.eq[3 * c + 1], E2 = W.u.b.eq[3 * c + 2];
                    const float e0 = fmaf(E0.x, lu, fmaf(E0.y, lv, E0.z));
                    const float e1 = fmaf(E1.x, lu, fmaf(E1.y, lv, E1.z));
                    const float e2 = fmaf(E2.x, lu, fmaf(E2.y, lv, E2.z));
                    const float t = fmaf(E0.w, lu, fmaf(E1.w, lv, E2.w));
                    if (fminf(e0, fminf(e1, e2)) >= 0.0f && t < tbest) { tbest = t; best = c; }
                }
                if (INSTR && on) bc.tri2d += (unsigned)ng;
                if (best >= 0) best = W.u.b.cid[best];
                if (!on) best = -1;
                int fate = -1, src = -1, depth = 0;
                unsigned long long sig = 0;
                if (on) {
                    if (best < 0) cn.pmiss++;
                    else {
                        atomicAdd(&s_hist[warp][0], 1u);
                        if (INSTR) sig = (unsigned long long)(a.dz.perm[tbase + best] + 1);
                        fate = shade<TORQUE, 0u, GLOSSY, ANALOG ? 1 : 0>(__ldg(gtri + 3 * best), __ldg(gtri + 3 * best + 1), __ldg(gtri + 3 * best + 2), tbest,
                                     best, g, i, a.B, a.deposit, o, d, src, depth, acc, acc_t, a.dz.esc, tbase + best, a.dz.shin);
                        if (fate == SHADE_ESCAPES) { cn.segments++; cn.escaped++; cn.mesc++; }
                        if (fate == SHADE_ABSORBED) cn.absorbed++;
                        if (fate == SHADE_CAPPED) cn.capped++;
                    }
                    if (INSTR && fate != SHADE_CONTINUE && a.sig_out) a.sig_out[p * a.N + i] = sig;
                }
                pool_push(fate == SHADE_CONTINUE, o, d, i, (uint32_t)p, ((uint32_t)depth << 27) | (uint32_t)src, sig);
            }
            sb += nb;
            if (nb < nb_max && (sb & (2u * nb - 1u)) == 0u) nb <<= 1;
        }

        // S7 for the tile's primaries: warp reduction in fp64, then one fixed-point atomic per component
        flush_tile_acc<TORQUE>(a, p, acc, acc_t, lane);
    };

    // ---- persistent loop: tiles until the pool is worth draining ----
    bool more = true;
    for (;;) {
        if (more) {
            unsigned long long tile = 0;
            if (lane == 0) tile = atomicAdd(a.work_counter, 1ULL);
            tile = __shfl_sync(FULL, tile, 0);
            if (tile >= total_tiles) more = false;
            else process_tile(tile);
        }
        __syncwarp();
        const uint32_t cnt = pool.tail - pool.head;
        if (cnt >= (uint32_t)POOL_HIGH || (!more && cnt != 0u)) { drain(); __syncwarp(); }
        if (!more && pool.tail == pool.head) break;
    }
    flush_counters<INSTR>(a, cn, s_hist[warp], lane);
    flush_beam_counters(a, bc, lane);
}

} // namespace

int srp_beam_blocks_per_sm() { return blocks_per_sm(beam_trace_kernel<false, false, false, false>); }

// Words of global memory the beam kernel's per-warp ray pools need, and the ring capacity per warp.
size_t srp_beam_pool_words(int num_sms, bool instrumented, int tile_rays, int *cap_out)
{
    int per_sm = 0;
    const int occ[6] = { blocks_per_sm(beam_trace_kernel<true, false, false, false>), blocks_per_sm(beam_trace_kernel<true, false, true, false>),
                         blocks_per_sm(beam_trace_kernel<false, false, false, false>), blocks_per_sm(beam_trace_kernel<false, false, true, false>),
                         blocks_per_sm(beam_trace_kernel<false, true, false, false>), blocks_per_sm(beam_trace_kernel<false, true, true, false>) };
    for (int v = instrumented ? 0 : 2; v < (instrumented ? 2 : 6); ++v) if (occ[v] > per_sm) per_sm = occ[v];
    if (per_sm < 1) per_sm = 1;
    int cap = 64;
    while (cap < POOL_HIGH + tile_rays + 64) cap <<= 1;
    *cap_out = cap;
    return (size_t)num_sms * per_sm * TRACE_WARPS * (instrumented ? POOL_FIELDS_INSTR : POOL_FIELDS) * (size_t)cap;
}

cudaError_t srp_launch_beam(const TraceArgs &a, bool instrumented, int num_sms, cudaStream_t stream)
{
    return SRP_LAUNCH3(beam_trace_kernel);
}
