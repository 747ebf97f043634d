// trace_beam.cu -- beam_trace_kernel (S2-S5 for the primaries of designs with a BVH, stratified sampler): the
// primaries of a tile are traced as beams and shaded; photons that go on are handed to the bounce kernel
// (trace_bounce.cu) through the ray queue.
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
// Bounce rays are incoherent: they go to the ray queue and through per-ray traversal in the bounce
// kernel.  A sub-block whose lists overflow is halved; a single group that still overflows (a beam
// along an edge-on panel, a bundle of thin facets) sends its 32 primaries to the queue as well, so
// any input is handled.
#ifndef BEAM_BLOCKS_PER_SM
#define BEAM_BLOCKS_PER_SM 4        // 4 blocks with 240-candidate lists beat 5 with 160 (-4 %), 6 with 144 (+7 %), 8 with 96 (+35 %)
#endif
#ifndef BEAM_SB_DEF
#define BEAM_SB_DEF 256
#endif
constexpr int BEAM_SB = BEAM_SB_DEF;        // rays per sub-block
#ifndef BEAM_CMAX_DEF
#define BEAM_CMAX_DEF 240
#endif
constexpr int BEAM_CMAX = BEAM_CMAX_DEF;      // candidate triangles per sub-block
#ifndef BEAM_QN_DEF
#define BEAM_QN_DEF 160
#endif
constexpr int BEAM_QN = BEAM_QN_DEF;        // node queue of the sub-block descent
constexpr int BEAM_EN = 64;         // tile entry list: internal nodes
constexpr int BEAM_EL = 96;         // tile entry list: leaf links (<= 32 when a level starts, + 2 x 32 in that level)

struct BeamFrame {                  // warp-uniform per pair
    float3 uh, vh, auh, avh;        // u/2, v/2 and their absolute values
    float csu, csv;                 // cell size along u and v
    float icsu, icsv;               // and their reciprocals
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
#ifdef SRP_NO_LD256
    const float4 n0 = __ldg(nodes + 4 * node), n1 = __ldg(nodes + 4 * node + 1), n2 = __ldg(nodes + 4 * node + 2),
                 n3 = __ldg(nodes + 4 * node + 3);
#else
    const F8 lo_ = ldg256(nodes + 4 * node), hi_ = ldg256(nodes + 4 * node + 2);
    const float4 n0 = lo_.a, n1 = lo_.b, n2 = hi_.a, n3 = hi_.b;
#endif
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
    // leaves hold <= 2 triangles by default (SRP_LEAF_MAX): two predicated stores each, then whatever is left
    if (cnt0 > 0) cid[pos] = first0;
    if (cnt0 > 1) cid[pos + 1] = first0 + 1;
    for (int t = 2; t < cnt0; ++t) cid[pos + t] = first0 + t;
    pos += cnt0;
    if (cnt1 > 0) cid[pos] = first1;
    if (cnt1 > 1) cid[pos + 1] = first1 + 1;
    for (int t = 2; t < cnt1; ++t) cid[pos + t] = first1 + t;
    ncand += total;
    return true;
}


struct BeamSmem {                   // per warp
    float4 eq[3 * BEAM_CMAX];       // (A0,B0,C0,Wu) (A1,B1,C1,Wv) (A2,B2,C2,Wc) per candidate
    int cid[BEAM_CMAX];             // candidate -> sorted triangle index
    unsigned short cbox[BEAM_CMAX]; // the cells of the 16 x 16 sub-block its projection can touch, 4 bits each:
                                    // x0 | x1 << 4 | y0 << 8 | y1 << 12 (x0 = 15, x1 = 0: none)
    int enode[BEAM_EN];
    int eleaf[BEAM_EL];
    int nq[BEAM_QN];                // node queue of the sub-block descent; afterwards the groups' candidate lists
                                    // (one byte per entry) live here
};
static_assert(BEAM_SB <= 256, "cbox holds 4-bit cell coordinates");
static_assert(BEAM_QN * 4 >= BEAM_CMAX, "the group list lives in the node queue");

template <bool INSTR, bool TORQUE, bool GLOSSY, bool ANALOG>
__global__ void __launch_bounds__(TRACE_THREADS, BEAM_BLOCKS_PER_SM)
beam_trace_kernel(const TraceArgs a)
{
    extern __shared__ __align__(16) unsigned char s_dyn[];     // BeamSmem per warp: more than the 48 KB a static array may have
    BeamSmem *s_w = reinterpret_cast<BeamSmem *>(s_dyn);
    __shared__ unsigned s_hist[TRACE_WARPS][16];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    if (lane < 16) s_hist[warp][lane] = 0;
    __syncwarp();
    BeamSmem &W = s_w[warp];
    LaneCounters cn = { 0, 0, 0, 0, 0, 0, 0, 0 };
    BeamCounters bc = { 0, 0, 0, 0, 0, 0, 0, 0 };
    const uint32_t ldx = compact_even_bits((uint32_t)lane), ldy = compact_even_bits((uint32_t)lane >> 1);
    const float inv_nx = 1.0f / (float)(1u << ((a.log2N + 1) >> 1)), inv_ny = 1.0f / (float)(1u << (a.log2N >> 1));

    // Appends this lane's ray (if `push`) to the ray queue; warp-wide call.  The warp reserves RQ_CHUNK slots of the
    // queue at a time (one atomic per ~30 pushes instead of one per push); slots it has reserved and not filled when
    // it stops are marked dead for the bounce kernel.
    uint32_t ch_next = 0, ch_end = 0;                              // warp-uniform: the warp's reserved slots
    auto queue_push = [&](bool push, const float3 &o, const float3 &d, uint32_t i, uint32_t p, uint32_t sd,
                         unsigned long long sig) {
        const unsigned m = __ballot_sync(FULL, push);
        if (m == 0u) return;
        const uint32_t cnt = (uint32_t)__popc(m);
        if (ch_next + cnt > ch_end) {                              // not enough room left: give the rest up, take a new chunk
            for (uint32_t x = ch_next + (uint32_t)lane; x < ch_end; x += 32u) rq_mark_dead(a, x);
            uint32_t base = 0;
            if (lane == 0) base = atomicAdd(a.rq_ctr, RQ_CHUNK);
            ch_next = __shfl_sync(FULL, base, 0); ch_end = ch_next + RQ_CHUNK;
        }
        if (push) {
            const uint32_t pos = ch_next + (uint32_t)__popc(m & lt_mask);
            SRP_CHECK(pos < a.rq_cap, "ray queue");
            rq_store<INSTR>(a, pos, o, d, i, p, sd, sig);
        }
        ch_next += cnt;
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
        bf.icsu = 1.0f / bf.csu; bf.icsv = 1.0f / bf.csv;
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
        if (lane == 0) W.enode[0] = 0;
        __syncwarp();
        for (int lvl = 0; lvl < 24 && n_en > 0 && n_en <= 32 && n_el <= 32; ++lvl) {
            const int node = lane < n_en ? W.enode[lane] : -1;
            __syncwarp();
            bool h0, h1; int l0, l1;
            beam_node<INSTR>(gnodes, node, bf, t_offu, t_offv, t_wu, t_wv, h0, h1, l0, l1, bc.beam_box);
            const bool p0 = h0 && l0 >= 0, p1 = h1 && l1 >= 0, f0 = h0 && l0 < 0, f1 = h1 && l1 < 0;
            const unsigned mp0 = __ballot_sync(FULL, p0), mp1 = __ballot_sync(FULL, p1);
            const unsigned mf0 = __ballot_sync(FULL, f0), mf1 = __ballot_sync(FULL, f1);
            const int np0 = __popc(mp0), nf0 = __popc(mf0), nf1 = __popc(mf1);
            SRP_CHECK(np0 + __popc(mp1) <= BEAM_EN, "entry nodes"); SRP_CHECK(n_el + nf0 + nf1 <= BEAM_EL, "entry leaves");
            if (p0) W.enode[__popc(mp0 & lt_mask)] = l0;
            if (p1) W.enode[np0 + __popc(mp1 & lt_mask)] = l1;
            if (f0) W.eleaf[n_el + __popc(mf0 & lt_mask)] = l0;
            if (f1) W.eleaf[n_el + nf0 + __popc(mf1 & lt_mask)] = l1;
            n_en = np0 + __popc(mp1); n_el += nf0 + nf1;
            __syncwarp();
        }
        if (n_en == 0 && n_el == 0) {                             // the tile's beam meets nothing: nt primary misses
            const unsigned c = nt >= 32u ? nt >> 5 : (unsigned)(lane < (int)nt);
            cn.launched += c; cn.pmiss += c; cn.segments += c; bc.tile_miss += c;
            return;
        }

        // Sub-blocks are adaptive: a block whose lists overflow is halved (down to one group of 32 rays, whose
        // rays then go to the ray queue for per-ray traversal); the size grows back at the next aligned position.
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
                for (int x = lane; x < n_en; x += 32) W.nq[x] = W.enode[x];
                int qn = n_en;
                for (int base = 0; base < n_el && !ovf; base += 32) {
                    const int x = base + lane;
                    int first = 0, cnt = 0;
                    if (x < n_el) { const unsigned u = (unsigned)~W.eleaf[x]; first = (int)(u >> 3); cnt = (int)(u & 7u) + 1; }
                    if (!beam_push_tris(W.cid, ncand, first, cnt, 0, 0, lane)) ovf = true;
                }
                __syncwarp();
                while (qn > 0 && !ovf) {
                    const int take = qn < 32 ? qn : 32;
                    const int node = lane < take ? W.nq[qn - take + lane] : -1;
                    qn -= take;
                    __syncwarp();
                    bool h0, h1; int l0, l1;
                    beam_node<INSTR>(gnodes, node, bf, s_offu, s_offv, s_wu, s_wv, h0, h1, l0, l1, bc.beam_box);
                    const bool p0 = h0 && l0 >= 0, p1 = h1 && l1 >= 0, f0 = h0 && l0 < 0, f1 = h1 && l1 < 0;
                    const unsigned mp0 = __ballot_sync(FULL, p0), mp1 = __ballot_sync(FULL, p1);
                    const int np0 = __popc(mp0), np1 = __popc(mp1);
                    if (qn + np0 + np1 > BEAM_QN) { ovf = true; break; }
                    if (p0) W.nq[qn + __popc(mp0 & lt_mask)] = l0;
                    if (p1) W.nq[qn + np0 + __popc(mp1 & lt_mask)] = l1;
                    qn += np0 + np1;
                    if (__any_sync(FULL, f0 || f1)) {
                        const unsigned u0 = (unsigned)~l0, u1 = (unsigned)~l1;
                        if (!beam_push_tris(W.cid, ncand, (int)(u0 >> 3), f0 ? (int)(u0 & 7u) + 1 : 0, (int)(u1 >> 3),
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
                        const int f = W.cid[c];
                        if (INSTR) bc.setups++;
                        float4 bb;
                        beam_setup(__ldg(gtri + 3 * f), __ldg(gtri + 3 * f + 1), __ldg(gtri + 3 * f + 2), em, s_offu, s_offv,
                                   W.eq + 3 * c, &bb);
                        // cells of the sub-block (16 x 16) the triangle's bounding rectangle touches, widened by the
                        // projection error bound: a ray outside them is outside the triangle
                        const float x0 = floorf((bb.x - bf.margin) * bf.icsu), x1 = floorf((bb.y + bf.margin) * bf.icsu);
                        const float y0 = floorf((bb.z - bf.margin) * bf.icsv), y1 = floorf((bb.w + bf.margin) * bf.icsv);
                        const bool none = !(bb.x <= bb.y) || x1 < 0.f || y1 < 0.f || x0 > 15.f || y0 > 15.f;
                        W.cbox[c] = none ? (unsigned short)0x000f
                                         : (unsigned short)((unsigned)fmaxf(x0, 0.f) | ((unsigned)fminf(x1, 15.f) << 4) |
                                                            ((unsigned)fmaxf(y0, 0.f) << 8) | ((unsigned)fminf(y1, 15.f) << 12));
                    }
                    __syncwarp();
                }
            }

            // groups of 32 rays
            for (uint32_t gs = sb; gs < sb + nb; gs += 32) {
                const uint32_t gcx = compact_even_bits(gs) - scx0, gcy = compact_even_bits(gs >> 1) - scy0;
                int ng = 0;
                unsigned char *glist = reinterpret_cast<unsigned char *>(W.nq);
                if (!ovf) {
                    const float gu0 = (float)gcx * bf.csu, gu1 = (float)(gcx + g_wx) * bf.csu;
                    const float gv0 = (float)gcy * bf.csv, gv1 = (float)(gcy + g_wy) * bf.csv;
                    for (int base = 0; base < ncand; base += 32) {
                        const int c = base + lane;
                        bool keep = false;
                        const unsigned cb = c < ncand ? W.cbox[c] : 0x000fu;
                        if ((cb & 15u) < gcx + g_wx && ((cb >> 4) & 15u) >= gcx && ((cb >> 8) & 15u) < gcy + g_wy && (cb >> 12) >= gcy) {
                            if (INSTR) bc.rect++;
                            const float4 E0 = W.eq[3 * c], E1 = W.eq[3 * c + 1], E2 = W.eq[3 * c + 2];
                            // largest value of each edge function over the rectangle (monotone in fp32 too)
                            const float m0 = fmaf(E0.x, E0.x >= 0.f ? gu1 : gu0, fmaf(E0.y, E0.y >= 0.f ? gv1 : gv0, E0.z));
                            const float m1 = fmaf(E1.x, E1.x >= 0.f ? gu1 : gu0, fmaf(E1.y, E1.y >= 0.f ? gv1 : gv0, E1.z));
                            const float m2 = fmaf(E2.x, E2.x >= 0.f ? gu1 : gu0, fmaf(E2.y, E2.y >= 0.f ? gv1 : gv0, E2.z));
                            keep = fminf(m0, fminf(m1, m2)) >= 0.0f;
                        }
                        const unsigned m = __ballot_sync(FULL, keep);
                        SRP_CHECK(ng + __popc(m) <= BEAM_CMAX, "group list");
                        if (keep) glist[ng + __popc(m & lt_mask)] = (unsigned char)c;
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
                    queue_push(on, o, d, i, (uint32_t)p, SRC_NONE, 0ULL);
                    continue;
                }
                // O-step 4 against the shared list: all lanes converged, operands broadcast
                float tbest = FLT_MAX;
                int best = -1;
                for (int e = 0; e < ng; ++e) {
                    const int c = glist[e];
                    const float4 E0 = W.eq[3 * c], E1 = W.eq[3 * c + 1], E2 = W.eq[3 * c + 2];
                    const float e0 = fmaf(E0.x, lu, fmaf(E0.y, lv, E0.z));
                    const float e1 = fmaf(E1.x, lu, fmaf(E1.y, lv, E1.z));
                    const float e2 = fmaf(E2.x, lu, fmaf(E2.y, lv, E2.z));
                    const float t = fmaf(E0.w, lu, fmaf(E1.w, lv, E2.w));
                    if (fminf(e0, fminf(e1, e2)) >= 0.0f && t < tbest) { tbest = t; best = c; }
                }
                if (INSTR && on) bc.tri2d += (unsigned)ng;
                if (best >= 0) best = W.cid[best];
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
                queue_push(fate == SHADE_CONTINUE, o, d, i, (uint32_t)p, ((uint32_t)depth << 27) | (uint32_t)src, sig);
            }
            sb += nb;
            if (nb < nb_max && (sb & (2u * nb - 1u)) == 0u) nb <<= 1;
        }

        // S7 for the tile's primaries: warp reduction in fp64, then one fixed-point atomic per component
        flush_tile_acc<TORQUE>(a, p, acc, acc_t, lane);
    };

    // ---- persistent loop: tiles until they run out, or until the ray queue is full enough for the bounce kernel
    // to take over (the host then launches this kernel again; the tile counter carries on) ----
    for (;;) {
        unsigned long long tile = ~0ULL;
        if (lane == 0 && *(volatile unsigned *)a.rq_ctr < a.rq_high) tile = a.tile_begin + atomicAdd(a.work_counter, 1ULL);
        tile = __shfl_sync(FULL, tile, 0);
        if (tile >= a.tile_end) break;
        process_tile(tile);
        __syncwarp();
    }
    for (uint32_t x = ch_next + (uint32_t)lane; x < ch_end; x += 32u) rq_mark_dead(a, x);   // unused slots of the last chunk
    flush_counters<INSTR>(a, cn, s_hist[warp], lane);
    flush_beam_counters(a, bc, lane);
}

} // namespace

constexpr size_t BEAM_SMEM_BYTES = sizeof(BeamSmem) * TRACE_WARPS;

int srp_beam_blocks_per_sm() { return blocks_per_sm(beam_trace_kernel<false, false, false, false>, BEAM_SMEM_BYTES); }

// Resident warps of the beam kernel at most (any build): each may add one tile's rays to the queue after the
// high-water mark is reached.
int srp_beam_warps(int num_sms)
{
    int per_sm = 0;
    const size_t sm = BEAM_SMEM_BYTES;
    const int occ[6] = { blocks_per_sm(beam_trace_kernel<true, false, false, false>, sm), blocks_per_sm(beam_trace_kernel<true, false, true, false>, sm),
                         blocks_per_sm(beam_trace_kernel<false, false, false, false>, sm), blocks_per_sm(beam_trace_kernel<false, false, true, false>, sm),
                         blocks_per_sm(beam_trace_kernel<false, true, false, false>, sm), blocks_per_sm(beam_trace_kernel<false, true, true, false>, sm) };
    for (int v = 0; v < 6; ++v) if (occ[v] > per_sm) per_sm = occ[v];
    if (per_sm < 1) per_sm = 1;
    return num_sms * per_sm * TRACE_WARPS;
}

cudaError_t srp_launch_beam(const TraceArgs &a, bool instrumented, int num_sms, cudaStream_t stream)
{
    const size_t dyn_smem = BEAM_SMEM_BYTES;
    return SRP_LAUNCH3(beam_trace_kernel);
}
