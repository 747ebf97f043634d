// trace_small.cu -- small_beam_kernel (S2-S7 for designs without a hierarchy, T <= SRP_BRUTE_MAX_TRIS, stratified
// sampler): "test all triangles" with per-tile 2-D set-ups, block culling and facet-side masks.
#include "trace_common.cuh"

namespace {

// ---- designs without a hierarchy (T <= SRP_BRUTE_MAX_TRIS), stratified sampler ----
// "Test all triangles" with the same two ideas as the beam kernel.  The primaries of
// a tile are parallel, so every triangle is set up ONCE per tile as three 2-D edge functions and a
// depth plane in the emitter frame (16 instructions per ray-triangle test instead of the ~45 of
// Moller-Trumbore), and a block of rays whose rectangle no edge function admits is a block of
// misses: no Philox call, no test.  Levels: tile -> 256 rays -> 32 rays (one per lane).  Bounce rays
// collect in the warp's shared-memory queue and are traced 32 at a time against all triangles
// (Moller-Trumbore from shared memory; every ray costs the same, so passes stay converged).
struct SmallSmem {                  // per warp
    float4 tri[3 * SRP_BRUTE_MAX_TRIS];     // the design's packed triangles (S4 for bounce rays, S5)
    float4 eq[3 * SRP_BRUTE_MAX_TRIS];      // per tile: edge functions + depth plane of every triangle
    unsigned char tl[SRP_BRUTE_MAX_TRIS], sl[SRP_BRUTE_MAX_TRIS], gl[SRP_BRUTE_MAX_TRIS];   // tile / sub-block / group lists
    unsigned long long vis[2][SRP_BRUTE_MAX_TRIS];   // per design: triangles with a vertex in front of / behind each facet
    WarpQueue q;
};

// Candidates of `in` (n_in of them; nullptr = all triangles 0..n_in-1) whose edge functions admit the
// rectangle [u0,u1] x [v0,v1] -> out; returns how many.  Warp-wide call.
template <bool INSTR>
__device__ __forceinline__ int small_filter(const float4 *eq, const unsigned char *in, int n_in, float u0, float u1,
                                            float v0, float v1, unsigned char *out, int lane, unsigned lt_mask,
                                            unsigned &n_rect)
{
    int n = 0;
    for (int base = 0; base < n_in; base += 32) {
        const int x = base + lane;
        bool keep = false;
        int c = 0;
        if (x < n_in) {
            if (INSTR) ++n_rect;
            c = in ? (int)in[x] : x;
            const float4 E0 = eq[3 * c], E1 = eq[3 * c + 1], E2 = eq[3 * c + 2];
            const float m0 = fmaf(E0.x, E0.x >= 0.f ? u1 : u0, fmaf(E0.y, E0.y >= 0.f ? v1 : v0, E0.z));
            const float m1 = fmaf(E1.x, E1.x >= 0.f ? u1 : u0, fmaf(E1.y, E1.y >= 0.f ? v1 : v0, E1.z));
            const float m2 = fmaf(E2.x, E2.x >= 0.f ? u1 : u0, fmaf(E2.y, E2.y >= 0.f ? v1 : v0, E2.z));
            keep = fminf(m0, fminf(m1, m2)) >= 0.0f;
        }
        const unsigned m = __ballot_sync(FULL, keep);
        SRP_CHECK(n + __popc(m) <= SRP_BRUTE_MAX_TRIS, "small-design list");
        if (keep) out[n + __popc(m & lt_mask)] = (unsigned char)c;
        n += __popc(m);
    }
    __syncwarp();
    return n;
}

template <bool MASKS, bool INSTR, bool TORQUE, bool GLOSSY, bool ANALOG>
__global__ void __launch_bounds__(TRACE_THREADS, 6)
small_beam_kernel(const TraceArgs a)
{
    __shared__ SmallSmem s_w[TRACE_WARPS];
    __shared__ unsigned long long s_qsig[INSTR ? TRACE_WARPS * QCAP : 1];
    __shared__ unsigned s_hist[TRACE_WARPS][16];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    if (lane < 16) s_hist[warp][lane] = 0;
    __syncwarp();
    SmallSmem &W = s_w[warp];
    WarpQueue &Q = W.q;
    unsigned long long *qsig = s_qsig + (INSTR ? warp * QCAP : 0);
    LaneCounters cn = { 0, 0, 0, 0, 0, 0, 0, 0 };
    BeamCounters bc = { 0, 0, 0, 0, 0, 0, 0, 0 };
    const unsigned long long total_tiles = (unsigned long long)a.n_pairs * a.tiles_per_pair;
    const uint32_t ldx = compact_even_bits((uint32_t)lane), ldy = compact_even_bits((uint32_t)lane >> 1);
    const float inv_nx = 1.0f / (float)(1u << ((a.log2N + 1) >> 1)), inv_ny = 1.0f / (float)(1u << (a.log2N >> 1));
    int loaded_k = -1;

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
        if (loaded_k != k) {
            const float4 *gtri = a.dz.tri + 3 * tbase;
            __syncwarp();
            for (int x = lane; x < 3 * T; x += 32) W.tri[x] = gtri[x];
            loaded_k = k;
            __syncwarp();
            // A ray that leaves facet f on the side of +n (or -n) can only hit triangles with a vertex on that
            // side of f's plane: two 64-bit masks per facet, built once per design.  The margin (1e-6 of the
            // design's extent) keeps only coplanar neighbours out, which exact arithmetic never hits.
            const float4 blo = a.dz.box[2 * k], bhi = a.dz.box[2 * k + 1];
            const float eps = 1.0e-6f * (fmaxf(fabsf(blo.x), fabsf(bhi.x)) + fmaxf(fabsf(blo.y), fabsf(bhi.y)) +
                                         fmaxf(fabsf(blo.z), fabsf(bhi.z)));
            for (int f = lane; f < T; f += 32) {
                const float4 q0 = W.tri[3 * f], q1 = W.tri[3 * f + 1], q2 = W.tri[3 * f + 2];
                float3 n = cross3(f3(q1.x, q1.y, q1.z), f3(q2.x, q2.y, q2.z));
                const float il = rsqrtf(dot3(n, n));
                n = f3(n.x * il, n.y * il, n.z * il);
                unsigned long long front = 0, back = 0;
                for (int t = 0; t < T; ++t) {
                    if (t == f) continue;
                    const float4 p0 = W.tri[3 * t], p1 = W.tri[3 * t + 1], p2 = W.tri[3 * t + 2];
                    const float3 r = f3(p0.x - q0.x, p0.y - q0.y, p0.z - q0.z);
                    const float d0 = dot3(n, r), d1 = d0 + dot3(n, f3(p1.x, p1.y, p1.z)), d2 = d0 + dot3(n, f3(p2.x, p2.y, p2.z));
                    if (fmaxf(d0, fmaxf(d1, d2)) > eps) front |= 1ULL << t;
                    if (fminf(d0, fminf(d1, d2)) < -eps) back |= 1ULL << t;
                }
                W.vis[0][f] = front; W.vis[1][f] = back;
            }
        }
        __syncwarp();
        RayGen g;
        g.j = (uint32_t)j; g.k = (uint32_t)k; g.key0 = a.key0; g.key1 = a.key1; g.sampler = 0; set_torque<TORQUE>(g, a, k);
        g.inv_nx = inv_nx; g.inv_ny = inv_ny;
        const float csu = em.du * inv_nx, csv = em.dv * inv_ny;
        const uint32_t start = (uint32_t)(q * a.tile_rays);
        const uint32_t end = (uint32_t)min((long long)a.N, (q + 1) * (long long)a.tile_rays);
        const uint32_t nt = end - start;                          // a power of two
        const int tbits = 31 - __clz((int)nt);
        int qcount = 0;                                           // warp-uniform
        float3 acc = f3(0, 0, 0), acc_t = f3(0, 0, 0);

        // a pass of <= 32 queued bounce rays against all triangles (S4, S6)
        auto secondary_pass = [&]() {
            const int take = qcount < 32 ? qcount : 32;
            bool alive = false;
            uint32_t i = 0;
            float3 o = f3(0, 0, 0), d = em.s;
            int src = -1, depth = 0;
            unsigned long long sig = 0;
            if (lane < take) {
                const int e = qcount - take + lane;
                o = f3(Q.ox[e], Q.oy[e], Q.oz[e]); d = f3(Q.dx[e], Q.dy[e], Q.dz[e]);
                i = Q.i[e]; src = Q.src_depth[e] & 0x07ffffff; depth = (int)((unsigned)Q.src_depth[e] >> 27);
                if (INSTR) sig = qsig[e];
                alive = true;
            }
            qcount -= take;
            __syncwarp();
            int fate = -1;
            if (alive) {
                float tbest = FLT_MAX; int best = -1;
                cn.segments++;
                {   // only the triangles on the side of the source facet the ray leaves on, in index order
                    const float3 ns = cross3(f3(W.tri[3 * src + 1].x, W.tri[3 * src + 1].y, W.tri[3 * src + 1].z),
                                             f3(W.tri[3 * src + 2].x, W.tri[3 * src + 2].y, W.tri[3 * src + 2].z));
                    unsigned long long m = W.vis[dot3(ns, d) > 0.0f ? 0 : 1][src];
                    if (INSTR) cn.n_tri += (unsigned)__popcll(m);
                    while (m) {
                        const int f = __ffsll((long long)m) - 1;
                        m &= m - 1;
                        tri_test(W.tri[3 * f], W.tri[3 * f + 1], W.tri[3 * f + 2], o, d, f, tbest, best);
                    }
                }
                if (best < 0) cn.escaped++;
                else {
                    atomicAdd(&s_hist[warp][depth], 1u);
                    if (INSTR) sig = sig * 1000003ULL + (unsigned long long)(a.dz.perm[tbase + best] + 1);
                    fate = shade<TORQUE, 0u, GLOSSY, ANALOG ? 1 : 0>(W.tri[3 * best], W.tri[3 * best + 1], W.tri[3 * best + 2], tbest, best, g, i, a.B,
                                 a.deposit, o, d, src, depth, acc, acc_t, MASKS ? a.dz.esc : nullptr, tbase + best, a.dz.shin);
                    if (MASKS && fate == SHADE_ESCAPES) { cn.segments++; cn.escaped++; cn.mesc++; }
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
        };

        // tile level: set every triangle up in the tile's local emitter frame; which ones touch the tile?
        const uint32_t tcx0 = compact_even_bits(start), tcy0 = compact_even_bits(start >> 1);
        const float offu = fmaf((float)tcx0 * inv_nx, em.du, em.u0), offv = fmaf((float)tcy0 * inv_ny, em.dv, em.v0);
        for (int c = lane; c < T; c += 32) {
            if (INSTR) bc.setups++;
            beam_setup(W.tri[3 * c], W.tri[3 * c + 1], W.tri[3 * c + 2], em, offu, offv, W.eq + 3 * c);
        }
        __syncwarp();
        const float t_wu = (float)(1u << ((tbits + 1) >> 1)) * csu, t_wv = (float)(1u << (tbits >> 1)) * csv;
        const int n_tl = small_filter<INSTR>(W.eq, nullptr, T, 0.0f, t_wu, 0.0f, t_wv, W.tl, lane, lt_mask, bc.rect);
        if (n_tl == 0) {
            const unsigned c = nt >= 32u ? nt >> 5 : (unsigned)(lane < (int)nt);
            cn.launched += c; cn.pmiss += c; cn.segments += c; bc.tile_miss += c;
            continue;
        }
        const uint32_t nb = nt < 256u ? nt : 256u;               // rays per sub-block
        const int sbits = 31 - __clz((int)nb);
        const uint32_t s_wx = 1u << ((sbits + 1) >> 1), s_wy = 1u << (sbits >> 1);
        const uint32_t g_wx = nb >= 32u ? 8u : s_wx, g_wy = nb >= 32u ? 4u : s_wy;
        for (uint32_t sb = start; sb < end; sb += nb) {
            const uint32_t scx = compact_even_bits(sb) - tcx0, scy = compact_even_bits(sb >> 1) - tcy0;   // cells from the tile corner
            const int n_sl = small_filter<INSTR>(W.eq, W.tl, n_tl, (float)scx * csu, (float)(scx + s_wx) * csu, (float)scy * csv,
                                          (float)(scy + s_wy) * csv, W.sl, lane, lt_mask, bc.rect);
            if (n_sl == 0) {
                const unsigned c = nb >= 32u ? nb >> 5 : (unsigned)(lane < (int)nb);
                cn.launched += c; cn.pmiss += c; cn.segments += c; bc.block_miss += c;
                continue;
            }
            for (uint32_t gs = sb; gs < sb + nb; gs += 32) {
                const uint32_t gcx = compact_even_bits(gs) - tcx0, gcy = compact_even_bits(gs >> 1) - tcy0;
                const int ng = small_filter<INSTR>(W.eq, W.sl, n_sl, (float)gcx * csu, (float)(gcx + g_wx) * csu, (float)gcy * csv,
                                            (float)(gcy + g_wy) * csv, W.gl, lane, lt_mask, bc.rect);
                if (ng == 0) {
                    const unsigned c = (unsigned)(lane < (int)nb);
                    cn.launched += c; cn.pmiss += c; cn.segments += c; bc.group_miss += c;
                    continue;
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
                    const uint32_t cx = nb >= 32u ? tcx0 + gcx + ldx : compact_even_bits(i);
                    const uint32_t cy = nb >= 32u ? tcy0 + gcy + ldy : compact_even_bits(i >> 1);
                    const float fu = ((float)cx + xi0) * inv_nx, fv = ((float)cy + xi1) * inv_ny;
                    const float pu = fmaf(fu, em.du, em.u0), pv = fmaf(fv, em.dv, em.v0);
                    o = f3(fmaf(pu, em.u.x, fmaf(pv, em.v.x, em.worg * em.s.x)),
                           fmaf(pu, em.u.y, fmaf(pv, em.v.y, em.worg * em.s.y)),
                           fmaf(pu, em.u.z, fmaf(pv, em.v.z, em.worg * em.s.z)));
                    lu = ((float)(cx - tcx0) + xi0) * csu;
                    lv = ((float)(cy - tcy0) + xi1) * csv;
                    cn.launched++; cn.segments++;
                }
                // O-step 4 against the group's list: all lanes converged, operands broadcast
                float tbest = FLT_MAX;
                int best = -1;
                for (int e = 0; e < ng; ++e) {
                    const int c = W.gl[e];
                    const float4 E0 = W.eq[3 * c], E1 = W.eq[3 * c + 1], E2 = W.eq[3 * c + 2];
                    const float e0 = fmaf(E0.x, lu, fmaf(E0.y, lv, E0.z));
                    const float e1 = fmaf(E1.x, lu, fmaf(E1.y, lv, E1.z));
                    const float e2 = fmaf(E2.x, lu, fmaf(E2.y, lv, E2.z));
                    const float t = fmaf(E0.w, lu, fmaf(E1.w, lv, E2.w));
                    // ties -> smallest index, as O-step 4 (the list is in index order)
                    if (fminf(e0, fminf(e1, e2)) >= 0.0f && t < tbest) { tbest = t; best = c; }
                }
                if (INSTR && on) bc.tri2d += (unsigned)ng;
                if (!on) best = -1;
                int fate = -1, src = -1, depth = 0;
                unsigned long long sig = 0;
                if (on) {
                    if (best < 0) cn.pmiss++;
                    else {
                        atomicAdd(&s_hist[warp][0], 1u);
                        if (INSTR) sig = (unsigned long long)(a.dz.perm[tbase + best] + 1);
                        fate = shade<TORQUE, 0u, GLOSSY, ANALOG ? 1 : 0>(W.tri[3 * best], W.tri[3 * best + 1], W.tri[3 * best + 2], tbest, best, g, i, a.B,
                                     a.deposit, o, d, src, depth, acc, acc_t, MASKS ? a.dz.esc : nullptr, tbase + best, a.dz.shin);
                        if (MASKS && fate == SHADE_ESCAPES) { cn.segments++; cn.escaped++; cn.mesc++; }
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
                while (qcount >= 32) secondary_pass();
            }
        }
        while (qcount > 0) secondary_pass();

        // S7: warp reduction in fp64, then one fixed-point atomic per component
        flush_tile_acc<TORQUE>(a, p, acc, acc_t, lane);
    }
    flush_counters<INSTR>(a, cn, s_hist[warp], lane);
    flush_beam_counters(a, bc, lane);
}

} // namespace

int srp_small_blocks_per_sm() { return blocks_per_sm(small_beam_kernel<false, false, false, false, false>); }

cudaError_t srp_launch_small(const TraceArgs &a, bool instrumented, int num_sms, cudaStream_t stream)
{
    const size_t dyn_smem = 0;
    return a.dz.esc ? SRP_LAUNCH3(small_beam_kernel, true,) : SRP_LAUNCH3(small_beam_kernel, false,);
}
