// srp_api.cu -- the extern "C" boundary of libsrp_b200 (include/srp.h): argument validation,
// handle ownership, workspace, and the enqueue order of the kernels in mesh_gen.cu / lbvh.cu /
// trace.cu.  No arithmetic of the method lives here.
#include <cstdio>
#include <cmath>
#include <cstring>
#include <new>
#include "srp_internal.cuh"
#include "escape_bins.cuh"

namespace {

srp_status fail(srp_context *ctx, srp_status st, const char *what, cudaError_t e = cudaSuccess)
{
    if (ctx) {
        ctx->last_error = what;
        if (e != cudaSuccess) { ctx->last_error += ": "; ctx->last_error += cudaGetErrorString(e); }
    }
    return st;
}

srp_status cuda_fail(srp_context *ctx, const char *what, cudaError_t e)
{
    return fail(ctx, e == cudaErrorMemoryAllocation ? SRP_ERR_OOM : SRP_ERR_CUDA, what, e);
}

void count_launches(srp_context *ctx, unsigned n) { ctx->launches_total += n; ctx->launches_call += n; }

#define TRY_CUDA(ctx, call, what) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(ctx, what, e_); } while (0)

// design arrays come from the context's own stream-ordered pool (no device-wide synchronisation per build; the
// device's default pool is left alone)
cudaError_t pool_alloc(srp_context *ctx, void **p, size_t bytes)
{
    return cudaMallocFromPoolAsync(p, bytes, ctx->mempool, ctx->stream);
}
template <typename T> cudaError_t pool_alloc(srp_context *ctx, T **p, size_t bytes) { return pool_alloc(ctx, (void **)p, bytes); }

// Fixed-point scale of the accumulators: the largest power of two <= 2^32 with which N photons of at most B + 1 hits
// (each deposit at most 2 photon weights; torque arms are summed in units of the design's extent) stay below 2^62.
double acc_scale_for(double photons, int B)
{
    const double bound = photons * 2.0 * (double)(B + 2);
    int bits = SRP_ACC_BITS_MAX;
    while (bits > 0 && bound * ldexp(1.0, bits) >= ldexp(1.0, 62)) --bits;
    return ldexp(1.0, bits);
}

void free_designs_mem(srp_context *ctx, srp_designs *d)
{
    void *ptrs[11] = { d->verts_orig, d->mats_orig, d->tri, d->nodes, d->tri_off_dev, d->box, d->perm, d->esc, d->nplane, d->shin, d->nodes4 };
    for (void *q : ptrs)
        if (q) cudaFreeAsync(q, ctx->stream);
}

// allocates everything that depends on tri_off / sumT
srp_status alloc_designs(srp_context *ctx, srp_designs *d)
{
    const long long sumT = d->sumT;
    TRY_CUDA(ctx, pool_alloc(ctx, &d->verts_orig, sizeof(float) * 9 * sumT), "alloc verts");
    TRY_CUDA(ctx, pool_alloc(ctx, &d->mats_orig, sizeof(float) * 3 * sumT), "alloc mats");
    TRY_CUDA(ctx, pool_alloc(ctx, &d->tri, sizeof(float4) * 3 * sumT), "alloc packed triangles");
    if (d->has_bvh) TRY_CUDA(ctx, pool_alloc(ctx, &d->nodes, sizeof(float4) * 4 * sumT), "alloc nodes");
#ifdef SRP_BVH4
    if (d->has_bvh) TRY_CUDA(ctx, pool_alloc(ctx, &d->nodes4, sizeof(float4) * 8 * sumT), "alloc wide nodes");
#endif
    TRY_CUDA(ctx, pool_alloc(ctx, &d->tri_off_dev, sizeof(long long) * (d->D + 1)), "alloc offsets");
    TRY_CUDA(ctx, pool_alloc(ctx, &d->box, sizeof(float4) * 2 * d->D), "alloc boxes");
    TRY_CUDA(ctx, pool_alloc(ctx, &d->perm, sizeof(int) * sumT), "alloc perm");
    TRY_CUDA(ctx, cudaMemcpyAsync(d->tri_off_dev, d->tri_off.data(), sizeof(long long) * (d->D + 1),
                                  cudaMemcpyHostToDevice, ctx->stream), "copy offsets");
    // d->tri_off (the pageable source) lives as long as the handle
    return SRP_OK;
}

srp_status ensure_workspace(srp_context *ctx, size_t accum_items)
{
    if (!ctx->stats) TRY_CUDA(ctx, cudaMalloc(&ctx->stats, sizeof(DevStats)), "alloc stats");
    if (!ctx->rounds_total) {
        TRY_CUDA(ctx, cudaMalloc(&ctx->rounds_total, sizeof(unsigned long long)), "alloc round counter");
        TRY_CUDA(ctx, cudaMemsetAsync(ctx->rounds_total, 0, sizeof(unsigned long long), ctx->stream), "zero round counter");
    }
    if (!ctx->work_counter) TRY_CUDA(ctx, cudaMalloc(&ctx->work_counter, SRP_PIPES * sizeof(unsigned long long)), "alloc counter");
    if (ctx->accum_items < accum_items) {
        TRY_CUDA(ctx, cudaStreamSynchronize(ctx->stream), "sync before workspace growth");
        cudaFree(ctx->accum); ctx->accum = nullptr; ctx->accum_items = 0;
        TRY_CUDA(ctx, cudaMalloc(&ctx->accum, sizeof(long long) * accum_items), "alloc accumulators");
        ctx->accum_items = accum_items;
    }
    return SRP_OK;
}

// Beam tracing of the primaries (trace_beam.cu, beam_trace_kernel) pays when many rays share a triangle: a
// beam's candidate list is then short and serves many rays.  With about one ray per triangle (the
// 1M-triangle sail at N = 2^20) every beam overflows its lists, so primaries walk the BVH one by one.
bool want_beams(const srp_context *ctx, bool brute, long long max_tris, long long N, long long n_pairs)
{
    if (brute || ctx->opt.sampler != 0 || n_pairs >= (1LL << 32)) return false;   // pool entries hold p in 32 bits
    if (ctx->opt.primary_mode == 1) return false;
    if (ctx->opt.primary_mode == 2) return true;
    return N >= 8 * max_tris;
}

// The ray queues between the beam kernel and the bounce kernel.  The beam warps of a
// pipeline stop taking tiles once rq_high rays are queued; every resident warp may still add the rays of the tile it
// is working on, hence the reserve.  The memory is the caller's (srp_set_workspace) or, failing that, allocated here
// once.  Sets a.rq_* for ONE queue over all of the memory; launch_trace_all shares it out among the pipelines.
size_t queue_reserve(const srp_context *ctx, int tile_rays)
{
    // slots the resident beam warps can still take after the high-water mark: a tile's rays each, in chunks of 256 of
    // which up to 31 stay unfilled (marked dead) when a push does not fit
    return (size_t)srp_beam_warps(ctx->num_sms) * ((size_t)tile_rays + (size_t)tile_rays / 7 + 512);
}

srp_status ensure_queue(srp_context *ctx, TraceArgs &a, bool brute, bool instrumented)
{
    a.rq = nullptr; a.rq_cap = 0; a.rq_high = 0; a.rq_ctr = nullptr;
    if (!want_beams(ctx, brute, a.max_tris, a.N, a.n_pairs)) return SRP_OK;
    const size_t fields = instrumented ? SRP_RQ_FIELDS_INSTR : SRP_RQ_FIELDS;
    const size_t reserve = queue_reserve(ctx, a.tile_rays);
    const size_t min_rays = reserve + (1u << 20);
    if (!ctx->rq_ctr) {
        TRY_CUDA(ctx, cudaMalloc(&ctx->rq_ctr, 4 * SRP_PIPES * sizeof(unsigned)), "alloc queue counters");
        TRY_CUDA(ctx, cudaMemsetAsync(ctx->rq_ctr, 0, 4 * SRP_PIPES * sizeof(unsigned), ctx->stream), "zero queue counters");
    }
    if (ctx->rq_words < min_rays * fields) {
        if (ctx->rq && !ctx->rq_owned)
            return fail(ctx, SRP_ERR_OOM, "the workspace given to srp_set_workspace is too small for this call's ray queue");
        TRY_CUDA(ctx, cudaStreamSynchronize(ctx->stream), "sync before queue growth");
        cudaFree(ctx->rq); ctx->rq = nullptr; ctx->rq_words = 0; ctx->rq_owned = false;
        // Every round of a loop ends with a tail in which SMs idle; two pipelines hide each other's tails, and the
        // more rays a queue holds beyond its reserve, the fewer rounds there are: 128 M slots more by default
        // (4.6 GB; cfg3 against 32 M / 64 M / 256 M slots: +3.5 % / +1.2 % / -1.1 % time).  A caller who wants
        // another trade gives the workspace (srp_set_workspace).
#ifndef SRP_RQ_EXTRA
#define SRP_RQ_EXTRA (128u << 20)
#endif
        size_t rays = SRP_PIPES * min_rays + (size_t)(SRP_RQ_EXTRA);
        cudaError_t e = cudaMalloc(&ctx->rq, sizeof(unsigned) * rays * fields);
        if (e != cudaSuccess) {                                 // less room than we would like: the smallest queue that works
            cudaGetLastError();
            rays = min_rays;
            e = cudaMalloc(&ctx->rq, sizeof(unsigned) * rays * fields);
        }
        if (e != cudaSuccess) return cuda_fail(ctx, "alloc ray queue", e);
        ctx->rq_words = rays * fields; ctx->rq_owned = true;
    }
    const size_t rays = ctx->rq_words / fields;
    a.rq = ctx->rq; a.rq_ctr = ctx->rq_ctr;
    a.rq_cap = (unsigned)(rays < 0xfffffff0u ? rays : 0xfffffff0u);
    a.rq_high = (unsigned)(a.rq_cap - reserve);
    return SRP_OK;
}

// Destroys the loop graphs of earlier calls that have finished (all of them when `all`, after a sync by the caller).
void reap_graphs(srp_context *ctx, bool all)
{
    size_t keep = 0;
    for (size_t x = 0; x < ctx->graphs.size(); ++x) {
        srp_context::PendingGraph &g = ctx->graphs[x];
        if (all || cudaEventQuery(g.done) == cudaSuccess) {
            cudaGraphExecDestroy(g.exec); cudaGraphDestroy(g.graph); cudaEventDestroy(g.done);
        } else ctx->graphs[keep++] = g;
    }
    cudaGetLastError();                                        // cudaErrorNotReady of the query is not an error
    ctx->graphs.resize(keep);
}

// Enqueues S2-S7.  With beams: the beam kernel (primaries) and the bounce kernel (everything queued) alternate until
// the tiles run out.  How often is known only on the device (it depends on how many photons go on), so the loop is
// a conditional WHILE node of a CUDA graph: body = beam kernel, bounce kernel, and a one-thread kernel that sets the
// condition from the tile counter.  Nothing is synchronised and no launch is wasted.  Every round ends with a tail
// in which SMs run out of work (the last heavy tiles, the last long photon paths); so the tiles are shared out among
// SRP_PIPES such loops with a queue each, independent nodes of the same graph, and one loop's kernels fill the SMs
// that the other's tail leaves idle.
srp_status launch_trace_all(srp_context *ctx, const TraceArgs &a, bool brute, bool instrumented)
{
    if (!a.rq) {
        TRY_CUDA(ctx, srp_launch_trace(a, brute, instrumented, ctx->num_sms, ctx->stream), "trace launch");
        count_launches(ctx, 1);
        return SRP_OK;
    }
    const size_t fields = instrumented ? SRP_RQ_FIELDS_INSTR : SRP_RQ_FIELDS;
    const size_t reserve = queue_reserve(ctx, a.tile_rays);
    const unsigned long long total_tiles = (unsigned long long)a.n_pairs * a.tiles_per_pair;
    int pipes = SRP_PIPES;
    if (ctx->opt.plain_launches || total_tiles < 64 || (size_t)a.rq_cap < SRP_PIPES * (reserve + (1u << 20))) pipes = 1;
    // Shares of the tiles and of the queue memory beyond the reserves (uneven shares, tried so that the loops' rounds
    // would not fall into step, change nothing: 0.5 ... 0.7 all within 1 %).
#ifndef SRP_PIPE_SHARE0
#define SRP_PIPE_SHARE0 0.5
#endif
    const double share[SRP_PIPES] = { pipes == 1 ? 1.0 : SRP_PIPE_SHARE0, 1.0 - SRP_PIPE_SHARE0 };
    const size_t extra = (size_t)a.rq_cap - (size_t)pipes * reserve;
    TraceArgs ap[SRP_PIPES];
    size_t ray0 = 0;
    unsigned long long tile0 = 0;
    for (int q = 0; q < pipes; ++q) {
        ap[q] = a;
        ap[q].tile_begin = tile0;
        ap[q].tile_end = q == pipes - 1 ? total_tiles : tile0 + (unsigned long long)((double)total_tiles * share[q]);
        tile0 = ap[q].tile_end;
        ap[q].work_counter = a.work_counter + q;
        ap[q].rq_ctr = a.rq_ctr + 4 * q;
        ap[q].rq_cap = (unsigned)(reserve + (size_t)((double)extra * share[q]));
        ap[q].rq = a.rq + ray0 * fields;
        ray0 += ap[q].rq_cap;
        ap[q].rq_high = (unsigned)(ap[q].rq_cap - reserve);
    }
    count_launches(ctx, pipes);                               // at least one beam launch each; the rounds are counted on the device
    if (ctx->opt.plain_launches) {                          // a sufficient number of rounds; surplus ones find nothing to do
        const long long rounds = (long long)((double)a.n_pairs * (double)a.N / (double)ap[0].rq_high) + 1;
        for (long long r = 0; r < rounds; ++r) {
            TRY_CUDA(ctx, srp_launch_trace(ap[0], brute, instrumented, ctx->num_sms, ctx->stream), "beam launch");
            TRY_CUDA(ctx, srp_launch_bounce(ap[0], instrumented, ctx->num_sms, ctx->stream), "bounce launch");
        }
        return SRP_OK;
    }
    reap_graphs(ctx, false);
    srp_context::PendingGraph g = { nullptr, nullptr, nullptr };
    cudaError_t e = cudaGraphCreate(&g.graph, 0);
    for (int q = 0; q < pipes && e == cudaSuccess; ++q) {
        if (!ctx->capture_stream[q]) e = cudaStreamCreateWithFlags(&ctx->capture_stream[q], cudaStreamNonBlocking);
        cudaGraphConditionalHandle handle;
        if (e == cudaSuccess) e = cudaGraphConditionalHandleCreate(&handle, g.graph, 1, cudaGraphCondAssignDefault);
        cudaGraphNodeParams cp = { cudaGraphNodeTypeConditional };
        cp.conditional.handle = handle; cp.conditional.type = cudaGraphCondTypeWhile; cp.conditional.size = 1;
        cudaGraphNode_t cnode;
        if (e == cudaSuccess) e = cudaGraphAddNode(&cnode, g.graph, nullptr, 0, &cp);      // no dependencies: the loops run side by side
        if (e != cudaSuccess) break;
        cudaGraph_t body = cp.conditional.phGraph_out[0];
        cudaStream_t cs = ctx->capture_stream[q];
        e = cudaStreamBeginCaptureToGraph(cs, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed);
        if (e == cudaSuccess) {
            cudaError_t e1 = srp_launch_trace(ap[q], brute, instrumented, ctx->num_sms, cs);
            if (e1 == cudaSuccess) e1 = srp_launch_bounce(ap[q], instrumented, ctx->num_sms, cs);
            if (e1 == cudaSuccess) e1 = srp_launch_loop_cond(handle, ap[q], cs);
            cudaGraph_t same = nullptr;
            e = cudaStreamEndCapture(cs, &same);
            if (e1 != cudaSuccess) e = e1;
        }
    }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&g.exec, g.graph, 0);
    if (e == cudaSuccess) e = cudaGraphLaunch(g.exec, ctx->stream);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&g.done, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventRecord(g.done, ctx->stream);
    if (e != cudaSuccess) {
        if (g.exec) cudaGraphExecDestroy(g.exec);
        if (g.graph) cudaGraphDestroy(g.graph);
        if (g.done) cudaEventDestroy(g.done);
        return cuda_fail(ctx, "beam / bounce loop graph", e);
    }
    ctx->graphs.push_back(g);
    return SRP_OK;
}

// Escape masks (escape_mask.cu) are built the first time a call can repay them: the build costs about 0.1 us per
// triangle, a masked bounce ray saves about 10 ps per segment of the call, so `rays` (all photons of the call) must
// exceed the triangle count by a few 10^4.  They stay with the handle afterwards.  escape_masks: 0 never, 1 this
// rule, 2 always.
srp_status ensure_masks(srp_context *ctx, const srp_designs *dz, double rays)
{
    srp_designs *d = const_cast<srp_designs *>(dz);           // a cache inside the handle, not a change of its meaning
    if (d->esc || d->esc_failed || ctx->opt.escape_masks == 0 || (d->has_bvh && d->D > 65535)) return SRP_OK;
    if (ctx->opt.escape_masks == 1 && rays < 32768.0 * (double)d->sumT) return SRP_OK;
    unsigned *esc = nullptr;
    float4 *nplane = nullptr;
    if (pool_alloc(ctx, &esc, sizeof(unsigned) * 2 * ESC_WORDS * d->sumT) != cudaSuccess ||
        (d->has_bvh && pool_alloc(ctx, &nplane, sizeof(float4) * 2 * d->sumT) != cudaSuccess)) {
        cudaGetLastError();                                   // no room: trace without masks
        if (esc) cudaFreeAsync(esc, ctx->stream);
        d->esc_failed = true;
        return SRP_OK;
    }
    cudaError_t e;
    if (d->has_bvh) {
        d->nplane = nplane;
        e = srp_launch_node_planes(d->dev(), d->sumT, nplane, ctx->stream);
        if (e == cudaSuccess) e = srp_launch_escape_masks(d->dev(), d->maxT, esc, ctx->stream);
    } else {
        e = srp_launch_escape_masks_small(d->dev(), d->sumT, esc, ctx->stream);   // T <= 64: every pair of triangles
    }
    if (e != cudaSuccess) { cudaFreeAsync(esc, ctx->stream); return cuda_fail(ctx, "escape mask build", e); }
    count_launches(ctx, d->has_bvh ? 2 : 1);
    d->esc = esc;
    return SRP_OK;
}

srp_status check_trace_args(srp_context *ctx, const srp_designs *dz, const float *sun_dirs, int S,
                            long long N, int B, const void *out)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!dz || !sun_dirs || !out) return fail(ctx, SRP_ERR_INVALID, "null pointer argument");
    if (S <= 0) return fail(ctx, SRP_ERR_INVALID, "S must be positive");
    if (N <= 0 || N > (1LL << 31)) return fail(ctx, SRP_ERR_INVALID, "rays_per_dir must be in [1, 2^31]");
    if (B < 0 || B > 15) return fail(ctx, SRP_ERR_INVALID, "max_bounces must be in [0, 15]");
    if (ctx->opt.sampler == 0 && (N & (N - 1)) != 0)
        return fail(ctx, SRP_ERR_INVALID, "stratified sampler needs rays_per_dir to be a power of two");
    return SRP_OK;
}

TraceArgs make_args(srp_context *ctx, const srp_designs *dz, const float *sun_dirs, int S, const int *pairs,
                    long long n_pairs, long long N, int B, unsigned long long seed)
{
    TraceArgs a;
    memset(&a, 0, sizeof a);
    a.dz = dz->dev();
    a.sun_dirs = sun_dirs; a.pairs = pairs; a.n_pairs = n_pairs; a.S = S; a.N = N; a.B = B;
    a.log2N = 0;
    while ((1LL << a.log2N) < N) ++a.log2N;
    a.key0 = (uint32_t)seed; a.key1 = (uint32_t)(seed >> 32);
    a.sampler = ctx->opt.sampler; a.deposit = ctx->opt.deposit; a.P = ctx->opt.solar_pressure;
    a.accum = ctx->accum; a.acc_stride = 3; a.torque = 0; a.xcom = nullptr;
    a.stats = ctx->stats; a.work_counter = ctx->work_counter; a.rounds_total = ctx->rounds_total;
    a.acc_scale = acc_scale_for((double)N, B);
    // tile size: large tiles amortise the per-item set-up and the drain at the end of a tile; shrink
    // them only when there would be too few items to occupy every resident warp several times
    const bool brute = !dz->has_bvh;
    a.max_tris = dz->maxT;
    a.primary_mode = ctx->opt.primary_mode;
    const bool beam = brute ? (ctx->opt.sampler == 0 && ctx->opt.primary_mode != 1)
                            : want_beams(ctx, ctx->opt.force_brute != 0, a.max_tris, N, n_pairs);
    const long long warps = (long long)ctx->num_sms * srp_trace_blocks_per_sm(brute, beam);
#ifndef SRP_BEAM_TILE_MAX
#define SRP_BEAM_TILE_MAX 4096     // beam tiles: half the reserve of the ray queues (there is one per pipeline); same speed as 8192
#endif
    long long tile = (beam && !brute) ? SRP_BEAM_TILE_MAX : 8192;
    if (tile > N) tile = N;
    while (tile > 256 && n_pairs * ((N + tile - 1) / tile) < 8 * warps) tile >>= 1;
    a.tile_rays = (int)tile;
    a.tiles_per_pair = (N + tile - 1) / tile;
    a.tile_begin = 0; a.tile_end = (unsigned long long)n_pairs * a.tiles_per_pair;
    return a;
}

// out_second != nullptr: a second output from the same trace -- second = 1: the torque about x_com (DEVICE float[D,3],
// or nullptr = the origin), Eq. 4; second = 2: the direct part of the force.
srp_status run_forces(srp_context *ctx, const srp_designs *dz, const float *sun_dirs, int S, const int *pairs,
                      long long n_pairs, long long N, int B, unsigned long long seed, float *out,
                      const float *x_com = nullptr, float *out_second = nullptr, int second = 1)
{
    float *out_torques = out_second;
    const int stride = out_torques ? 6 : 3;
    ctx->launches_call = 0;
    if (out_torques && ctx->opt.instrumented)
        return fail(ctx, SRP_ERR_UNSUPPORTED, "a second output is not available from the instrumented kernels");
    srp_status st = ensure_workspace(ctx, (size_t)n_pairs * stride);
    if (st != SRP_OK) return st;
    if (B > 0 && !(ctx->opt.force_brute != 0)) {
        st = ensure_masks(ctx, dz, (double)n_pairs * (double)N);
        if (st != SRP_OK) return st;
    }
    TraceArgs a = make_args(ctx, dz, sun_dirs, S, pairs, n_pairs, N, B, seed);
    a.accum = ctx->accum; a.acc_stride = stride; a.torque = out_torques ? second : 0; a.xcom = x_com;
    if (ctx->opt.escape_masks == 0) a.dz.esc = nullptr;        // masks an earlier call built stay unused
    TRY_CUDA(ctx, cudaMemsetAsync(ctx->accum, 0, sizeof(long long) * stride * n_pairs, ctx->stream), "zero accumulators");
    TRY_CUDA(ctx, cudaMemsetAsync(ctx->stats, 0, sizeof(DevStats), ctx->stream), "zero stats");
    TRY_CUDA(ctx, cudaMemsetAsync(ctx->work_counter, 0, SRP_PIPES * sizeof(unsigned long long), ctx->stream), "zero counter");
    const bool brute = !dz->has_bvh || ctx->opt.force_brute != 0;
    st = ensure_queue(ctx, a, brute, ctx->opt.instrumented != 0);
    if (st != SRP_OK) return st;
    st = launch_trace_all(ctx, a, brute, ctx->opt.instrumented != 0);
    if (st != SRP_OK) return st;
    TRY_CUDA(ctx, srp_launch_finalize(a, out, out_torques, ctx->stream), "finalize launch");
    count_launches(ctx, 1);
    return SRP_OK;
}

} // namespace

extern "C" {

srp_status srp_create(srp_context **out, int cuda_device, void *cuda_stream)
{
    if (!out) return SRP_ERR_INVALID;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || cuda_device < 0 || cuda_device >= count)
        return SRP_ERR_CUDA;                      // no device: there is no CPU fallback
    if (cudaSetDevice(cuda_device) != cudaSuccess) return SRP_ERR_CUDA;
    srp_context *ctx = new (std::nothrow) srp_context();
    if (!ctx) return SRP_ERR_OOM;
    ctx->device = cuda_device;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->opt.solar_pressure = 4.56e-6; ctx->opt.sampler = 0; ctx->opt.deposit = 0;
    ctx->opt.force_brute = 0; ctx->opt.instrumented = 0; ctx->opt.primary_mode = 0; ctx->opt.escape_masks = 1;
    ctx->opt.plain_launches = 0; ctx->opt.leaf_max = 0; ctx->opt.bvh_builder = 0;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cuda_device) == cudaSuccess) ctx->num_sms = prop.multiProcessorCount;
    {   // a pool of the context's own that keeps freed blocks: builds reuse them instead of going back to the driver
        cudaMemPoolProps props;
        memset(&props, 0, sizeof props);
        props.allocType = cudaMemAllocationTypePinned; props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice; props.location.id = cuda_device;
        if (cudaMemPoolCreate(&ctx->mempool, &props) != cudaSuccess) { delete ctx; return SRP_ERR_CUDA; }
        unsigned long long keep = ~0ULL;
        cudaMemPoolSetAttribute(ctx->mempool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    *out = ctx;
    return SRP_OK;
}

srp_status srp_destroy(srp_context *ctx)
{
    if (!ctx) return SRP_ERR_INVALID;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    reap_graphs(ctx, true);
    for (cudaStream_t cs : ctx->capture_stream)
        if (cs) cudaStreamDestroy(cs);
    cudaFree(ctx->accum); cudaFree(ctx->stats); cudaFree(ctx->work_counter); cudaFree(ctx->rq_ctr);
    if (ctx->rq_owned) cudaFree(ctx->rq);
    cudaFree(ctx->stage_dirs); cudaFree(ctx->stage_out);
    cudaFree(ctx->rounds_total);
    if (ctx->mempool) cudaMemPoolDestroy(ctx->mempool);       // designs not freed by now go with it
    delete ctx;
    return SRP_OK;
}

srp_status srp_set_options(srp_context *ctx, const srp_options *opt)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!opt) return fail(ctx, SRP_ERR_INVALID, "null options");
    if (!(opt->solar_pressure > 0.0) || opt->sampler < 0 || opt->sampler > 1 || opt->deposit < 0 || opt->deposit > 1 ||
        opt->primary_mode < 0 || opt->primary_mode > 2 || opt->escape_masks < 0 || opt->escape_masks > 2 ||
        opt->plain_launches < 0 || opt->plain_launches > 1 || opt->leaf_max < 0 || opt->leaf_max > 8 ||
        opt->bvh_builder < 0 || opt->bvh_builder > 1)
        return fail(ctx, SRP_ERR_INVALID, "option out of range");
    ctx->opt = *opt;
    return SRP_OK;
}

srp_status srp_get_options(const srp_context *ctx, srp_options *opt)
{
    if (!ctx || !opt) return SRP_ERR_INVALID;
    *opt = ctx->opt;
    return SRP_OK;
}

const char *srp_last_error(const srp_context *ctx) { return ctx ? ctx->last_error.c_str() : "null context"; }

int srp_family_n_params(srp_family family)
{
    switch (family) {
    case SRP_FAMILY_PLATE: return 3; case SRP_FAMILY_BOXWING: return 2; case SRP_FAMILY_DETAILED: return 2;
    case SRP_FAMILY_BOXWING6: return 6; case SRP_FAMILY_SAIL: return 1; case SRP_FAMILY_BOXWING_T: return 2; default: return -1;
    }
}

long long srp_family_tri_count(srp_family family) { return srp_family_tris_host((int)family); }

srp_status srp_build_designs(srp_context *ctx, srp_family family, const float *theta, int D, int n_params,
                             unsigned long long mesh_seed, srp_designs **out)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!out) return fail(ctx, SRP_ERR_INVALID, "null output handle");
    *out = nullptr;
    const long long T = srp_family_tris_host((int)family);
    if (T < 0) return fail(ctx, SRP_ERR_INVALID, "unknown family");
    if (!theta) return fail(ctx, SRP_ERR_INVALID, "null theta");
    if (D <= 0 || D > 65535) return fail(ctx, SRP_ERR_INVALID, "D must be in [1, 65535]");
    if (n_params != srp_family_n_params(family)) return fail(ctx, SRP_ERR_INVALID, "wrong n_params for this family");
    if ((long long)D * T >= (1LL << 31)) return fail(ctx, SRP_ERR_INVALID, "too many triangles in one batch");
    if (T >= (1LL << 27) - 1) return fail(ctx, SRP_ERR_INVALID, "design too large (a ray's source triangle is a 27-bit field)");
    cudaSetDevice(ctx->device);
    srp_designs *d = new (std::nothrow) srp_designs();
    if (!d) return fail(ctx, SRP_ERR_OOM, "host allocation");
    d->D = D; d->family = (int)family; d->sumT = (long long)D * T; d->maxT = T;
    d->tri_off.resize(D + 1);
    for (int k = 0; k <= D; ++k) d->tri_off[k] = (long long)k * T;
    d->has_bvh = T > SRP_BRUTE_MAX_TRIS;
    srp_status st = alloc_designs(ctx, d);
    if (st != SRP_OK) { free_designs_mem(ctx, d); delete d; return st; }
    cudaError_t e = srp_launch_mesh_gen((int)family, theta, D, n_params, mesh_seed, T, d->verts_orig,
                                        d->mats_orig, ctx->mempool, 0u, ctx->stream);
    int build_launches = 0;
    if (e == cudaSuccess) e = srp_launch_build(d, ctx->opt.leaf_max, ctx->opt.bvh_builder, ctx->mempool, ctx->stream, &build_launches);
    if (e == cudaSuccess && d->nodes4) { e = srp_launch_collapse4(d, ctx->stream); ++build_launches; }
    if (e != cudaSuccess) { free_designs_mem(ctx, d); delete d; return cuda_fail(ctx, "design build", e); }
    ctx->launches_total += 2 + build_launches;                         // mesh generation: 2 kernels
    *out = d;
    return SRP_OK;
}

srp_status srp_build_designs_from_meshes(srp_context *ctx, const float *verts, const float *mats,
                                         const long long *tri_offsets, int D, srp_designs **out)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!out) return fail(ctx, SRP_ERR_INVALID, "null output handle");
    *out = nullptr;
    if (!verts || !mats || !tri_offsets) return fail(ctx, SRP_ERR_INVALID, "null pointer argument");
    if (D <= 0 || D > 65535) return fail(ctx, SRP_ERR_INVALID, "D must be in [1, 65535]");
    if (tri_offsets[0] != 0) return fail(ctx, SRP_ERR_INVALID, "tri_offsets[0] must be 0");
    long long maxT = 0;
    for (int k = 0; k < D; ++k) {
        const long long t = tri_offsets[k + 1] - tri_offsets[k];
        if (t <= 0) return fail(ctx, SRP_ERR_INVALID, "tri_offsets must be strictly increasing");
        if (t >= (1LL << 27) - 1) return fail(ctx, SRP_ERR_INVALID, "design too large (a ray's source triangle is a 27-bit field)");
        if (t > maxT) maxT = t;
    }
    if (tri_offsets[D] >= (1LL << 31)) return fail(ctx, SRP_ERR_INVALID, "too many triangles in one batch");
    cudaSetDevice(ctx->device);
    srp_designs *d = new (std::nothrow) srp_designs();
    if (!d) return fail(ctx, SRP_ERR_OOM, "host allocation");
    d->D = D; d->family = -1; d->sumT = tri_offsets[D]; d->maxT = maxT;
    d->tri_off.assign(tri_offsets, tri_offsets + D + 1);
    d->has_bvh = maxT > SRP_BRUTE_MAX_TRIS;
    srp_status st = alloc_designs(ctx, d);
    if (st != SRP_OK) { free_designs_mem(ctx, d); delete d; return st; }
    cudaError_t e = cudaMemcpyAsync(d->verts_orig, verts, sizeof(float) * 9 * d->sumT, cudaMemcpyDeviceToDevice, ctx->stream);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(d->mats_orig, mats, sizeof(float) * 3 * d->sumT, cudaMemcpyDeviceToDevice, ctx->stream);
    int build_launches = 0;
    if (e == cudaSuccess) e = srp_launch_build(d, ctx->opt.leaf_max, ctx->opt.bvh_builder, ctx->mempool, ctx->stream, &build_launches);
    if (e == cudaSuccess && d->nodes4) { e = srp_launch_collapse4(d, ctx->stream); ++build_launches; }
    if (e != cudaSuccess) { free_designs_mem(ctx, d); delete d; return cuda_fail(ctx, "design build", e); }
    ctx->launches_total += build_launches;
    *out = d;
    return SRP_OK;
}

srp_status srp_designs_info(const srp_designs *dz, int *D, long long *tri_offsets_host)
{
    if (!dz) return SRP_ERR_INVALID;
    if (D) *D = dz->D;
    if (tri_offsets_host) memcpy(tri_offsets_host, dz->tri_off.data(), sizeof(long long) * (dz->D + 1));
    return SRP_OK;
}

srp_status srp_designs_read_mesh(srp_context *ctx, const srp_designs *dz, int design, float *verts_host,
                                 float *mats_host)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!dz || design < 0 || design >= dz->D) return fail(ctx, SRP_ERR_INVALID, "bad design index");
    cudaSetDevice(ctx->device);
    TRY_CUDA(ctx, cudaStreamSynchronize(ctx->stream), "sync");
    const long long b = dz->tri_off[design], T = dz->tri_off[design + 1] - b;
    if (verts_host) TRY_CUDA(ctx, cudaMemcpy(verts_host, dz->verts_orig + 9 * b, sizeof(float) * 9 * T, cudaMemcpyDeviceToHost), "read verts");
    if (mats_host) TRY_CUDA(ctx, cudaMemcpy(mats_host, dz->mats_orig + 3 * b, sizeof(float) * 3 * T, cudaMemcpyDeviceToHost), "read mats");
    return SRP_OK;
}

srp_status srp_designs_read_bvh(srp_context *ctx, const srp_designs *dz, int design, long long *n_nodes,
                                float *nodes_host, int *perm_host)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!dz || design < 0 || design >= dz->D) return fail(ctx, SRP_ERR_INVALID, "bad design index");
    cudaSetDevice(ctx->device);
    TRY_CUDA(ctx, cudaStreamSynchronize(ctx->stream), "sync");
    const long long b = dz->tri_off[design], T = dz->tri_off[design + 1] - b;
    const long long nn = dz->has_bvh ? (T > 1 ? T - 1 : 1) : 0;
    if (n_nodes) *n_nodes = nn;
    if (nodes_host && nn > 0)
        TRY_CUDA(ctx, cudaMemcpy(nodes_host, dz->nodes + 4 * b, sizeof(float4) * 4 * nn, cudaMemcpyDeviceToHost), "read nodes");
    if (perm_host) TRY_CUDA(ctx, cudaMemcpy(perm_host, dz->perm + b, sizeof(int) * T, cudaMemcpyDeviceToHost), "read perm");
    return SRP_OK;
}

srp_status srp_designs_set_shininess(srp_context *ctx, srp_designs *dz, const float *shininess)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!dz) return fail(ctx, SRP_ERR_INVALID, "null designs handle");
    cudaSetDevice(ctx->device);
    if (!shininess) {                                  // back to ideal mirrors
        if (dz->shin) cudaFreeAsync(dz->shin, ctx->stream);
        dz->shin = nullptr;
        return SRP_OK;
    }
    if (!dz->shin) TRY_CUDA(ctx, pool_alloc(ctx, &dz->shin, sizeof(float) * dz->sumT), "alloc shininess");
    TRY_CUDA(ctx, srp_launch_gather_shininess(dz->dev(), dz->sumT, shininess, dz->shin, ctx->stream), "shininess gather");
    return SRP_OK;
}

srp_status srp_free_designs(srp_context *ctx, srp_designs *dz)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!dz) return SRP_OK;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    free_designs_mem(ctx, dz);
    delete dz;
    return SRP_OK;
}

srp_status srp_forces(srp_context *ctx, const srp_designs *dz, const float *sun_dirs, int S, long long N, int B,
                      unsigned long long seed, float *out)
{
    srp_status st = check_trace_args(ctx, dz, sun_dirs, S, N, B, out);
    if (st != SRP_OK) return st;
    cudaSetDevice(ctx->device);
    return run_forces(ctx, dz, sun_dirs, S, nullptr, (long long)dz->D * S, N, B, seed, out);
}

srp_status srp_forces_torques(srp_context *ctx, const srp_designs *dz, const float *sun_dirs, int S, long long N, int B,
                              unsigned long long seed, const float *x_com, float *out_forces, float *out_torques)
{
    srp_status st = check_trace_args(ctx, dz, sun_dirs, S, N, B, out_forces);
    if (st != SRP_OK) return st;
    if (!out_torques) return fail(ctx, SRP_ERR_INVALID, "null pointer argument");
    cudaSetDevice(ctx->device);
    return run_forces(ctx, dz, sun_dirs, S, nullptr, (long long)dz->D * S, N, B, seed, out_forces, x_com, out_torques);
}

srp_status srp_forces_torques_pairs(srp_context *ctx, const srp_designs *dz, const float *sun_dirs, int S,
                                    const int *pairs, long long n_pairs, long long N, int B, unsigned long long seed,
                                    const float *x_com, float *out_forces, float *out_torques)
{
    srp_status st = check_trace_args(ctx, dz, sun_dirs, S, N, B, out_forces);
    if (st != SRP_OK) return st;
    if (!out_torques) return fail(ctx, SRP_ERR_INVALID, "null pointer argument");
    if (!pairs || n_pairs <= 0) return fail(ctx, SRP_ERR_INVALID, "bad pair list");
    cudaSetDevice(ctx->device);
    return run_forces(ctx, dz, sun_dirs, S, pairs, n_pairs, N, B, seed, out_forces, x_com, out_torques);
}

srp_status srp_forces_split(srp_context *ctx, const srp_designs *dz, const float *sun_dirs, int S, long long N, int B,
                            unsigned long long seed, float *out_forces, float *out_direct)
{
    srp_status st = check_trace_args(ctx, dz, sun_dirs, S, N, B, out_forces);
    if (st != SRP_OK) return st;
    if (!out_direct) return fail(ctx, SRP_ERR_INVALID, "null pointer argument");
    cudaSetDevice(ctx->device);
    return run_forces(ctx, dz, sun_dirs, S, nullptr, (long long)dz->D * S, N, B, seed, out_forces, nullptr, out_direct, 2);
}

srp_status srp_forces_split_pairs(srp_context *ctx, const srp_designs *dz, const float *sun_dirs, int S, const int *pairs,
                                  long long n_pairs, long long N, int B, unsigned long long seed, float *out_forces,
                                  float *out_direct)
{
    srp_status st = check_trace_args(ctx, dz, sun_dirs, S, N, B, out_forces);
    if (st != SRP_OK) return st;
    if (!out_direct) return fail(ctx, SRP_ERR_INVALID, "null pointer argument");
    if (!pairs || n_pairs <= 0) return fail(ctx, SRP_ERR_INVALID, "bad pair list");
    cudaSetDevice(ctx->device);
    return run_forces(ctx, dz, sun_dirs, S, pairs, n_pairs, N, B, seed, out_forces, nullptr, out_direct, 2);
}

srp_status srp_thermal_forces(srp_context *ctx, const srp_designs *dz, const float *facet_power, long long N, int B,
                              unsigned long long seed, float *out_forces)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!dz || !facet_power || !out_forces) return fail(ctx, SRP_ERR_INVALID, "null pointer argument");
    if (N <= 0 || N > (1LL << 31)) return fail(ctx, SRP_ERR_INVALID, "rays_per_facet must be in [1, 2^31]");
    if (B < 0 || B > 15) return fail(ctx, SRP_ERR_INVALID, "max_bounces must be in [0, 15]");
    if (dz->sumT >= (1LL << 31)) return fail(ctx, SRP_ERR_UNSUPPORTED, "too many triangles for the emitter list");
    cudaSetDevice(ctx->device);
    ctx->launches_call = 0;
    srp_status st = ensure_workspace(ctx, (size_t)dz->D * 3);
    if (st != SRP_OK) return st;
    st = ensure_masks(ctx, dz, (double)N * (double)dz->sumT);
    if (st != SRP_OK) return st;
    TraceArgs a;
    memset(&a, 0, sizeof a);
    a.dz = dz->dev();
    a.n_pairs = dz->D; a.S = 1; a.N = N; a.B = B;
    if (ctx->opt.escape_masks == 0) a.dz.esc = nullptr;
    a.key0 = (uint32_t)seed; a.key1 = (uint32_t)(seed >> 32);
    a.sampler = 0; a.deposit = ctx->opt.deposit; a.P = ctx->opt.solar_pressure;
    a.accum = ctx->accum; a.acc_stride = 3; a.stats = ctx->stats; a.work_counter = ctx->work_counter;
    a.rounds_total = ctx->rounds_total;
    a.acc_scale = acc_scale_for((double)N, B + 1);             // per design: the facets' weights |W_f| / P_k sum to 1
    a.tile_rays = (int)(N < 8192 ? N : 8192);
    a.tiles_per_pair = (N + a.tile_rays - 1) / a.tile_rays;
    int *emit_list = nullptr, *n_emit = nullptr;
    float *design_power = nullptr;
    cudaError_t e = pool_alloc(ctx, &emit_list, sizeof(int) * dz->sumT);
    if (e == cudaSuccess) e = pool_alloc(ctx, &n_emit, sizeof(int));
    if (e == cudaSuccess) e = pool_alloc(ctx, &design_power, sizeof(float) * dz->D);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->accum, 0, sizeof(long long) * 3 * dz->D, ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->stats, 0, sizeof(DevStats), ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->work_counter, 0, SRP_PIPES * sizeof(unsigned long long), ctx->stream);
    if (e == cudaSuccess)
        e = srp_launch_thermal(a, facet_power, dz->sumT, emit_list, n_emit, design_power, out_forces, ctx->num_sms, ctx->stream);
    if (emit_list) cudaFreeAsync(emit_list, ctx->stream);      // stream-ordered: after the kernels that use them
    if (n_emit) cudaFreeAsync(n_emit, ctx->stream);
    if (design_power) cudaFreeAsync(design_power, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, "thermal forces", e);
    count_launches(ctx, 4);
    return SRP_OK;
}

srp_status srp_forces_pairs(srp_context *ctx, const srp_designs *dz, const float *sun_dirs, int S, const int *pairs,
                            long long n_pairs, long long N, int B, unsigned long long seed, float *out)
{
    srp_status st = check_trace_args(ctx, dz, sun_dirs, S, N, B, out);
    if (st != SRP_OK) return st;
    if (!pairs || n_pairs <= 0) return fail(ctx, SRP_ERR_INVALID, "bad pair list");
    cudaSetDevice(ctx->device);
    return run_forces(ctx, dz, sun_dirs, S, pairs, n_pairs, N, B, seed, out);
}

srp_status srp_forces_host(srp_context *ctx, const srp_designs *dz, const float *sun_dirs_host, int S, long long N,
                           int B, unsigned long long seed, float *out_host)
{
    srp_status st = check_trace_args(ctx, dz, sun_dirs_host, S, N, B, out_host);
    if (st != SRP_OK) return st;
    cudaSetDevice(ctx->device);
    const size_t n_dirs = (size_t)S * 3, n_out = (size_t)dz->D * S * 3;
    if (ctx->stage_dirs_items < n_dirs) {
        cudaFree(ctx->stage_dirs); ctx->stage_dirs = nullptr; ctx->stage_dirs_items = 0;
        TRY_CUDA(ctx, cudaMalloc(&ctx->stage_dirs, sizeof(float) * n_dirs), "alloc staging");
        ctx->stage_dirs_items = n_dirs;
    }
    if (ctx->stage_out_items < n_out) {
        cudaFree(ctx->stage_out); ctx->stage_out = nullptr; ctx->stage_out_items = 0;
        TRY_CUDA(ctx, cudaMalloc(&ctx->stage_out, sizeof(float) * n_out), "alloc staging");
        ctx->stage_out_items = n_out;
    }
    TRY_CUDA(ctx, cudaMemcpyAsync(ctx->stage_dirs, sun_dirs_host, sizeof(float) * n_dirs, cudaMemcpyHostToDevice, ctx->stream), "h2d sun_dirs");
    st = run_forces(ctx, dz, ctx->stage_dirs, S, nullptr, (long long)dz->D * S, N, B, seed, ctx->stage_out);
    if (st != SRP_OK) return st;
    TRY_CUDA(ctx, cudaMemcpyAsync(out_host, ctx->stage_out, sizeof(float) * n_out, cudaMemcpyDeviceToHost, ctx->stream), "d2h forces");
    TRY_CUDA(ctx, cudaStreamSynchronize(ctx->stream), "sync");
    return SRP_OK;
}

srp_status srp_forces_per_sample(srp_context *ctx, srp_family family, const float *theta, int n_params,
                                 const float *sun_dirs, long long M, long long N, int B, unsigned long long seed,
                                 unsigned long long mesh_seed, float *out)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!theta || !sun_dirs || !out) return fail(ctx, SRP_ERR_INVALID, "null pointer argument");
    const long long T = srp_family_tris_host((int)family);
    if (T < 0) return fail(ctx, SRP_ERR_INVALID, "unknown family");
    if (n_params != srp_family_n_params(family)) return fail(ctx, SRP_ERR_INVALID, "wrong n_params for this family");
    if (T > srp_sample_max_tris()) return fail(ctx, SRP_ERR_UNSUPPORTED, "a record's mesh must fit a thread block's shared memory");
    if (M <= 0 || M >= (1LL << 32)) return fail(ctx, SRP_ERR_INVALID, "M must be in [1, 2^32)");
    if (N <= 0 || N > (1LL << 31)) return fail(ctx, SRP_ERR_INVALID, "rays_per_record must be in [1, 2^31]");
    if (B < 0 || B > 15) return fail(ctx, SRP_ERR_INVALID, "max_bounces must be in [0, 15]");
    if (ctx->opt.sampler == 0 && (N & (N - 1)) != 0)
        return fail(ctx, SRP_ERR_INVALID, "stratified sampler needs rays_per_record to be a power of two");
    cudaSetDevice(ctx->device);
    ctx->launches_call = 0;
    srp_status st = ensure_workspace(ctx, 3);
    if (st != SRP_OK) return st;
    TRY_CUDA(ctx, cudaMemsetAsync(ctx->stats, 0, sizeof(DevStats), ctx->stream), "zero stats");
    // chunks of records: meshes for a chunk (S0), then its photons (the kernel boxes and packs each record on the way in)
    long long chunk = (1LL << 30) / (96 * T);                       // ~1 GiB of mesh per chunk: many waves of blocks per launch
    if (chunk > 32768) chunk = 32768;
    if (chunk > M) chunk = M;
    if (chunk < 1) chunk = 1;
    srp_designs d;
    d.D = (int)chunk; d.family = (int)family; d.sumT = chunk * T; d.maxT = T; d.has_bvh = false;
    d.tri_off.resize(chunk + 1);
    for (long long k = 0; k <= chunk; ++k) d.tri_off[k] = k * T;
    st = alloc_designs(ctx, &d);
    cudaError_t e = cudaSuccess;
    for (long long m0 = 0; m0 < M && st == SRP_OK && e == cudaSuccess; m0 += chunk) {
        const int Dc = (int)(M - m0 < chunk ? M - m0 : chunk);
        d.D = Dc; d.sumT = (long long)Dc * T;
        e = srp_launch_mesh_gen((int)family, theta + (size_t)m0 * n_params, Dc, n_params, mesh_seed, T, d.verts_orig,
                                d.mats_orig, ctx->mempool, (unsigned)m0, ctx->stream);
        if (e != cudaSuccess) break;
        TraceArgs a;                                                // the sample kernel boxes and packs a record itself (S1 without a hierarchy)
        memset(&a, 0, sizeof a);
        a.dz = d.dev();
        a.sun_dirs = sun_dirs + 3 * m0; a.n_pairs = Dc; a.S = Dc; a.N = N; a.B = B;
        while ((1LL << a.log2N) < N) ++a.log2N;
        a.key0 = (uint32_t)seed; a.key1 = (uint32_t)(seed >> 32);
        a.sampler = ctx->opt.sampler; a.deposit = ctx->opt.deposit; a.P = ctx->opt.solar_pressure;
        a.stats = ctx->stats; a.max_tris = T; a.acc_scale = 1.0;
        e = srp_launch_sample(a, d.verts_orig, d.mats_orig, out + 3 * m0, (unsigned)m0, ctx->num_sms, ctx->stream);
        count_launches(ctx, 2 + 1);
    }
    free_designs_mem(ctx, &d);                                      // stream-ordered: after the last chunk's kernels
    if (st != SRP_OK) return st;
    if (e != cudaSuccess) return cuda_fail(ctx, "per-sample designs", e);
    return SRP_OK;
}

srp_status srp_first_hits(srp_context *ctx, const srp_designs *dz, const float *sun_dirs, int S, const int *pairs,
                          long long n_pairs, long long N, unsigned long long seed, int method, int *out_prim)
{
    srp_status st = check_trace_args(ctx, dz, sun_dirs, S, N, 0, out_prim);
    if (st != SRP_OK) return st;
    if (!pairs || n_pairs <= 0 || method < 0 || method > 1) return fail(ctx, SRP_ERR_INVALID, "bad pair list or method");
    cudaSetDevice(ctx->device);
    st = ensure_workspace(ctx, 3);
    if (st != SRP_OK) return st;
    TraceArgs a = make_args(ctx, dz, sun_dirs, S, pairs, n_pairs, N, 0, seed);
    TRY_CUDA(ctx, srp_launch_first_hits(a, method, out_prim, ctx->stream), "first-hit launch");
    return SRP_OK;
}

srp_status srp_path_signatures(srp_context *ctx, const srp_designs *dz, const float *sun_dirs, int S,
                               const int *pairs, long long n_pairs, long long N, int B,
                               unsigned long long seed, unsigned long long *out_sig)
{
    srp_status st = check_trace_args(ctx, dz, sun_dirs, S, N, B, out_sig);
    if (st != SRP_OK) return st;
    if (!pairs || n_pairs <= 0) return fail(ctx, SRP_ERR_INVALID, "bad pair list");
    cudaSetDevice(ctx->device);
    st = ensure_workspace(ctx, (size_t)n_pairs * 3);
    if (st != SRP_OK) return st;
    if (B > 0 && ctx->opt.force_brute == 0) {
        st = ensure_masks(ctx, dz, (double)n_pairs * (double)N);
        if (st != SRP_OK) return st;
    }
    ctx->launches_call = 0;
    TraceArgs a = make_args(ctx, dz, sun_dirs, S, pairs, n_pairs, N, B, seed);
    a.accum = ctx->accum;
    a.sig_out = out_sig;
    if (ctx->opt.escape_masks == 0) a.dz.esc = nullptr;
    TRY_CUDA(ctx, cudaMemsetAsync(out_sig, 0, sizeof(unsigned long long) * n_pairs * N, ctx->stream), "zero signatures");
    TRY_CUDA(ctx, cudaMemsetAsync(ctx->accum, 0, sizeof(long long) * 3 * n_pairs, ctx->stream), "zero accumulators");
    TRY_CUDA(ctx, cudaMemsetAsync(ctx->stats, 0, sizeof(DevStats), ctx->stream), "zero stats");
    TRY_CUDA(ctx, cudaMemsetAsync(ctx->work_counter, 0, SRP_PIPES * sizeof(unsigned long long), ctx->stream), "zero counter");
    const bool brute = !dz->has_bvh || ctx->opt.force_brute != 0;
    st = ensure_queue(ctx, a, brute, true);
    if (st != SRP_OK) return st;
    return launch_trace_all(ctx, a, brute, true);
}

srp_status srp_get_stats(srp_context *ctx, srp_stats *host_out)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!host_out) return fail(ctx, SRP_ERR_INVALID, "null output");
    cudaSetDevice(ctx->device);
    if (!ctx->stats) { memset(host_out, 0, sizeof *host_out); return SRP_OK; }
    TRY_CUDA(ctx, cudaStreamSynchronize(ctx->stream), "sync");
    static_assert(sizeof(DevStats) == sizeof(srp_stats), "stats layout");
    TRY_CUDA(ctx, cudaMemcpy(host_out, ctx->stats, sizeof(DevStats), cudaMemcpyDeviceToHost), "read stats");
    // the loop's kernels: beam + bounce per round that queued rays, one more beam launch that found the tiles spent
    // or queued nothing, and the loop-condition kernel of each round when the loop is a graph
    host_out->kernel_launches = ctx->launches_call + host_out->loop_rounds * (ctx->opt.plain_launches ? 2ULL : 3ULL);
    return SRP_OK;
}

srp_status srp_launch_count(srp_context *ctx, unsigned long long *n_kernels)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!n_kernels) return fail(ctx, SRP_ERR_INVALID, "null output");
    cudaSetDevice(ctx->device);
    unsigned long long rounds = 0;
    TRY_CUDA(ctx, cudaStreamSynchronize(ctx->stream), "sync");
    if (ctx->rounds_total) TRY_CUDA(ctx, cudaMemcpy(&rounds, ctx->rounds_total, sizeof rounds, cudaMemcpyDeviceToHost), "read rounds");
    *n_kernels = ctx->launches_total + rounds * (ctx->opt.plain_launches ? 2ULL : 3ULL);
    return SRP_OK;
}

unsigned long long srp_workspace_bytes_min(const srp_context *ctx)
{
    if (!ctx) return 0;
    return (unsigned long long)((queue_reserve(ctx, SRP_BEAM_TILE_MAX) + (1u << 20)) * SRP_RQ_FIELDS_INSTR * sizeof(unsigned));
}

srp_status srp_set_workspace(srp_context *ctx, void *ptr, unsigned long long bytes)
{
    if (!ctx) return SRP_ERR_INVALID;
    cudaSetDevice(ctx->device);
    if ((ptr == nullptr) != (bytes == 0)) return fail(ctx, SRP_ERR_INVALID, "workspace pointer and size must both be given, or neither");
    if (ptr && ((uintptr_t)ptr & 255u)) return fail(ctx, SRP_ERR_INVALID, "workspace must be 256-byte aligned");
    if (ptr && bytes < srp_workspace_bytes_min(ctx)) return fail(ctx, SRP_ERR_INVALID, "workspace smaller than srp_workspace_bytes_min");
    TRY_CUDA(ctx, cudaStreamSynchronize(ctx->stream), "sync before the workspace changes");
    if (ctx->rq_owned) cudaFree(ctx->rq);
    ctx->rq = (unsigned *)ptr; ctx->rq_words = (size_t)(bytes / sizeof(unsigned)); ctx->rq_owned = false;
    return SRP_OK;
}

srp_status srp_probe_peaks(srp_context *ctx, double *fp32_tflops, double *l2_read_gbs)
{
    if (!ctx) return SRP_ERR_INVALID;
    if (!fp32_tflops || !l2_read_gbs) return fail(ctx, SRP_ERR_INVALID, "null output");
    cudaSetDevice(ctx->device);
    TRY_CUDA(ctx, srp_run_probes(ctx->num_sms, ctx->stream, fp32_tflops, l2_read_gbs), "probes");
    return SRP_OK;
}

// ---- srp_forces_noalloc: the forces call for callers that must not allocate (include/srp.h) ----
// Its scratch -- the device counters every trace kernel updates and the fixed-point accumulators of the pairs --
// lives in this file-scope array instead of the context's cudaMalloc'ed workspace: every GPU that loads the
// library holds SRP_NOALLOC_SCRATCH_BYTES (1.5 MiB + 1 KiB) until the process exits.  In host code the array's
// name is only a handle; its device address comes from cudaGetSymbolAddress, once per device, with that device current.
#define SRP_NOALLOC_HEADER_BYTES 1024
#define SRP_NOALLOC_SCRATCH_BYTES (SRP_NOALLOC_HEADER_BYTES + (size_t)SRP_NOALLOC_MAX_PAIRS * 3 * sizeof(long long))
static __device__ __align__(256) unsigned char srp_noalloc_scratch[SRP_NOALLOC_SCRATCH_BYTES];
static_assert(sizeof(DevStats) <= 512 && (SRP_PIPES + 1) * sizeof(unsigned long long) <= 256, "header layout");

static cudaError_t noalloc_scratch_address(int device, unsigned char **out)
{
    static unsigned char *addr[64];                    // per device; written once, the same value from any thread
    if (device < 0 || device >= 64) return cudaErrorInvalidDevice;
    if (!addr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, srp_noalloc_scratch);     // the caller made `device` current
        if (e != cudaSuccess) return e;
        addr[device] = (unsigned char *)p;
    }
    *out = addr[device];
    return cudaSuccess;
}

srp_status srp_forces_noalloc(srp_context *ctx, const srp_designs *dz, const float *sun_dirs, int S, long long N, int B,
                              unsigned long long seed, float *out)
{
    srp_status st = check_trace_args(ctx, dz, sun_dirs, S, N, B, out);
    if (st != SRP_OK) return st;
    const long long n_pairs = (long long)dz->D * S;
    if (n_pairs > SRP_NOALLOC_MAX_PAIRS)
        return fail(ctx, SRP_ERR_INVALID, "srp_forces_noalloc: designs x directions exceeds SRP_NOALLOC_MAX_PAIRS (65536)");
    if (ctx->opt.instrumented) return fail(ctx, SRP_ERR_UNSUPPORTED, "srp_forces_noalloc: not with the instrumented kernels");
    const bool brute = !dz->has_bvh || ctx->opt.force_brute != 0;
    if (want_beams(ctx, brute, dz->maxT, N, n_pairs))
        return fail(ctx, SRP_ERR_UNSUPPORTED, "srp_forces_noalloc: this call would trace beams through a ray queue "
                                             "(designs with a BVH and rays_per_dir >= 8 x triangles); use srp_forces");
    cudaSetDevice(ctx->device);
    unsigned char *scratch = nullptr;
    TRY_CUDA(ctx, noalloc_scratch_address(ctx->device, &scratch), "address of the static scratch");
    ctx->launches_call = 0;
    TraceArgs a = make_args(ctx, dz, sun_dirs, S, nullptr, n_pairs, N, B, seed);
    a.stats = (DevStats *)scratch;                                             // [0, 512): counters
    a.work_counter = (unsigned long long *)(scratch + 512);                    // [512, 768): tile counters, loop rounds
    a.rounds_total = a.work_counter + SRP_PIPES;
    a.accum = (long long *)(scratch + SRP_NOALLOC_HEADER_BYTES);               // [1024, ...): 3 int64 per pair
    a.acc_stride = 3; a.torque = 0; a.xcom = nullptr;
    a.rq = nullptr; a.rq_cap = 0; a.rq_high = 0; a.rq_ctr = nullptr;
    // escape masks an earlier call built with these designs are used; none is built here (results do not depend on them)
    if (ctx->opt.escape_masks == 0 || ctx->opt.force_brute != 0) a.dz.esc = nullptr;
    // the array keeps the last call's contents: everything this call reads before writing starts at zero
    TRY_CUDA(ctx, cudaMemsetAsync(scratch, 0, SRP_NOALLOC_HEADER_BYTES + sizeof(long long) * 3 * (size_t)n_pairs, ctx->stream),
             "zero the static scratch");
    TRY_CUDA(ctx, srp_launch_trace(a, brute, false, ctx->num_sms, ctx->stream), "trace launch");
    TRY_CUDA(ctx, srp_launch_finalize(a, out, nullptr, ctx->stream), "finalize launch");
    count_launches(ctx, 2);
    return SRP_OK;
}

} // extern "C"
