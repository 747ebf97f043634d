// srp_internal.cuh -- shared declarations of libsrp_b200's translation units (CUDA path only;
// nothing under oracle/ includes this file).  See include/srp.h for the public C ABI and
// DESIGN.md for the data layout.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>
#include "srp.h"

#define SRP_PIPES 2                // beam / bounce loops that run side by side, each on its share of the tiles
#define SRP_BRUTE_MAX_TRIS 64      // designs with T <= this are traced without a hierarchy (one leaf)
#define SRP_LEAF_MAX 2             // subtrees with <= this many triangles become one leaf (cfg3 -7 %, cfg5 -3 % against 3)
#define SRP_ACC_BITS_MAX 32        // fixed-point fraction bits of the dimensionless force accumulators, at most

// Packed, BVH-sorted triangle: 3 x float4 = 48 B, fetched as three 16-byte loads.
//   q0 = (v0.x, v0.y, v0.z, alpha)   q1 = (e1.x, e1.y, e1.z, rho_s)   q2 = (e2.x, e2.y, e2.z, rho_d)
// BVH2 node: 4 x float4 = 64 B.
//   q0 = (lo0.x, lo0.y, lo0.z, hi0.x)  q1 = (hi0.y, hi0.z, lo1.x, lo1.y)
//   q2 = (lo1.z, hi1.x, hi1.y, hi1.z)  q3 = (link0, link1, -, -) as int bits
// link >= 0: node index (relative to the design's node base); link < 0: leaf, u = ~link,
// first = u >> 3 (sorted triangle index relative to the design's triangle base), count = (u & 7) + 1.
struct DesignsDev {
    const float4 *tri;        // [sumT * 3]
    const float4 *nodes;      // [sumT * 4]; node base of design k == tri_off[k]
    const float4 *nodes4;     // [sumT * 8]: 4-wide nodes folded from the BVH2 (bvh4.cu), same numbering; or nullptr
    const long long *tri_off; // [D + 1]
    const float4 *box;        // [D * 2]: (lo, -), (hi, -)
    const int *perm;          // [sumT]: sorted position -> original index within the design
    const unsigned *esc;      // [sumT * 14]: escape masks (escape_mask.cu), or nullptr
    const float *shin;        // [sumT] sorted order: Phong exponent of the specular lobe (R23), or nullptr = ideal mirrors
    const float4 *nplane;     // [sumT * 2]: per-node plane slab (n, dmin), (dmax) -- lbvh.cu; with esc
    int D;
    int has_bvh;
};

struct srp_designs {
    int D = 0;
    int family = -1;
    long long sumT = 0, maxT = 0;
    std::vector<long long> tri_off;     // host copy [D+1]
    float *verts_orig = nullptr;        // [sumT*9] original order (device)
    float *mats_orig = nullptr;         // [sumT*3]
    float4 *tri = nullptr;
    float4 *nodes = nullptr;
    float4 *nodes4 = nullptr;
    long long *tri_off_dev = nullptr;
    float4 *box = nullptr;
    int *perm = nullptr;
    unsigned *esc = nullptr;
    float4 *nplane = nullptr;
    float *shin = nullptr;
    bool esc_failed = false;  // the mask allocation failed once: do not try again
    bool has_bvh = false;
    DesignsDev dev() const {
        DesignsDev d;
        d.tri = tri; d.nodes = nodes; d.nodes4 = nodes4; d.tri_off = tri_off_dev; d.box = box; d.perm = perm; d.esc = esc; d.nplane = nplane; d.shin = shin; d.D = D;
        d.has_bvh = has_bvh ? 1 : 0;
        return d;
    }
};

struct DevStats {           // device mirror of srp_stats
    unsigned long long launched, primary_miss, absorbed, escaped, capped, segments;
    unsigned long long hits_at_depth[16];
    unsigned long long box_tests, tri_tests;
    unsigned long long beam_tile_miss, beam_block_miss, beam_group_miss, beam_fallback;
    unsigned long long beam_box_tests, tri2d_tests, tri_setups, rect_tests;
    unsigned long long mask_escapes;
    unsigned long long queued_rays, loop_rounds, kernel_launches;
};

struct srp_context {
    int device = 0;
    cudaStream_t stream = nullptr;
    srp_options opt;
    std::string last_error;
    int num_sms = 148;
    // workspace (grown on demand, never shrunk)
    long long *accum = nullptr;   size_t accum_items = 0;     // int64 fixed-point [pairs*3]
    DevStats *stats = nullptr;
    unsigned long long *work_counter = nullptr;
    unsigned *rq = nullptr;       size_t rq_words = 0;        // ray queue between the beam and the bounce kernel
    unsigned *rq_ctr = nullptr;                               // its counters: [0] tail, [1] head, [2] warps done
    bool rq_owned = false;                                    // allocated by the library (else srp_set_workspace)
    unsigned long long launches_total = 0;                    // kernels enqueued by the host since srp_create
    unsigned long long launches_call = 0;                     // ... by the last srp_forces* call
    unsigned long long *rounds_total = nullptr;               // device: loop rounds since srp_create
    cudaMemPool_t mempool = nullptr;                          // design arrays come from this private stream-ordered pool
    cudaStream_t capture_stream[SRP_PIPES] = { nullptr, nullptr };   // the beam / bounce loops are captured here into a graph
    struct PendingGraph { cudaGraphExec_t exec; cudaGraph_t graph; cudaEvent_t done; };
    std::vector<PendingGraph> graphs;                         // launched loops; destroyed once they have run
    float *stage_dirs = nullptr;  size_t stage_dirs_items = 0; // srp_forces_host staging
    float *stage_out = nullptr;   size_t stage_out_items = 0;
};

struct TraceArgs {
    DesignsDev dz;
    const float *sun_dirs;   // [S,3]
    const int *pairs;        // [n_pairs,2] or nullptr (then pair p = (p / S, p % S))
    long long n_pairs;
    int S;
    long long N;             // rays per direction
    int log2N;               // valid when sampler == 0
    int B;
    uint32_t key0, key1;
    int sampler, deposit;
    double P;
    long long *accum;        // [n_pairs*acc_stride]: force (and torque) sums in 2^-32 fixed point
    int acc_stride;          // 3, or 6 with a second output
    int torque;              // second output: 0 none, 1 torque about xcom (arm in units of the design's extent, see
                             // torque_arm_scale), 2 direct part of the force (deposits at depth 0)
    double acc_scale;        // 2^bits: the accumulators hold sums of deposits / w_ph in this fixed point (srp_api.cu,
                             // acc_scale_for: chosen per call so that N photons of B + 1 hits cannot overflow int64)
    const float *xcom;       // [D,3] centres of mass, or nullptr (origin)
    DevStats *stats;
    unsigned long long *work_counter;
    long long tiles_per_pair;
    unsigned long long tile_begin, tile_end;   // beam kernel: this launch works on tiles [tile_begin, tile_end) (a pipeline's share)
    int tile_rays;
    unsigned long long *sig_out;   // debug (instrumented kernels): [n_pairs, N] path signatures, or nullptr
    // ray queue (trace_beam.cu -> trace_bounce.cu): continuing photons the beam kernel hands to the bounce kernel
    unsigned *rq;                  // field-major: field f of ray r at rq[f * rq_cap + r]; nullptr = no beams
    unsigned rq_cap;               // rays the queue holds
    unsigned rq_high;              // beam warps stop taking tiles once this many rays are queued
    unsigned *rq_ctr;              // [0] tail (rays queued), [1] head (rays claimed), [2] bounce warps done
    unsigned long long *rounds_total;   // loop rounds since srp_create (srp_launch_count)
    long long max_tris;            // largest design of the batch
    int primary_mode;              // srp_options.primary_mode
};

// ---- launchers implemented in the .cu files (all enqueue on `stream`, return cudaError_t) ----
cudaError_t srp_launch_mesh_gen(int family, const float *theta, int D, int n_params,
                                unsigned long long mesh_seed, long long T, float *verts, float *mats,
                                cudaMemPool_t pool, unsigned k_offset, cudaStream_t stream);
// builder: srp_options.bvh_builder; *launches = kernels enqueued
cudaError_t srp_launch_build(srp_designs *dz, int leaf_max, int builder, cudaMemPool_t pool, cudaStream_t stream, int *launches);
cudaError_t srp_launch_sah_build(srp_designs *dz, const unsigned *vals, unsigned *vals_final, int leaf_max,
                                 cudaMemPool_t pool, cudaStream_t stream, int *launches);
cudaError_t srp_launch_collapse4(const srp_designs *dz, cudaStream_t stream);   // nodes -> nodes4
cudaError_t srp_launch_gather_shininess(const DesignsDev &dz, long long sumT, const float *shin_orig, float *shin_sorted, cudaStream_t stream);
cudaError_t srp_launch_node_planes(const DesignsDev &dz, long long sumT, float4 *nplane, cudaStream_t stream);
cudaError_t srp_launch_escape_masks_small(const DesignsDev &dz, long long sumT, unsigned *esc, cudaStream_t stream);
cudaError_t srp_launch_escape_masks(const DesignsDev &dz, long long maxT, unsigned *esc, cudaStream_t stream);
cudaError_t srp_launch_trace(const TraceArgs &a, bool brute, bool instrumented, int num_sms,
                             cudaStream_t stream);
cudaError_t srp_launch_bounce(const TraceArgs &a, bool instrumented, int num_sms, cudaStream_t stream);
cudaError_t srp_launch_loop_cond(cudaGraphConditionalHandle handle, const TraceArgs &a, cudaStream_t stream);
cudaError_t srp_launch_finalize(const TraceArgs &a, float *out_forces, float *out_torques, cudaStream_t stream);
cudaError_t srp_launch_first_hits(const TraceArgs &a, int method, int *out_prim, cudaStream_t stream);
cudaError_t srp_launch_thermal(const TraceArgs &a, const float *facet_power, long long sumT, int *emit_list, int *n_emit,
                               float *design_power, float *out_forces, int num_sms, cudaStream_t stream);
long long srp_sample_max_tris();
cudaError_t srp_launch_sample(const TraceArgs &a, const float *verts, const float *mats, float *out, unsigned k_offset, int num_sms,
                              cudaStream_t stream);
cudaError_t srp_run_probes(int num_sms, cudaStream_t stream, double *fp32_tflops, double *l2_gbs);

long long srp_family_tris_host(int family);
int srp_trace_blocks_per_sm(bool brute, bool beam);
int srp_beam_warps(int num_sms);                       // resident warps of the beam kernel (queue sizing)
#define SRP_RQ_FIELDS 9                                // origin, direction, ray index, pair index, src | depth << 27
#define SRP_RQ_FIELDS_INSTR 11                         // + 64-bit path signature
