/*
 * srp.h -- C ABI of libsrp_b200: batched Monte-Carlo solar-radiation-pressure (SRP) forces
 * on one NVIDIA B200 (sm_100a).
 *
 * The library computes, for every (design k, sun direction j) pair, the force
 *     F(omega_j, theta_k) = int_{M(theta_k)} f(x, omega_j, theta_k) dx      PAPER.md:131 (Eq. 3)
 * with f given by the light-to-force map of PAPER.md:125 (Eq. 2), by forward Monte-Carlo photon
 * tracing with multiple bounces (Sec. 3.2 "Estimation"), the reading of the paper
 * written out in DESIGN.md ("O-steps", R1-R17).  "takes design parameters and the light direction,
 * returns 3-D force": srp_build_designs is the "design parameters -> triangle mesh
 * with per-face material" map of PAPER.md:148 plus a per-design bounding-volume hierarchy (a binned-SAH
 * BVH2 by default; srp_options.bvh_builder = 1 gives the Karras-style linear BVH, the structure the
 * paper builds for its Fig. 8); srp_forces is the estimator.
 *
 * Conventions
 *  - Every function returns srp_status; outputs are untouched unless SRP_OK.  No exceptions cross
 *    the boundary.  srp_last_error(ctx) gives the text of the last failure of that context.
 *  - Pointers marked DEVICE are CUDA device pointers on the context's device (e.g. a torch tensor's
 *    data_ptr()); pointers marked HOST are ordinary host memory.  The caller owns every buffer it
 *    passes; the library owns the opaque handles, small counters and accumulators, and -- unless the caller provides
 *    it with srp_set_workspace -- the ray queue of the beam / bounce loop (cudaMalloc'ed on first use; a failed
 *    allocation is SRP_ERR_OOM, never a silent change of method).  Design arrays come from a stream-ordered memory
 *    pool of the context's own.
 *  - srp_build_designs* and srp_forces only ENQUEUE work on the context's stream; the caller
 *    synchronises that stream.  Functions documented "syncs" wait for the stream.
 *  - Same inputs + same seed => bit-identical output (integer fixed-point accumulation).
 *  - One context per host thread.  No CPU fallback exists: without a CUDA device every call fails.
 */
#ifndef SRP_B200_H
#define SRP_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct srp_context srp_context;   /* opaque: device, stream, options, workspace, last error */
typedef struct srp_designs srp_designs;   /* opaque: device meshes + BVHs of D designs              */

typedef enum {
    SRP_OK = 0,
    SRP_ERR_INVALID = -1,       /* bad argument, detected on the host before any launch */
    SRP_ERR_CUDA = -2,          /* a CUDA runtime call failed; text in srp_last_error    */
    SRP_ERR_OOM = -3,           /* device allocation failed                              */
    SRP_ERR_UNSUPPORTED = -4
} srp_status;

/* Mesh families (BASELINE.json configs 1-5).  theta layout per family:
 *   PLATE    n_params 3: (alpha, rho_s, rho_d) of the 1 m x 1 m plate            T = 2
 *   BOXWING  n_params 2: (panel length L [m], panel angle phi [rad])             T = 16
 *   DETAILED n_params 2: (dish tilt theta_dish, panel angle phi_pan) [rad]       T = 49840
 *   BOXWING6 n_params 6: (phi1, phi2, L, bus aspect a, rho_s panel, rho_d bus)   T = 16
 *   SAIL     n_params 1: (height-field amplitude [m], 0.05 in config 5)          T = 1019698
 *   BOXWING_T n_params 2: the BOXWING geometry tessellated (bus 8 x 8 cells per face,
 *            panels 8 x 16): "a representative satellite model (1 k faces)", PAPER.md:352   T = 1280 */
typedef enum {
    SRP_FAMILY_PLATE = 0,
    SRP_FAMILY_BOXWING = 1,
    SRP_FAMILY_DETAILED = 2,
    SRP_FAMILY_BOXWING6 = 3,
    SRP_FAMILY_SAIL = 4,
    SRP_FAMILY_BOXWING_T = 5
} srp_family;

typedef struct {
    double solar_pressure;  /* P = L/c of Eq. 2 [N/m^2]; default 4.56e-6 (1 AU)                    */
    int sampler;            /* 0 = stratified jittered grid in Morton order (default),
                               1 = i.i.d. uniform over the emitter rectangle                        */
    int deposit;            /* 0 = expected-value deposit (default), 1 = analog (sampled path only) */
    int force_brute;        /* 1 = ignore the BVH and test every triangle; test use   */
    int instrumented;       /* 1 = also count ray-box and ray-triangle tests (slower kernels)        */
    int primary_mode;       /* how the primaries of designs with a BVH are traced (stratified sampler):
                               0 = auto: as beams (blocks of rays share one BVH descent) when
                                   rays_per_dir >= 8 x the largest design's triangle count, else one by one,
                               1 = every primary walks the BVH on its own, 2 = beams always; test use   */
    int escape_masks;       /* per-triangle masks of the directions in which a ray leaving the triangle could hit
                               anything (designs with a BVH); bounce rays outside them are counted as escaped
                               without a traversal (results unchanged).  Built inside the first srp_forces* /
                               srp_thermal_forces call that wants them and kept with the designs handle (which
                               is therefore not to be used from two contexts at once).
                               0 = never, 1 (default) = when the call traces >= 32768 photons per triangle of
                               the batch (the build is repaid), 2 = always; test use                          */
    int plain_launches;     /* designs with a BVH traced as beams run a loop of two kernels (beam kernel, bounce kernel)
                               whose trip count is known only on the device.  0 (default) = the loop is a
                               conditional WHILE node of a CUDA graph; 1 = the same kernels as plain launches, a fixed
                               sufficient number of rounds (surplus rounds find nothing to do) -- for profilers that do
                               not list kernels inside conditional graph nodes.  Results are identical.            */
    int leaf_max;           /* subtrees with at most this many triangles become one leaf, 1..8; 0 = default (2).
                               Read by srp_build_designs*; test and tuning use                                       */
    int bvh_builder;        /* the hierarchy of designs with more than 64 triangles: 0 (default) = top-down binned
                               surface-area heuristic over the Morton order (bvh_sah.cu), 1 = linear BVH (Karras
                               hierarchy of the Morton codes, lbvh.cu; the structure of PAPER.md:366).  Same node
                               layout, same results up to the order of summation.  Read by srp_build_designs*      */
} srp_options;

/* Photon bookkeeping of the last srp_forces call (DESIGN.md "Pins" P8).
 * launched = primary_miss + absorbed + escaped + capped; segments = every ray cast.
 * box_tests / tri_tests are filled only when srp_options.instrumented = 1. */
typedef struct {
    unsigned long long launched, primary_miss, absorbed, escaped, capped, segments;
    unsigned long long hits_at_depth[16];
    unsigned long long box_tests, tri_tests;
    /* beam tracing of primaries: rays resolved as misses by a whole tile / sub-block / group of 32,
       and primaries that fell back to per-ray traversal because a beam list overflowed */
    unsigned long long beam_tile_miss, beam_block_miss, beam_group_miss, beam_fallback;
    /* instrumented only: work of the beam path -- beam-vs-box tests of the cooperative descents, 2-D
       (emitter-frame) ray-triangle tests, triangle set-ups (edge functions + depth plane), and
       rectangle-vs-triangle culling tests.  box_tests / tri_tests count per-ray slab tests and
       Moller-Trumbore tests only. */
    unsigned long long beam_box_tests, tri2d_tests, tri_setups, rect_tests;
    unsigned long long mask_escapes;   /* bounce rays resolved as "escaped" by the escape masks (also counted in
                                          escaped and segments) */
    unsigned long long queued_rays;    /* slots of the ray queue the beam kernel handed to the bounce kernel (rays, plus
                                          the few slots a beam warp reserved and did not fill) */
    unsigned long long loop_rounds;    /* rounds of the beam / bounce loop that had rays queued (counted on the device) */
    unsigned long long kernel_launches;/* kernels of this library the last srp_forces* / srp_thermal_forces call ran:
                                          those enqueued by the host plus, for the beam / bounce loop, the rounds the
                                          device counted (CUB's sort kernels of a build are not included) */
} srp_stats;

/* Creates a context on CUDA device `cuda_device`; `cuda_stream` is a cudaStream_t (may be NULL =
 * the legacy default stream) that all work of this context is enqueued on. */
srp_status srp_create(srp_context **ctx, int cuda_device, void *cuda_stream);
srp_status srp_destroy(srp_context *ctx);                       /* syncs; frees the workspace */
srp_status srp_set_options(srp_context *ctx, const srp_options *opt);
srp_status srp_get_options(const srp_context *ctx, srp_options *opt);
const char *srp_last_error(const srp_context *ctx);

/* Number of parameters / triangles of a family (host-side constants; -1 for an unknown family). */
int srp_family_n_params(srp_family family);
long long srp_family_tri_count(srp_family family);

/* S0 + S1: theta DEVICE float[D, n_params] row-major -> meshes (fp64 evaluation rounded once to fp32)
 * and per-design BVHs.  mesh_seed keys the per-facet Dirichlet(2,2,2) material draws and the sail's
 * noise.  n_params must equal srp_family_n_params(family).  Enqueues only. */
srp_status srp_build_designs(srp_context *ctx, srp_family family, const float *theta, int D,
                             int n_params, unsigned long long mesh_seed, srp_designs **out);

/* User-supplied meshes (the paper's general design->mesh map):
 * verts DEVICE float[sumT,3,3] (v0,v1,v2), mats DEVICE float[sumT,3] = (alpha, rho_s, rho_d), each >= 0 and
 * summing to 1 (they are used as given: the lobe draw reads alpha and alpha + rho_s as thresholds and takes the rest
 * as diffuse, the expected-value deposit uses all three; the Python binding checks host arrays),
 * tri_offsets HOST long long[D+1], tri_offsets[0] = 0, strictly increasing.  Enqueues only. */
srp_status srp_build_designs_from_meshes(srp_context *ctx, const float *verts, const float *mats,
                                         const long long *tri_offsets, int D, srp_designs **out);

/* D and the triangle offsets (HOST long long[D+1], may be NULL). */
srp_status srp_designs_info(const srp_designs *designs, int *D, long long *tri_offsets_host);

/* Reads back design `design`'s mesh in ORIGINAL triangle order: verts_host HOST float[T,3,3],
 * mats_host HOST float[T,3].  Either may be NULL.  Syncs; test use. */
srp_status srp_designs_read_mesh(srp_context *ctx, const srp_designs *designs, int design,
                                 float *verts_host, float *mats_host);

/* Reads back design `design`'s BVH for structural tests.  Syncs.
 *   n_nodes out: number of node records (0 if the design has no hierarchy -- brute-force leaf).
 *   nodes_host HOST float[n_nodes,16] (may be NULL): per node
 *     [0..5] child-0 box (lo xyz, hi xyz), [6..11] child-1 box, [12],[13] child links as int bits,
 *     [14],[15] unused.  A link >= 0 is a node index; a link < 0 encodes a leaf: u = ~link,
 *     first = u >> 3 (sorted triangle index within the design), count = (u & 7) + 1.
 *   perm_host HOST int[T] (may be NULL): sorted position -> original triangle index. */
srp_status srp_designs_read_bvh(srp_context *ctx, const srp_designs *designs, int design,
                                long long *n_nodes, float *nodes_host, int *perm_host);

srp_status srp_free_designs(srp_context *ctx, srp_designs *designs);   /* syncs */

/* S2-S7: sun_dirs DEVICE float[S,3], body->sun (the paper's omega), any non-zero
 * length (a zero or non-finite direction gives F = 0 for its pairs); rays_per_dir N > 0 (a power of two when sampler = 0); 0 <= max_bounces <= 15 reflections
 * followed (R5); seed keys Philox4x32-10 with counter (ray, direction, design, depth).
 * out_forces DEVICE float[D,S,3], newtons, body frame.  Enqueues only. */
srp_status srp_forces(srp_context *ctx, const srp_designs *designs, const float *sun_dirs, int S,
                      long long rays_per_dir, int max_bounces, unsigned long long seed,
                      float *out_forces);

/* Same, restricted to an explicit list of pairs: pairs DEVICE int[n_pairs,2] = (design k,
 * direction j), 0 <= k < D, 0 <= j < S (entries out of range are clamped into it on the device: memory-safe,
 * meaningless); out_forces DEVICE float[n_pairs,3].  The Philox counters use (k, j), so the result
 * of a pair equals the corresponding entry of the full srp_forces call bit for bit. */
srp_status srp_forces_pairs(srp_context *ctx, const srp_designs *designs, const float *sun_dirs, int S,
                            const int *pairs, long long n_pairs, long long rays_per_dir,
                            int max_bounces, unsigned long long seed, float *out_forces);

/* Forces AND torques (Eq. 4: tau = int (x - x_COM) x f(x) dx; the paper's simulator
 * returns both).  x_com DEVICE float[D,3]: centre of mass of each design in the body frame, or
 * NULL for the origin.  out_torques DEVICE float[D,S,3] (or [n_pairs,3]) in N m.  Every momentum deposit of
 * srp_forces, made at hit point x, also adds (x - x_COM) x deposit; out_forces is what srp_forces returns
 * (same photons; sums may differ in the last bits).  Enqueues only. */
srp_status srp_forces_torques(srp_context *ctx, const srp_designs *designs, const float *sun_dirs, int S,
                              long long rays_per_dir, int max_bounces, unsigned long long seed,
                              const float *x_com, float *out_forces, float *out_torques);
srp_status srp_forces_torques_pairs(srp_context *ctx, const srp_designs *designs, const float *sun_dirs, int S,
                                    const int *pairs, long long n_pairs, long long rays_per_dir, int max_bounces,
                                    unsigned long long seed, const float *x_com, float *out_forces,
                                    float *out_torques);

/* Forces and their DIRECT part (Fig. 5 rows 3-4: direct and indirect force maps; the
 * no-bounce variant): out_direct DEVICE float[D,S,3] (or [n_pairs,3]) = the momentum deposited where sun light first
 * meets the surface -- what srp_forces returns with max_bounces = 0 (same photons; bit for bit from the beam kernels,
 * to the rounding of per-lane fp32 partial sums otherwise) -- from the same trace that gives out_forces; the indirect part (everything deposited by light reflected at least once) is out_forces - out_direct.
 * Enqueues only. */
srp_status srp_forces_split(srp_context *ctx, const srp_designs *designs, const float *sun_dirs, int S,
                            long long rays_per_dir, int max_bounces, unsigned long long seed, float *out_forces,
                            float *out_direct);
srp_status srp_forces_split_pairs(srp_context *ctx, const srp_designs *designs, const float *sun_dirs, int S,
                                  const int *pairs, long long n_pairs, long long rays_per_dir, int max_bounces,
                                  unsigned long long seed, float *out_forces, float *out_direct);

/* Glossy specular lobes, PAPER.md:148 (meshes carry "per-face Phong material parameters"); R23.
 * shininess DEVICE float[sumT], ORIGINAL triangle order of all designs back to back (tri_offsets of
 * srp_designs_info): the Phong exponent n of each facet's specular part.  n >= 0: a photon that draws the specular
 * lobe leaves in a direction distributed as cos^n about the mirror direction (importance-sampled; directions below
 * the facet's horizon are redrawn, at most 8 times); n < 0: the ideal mirror, which is also what every facet is
 * while no shininess is set.  NULL removes the array.  The values are copied (reordered) on the context's stream;
 * they apply to every later srp_forces* / srp_thermal_forces / srp_path_signatures call on this handle.  With the
 * expected-value deposit a glossy facet's specular momentum is deposited per drawn direction (its mean has no
 * closed form under the horizon cut), the absorbed and diffuse parts in expectation as before.
 * SRP_ERR_INVALID on a null handle.  Enqueues only. */
srp_status srp_designs_set_shininess(srp_context *ctx, srp_designs *designs, const float *shininess);

/* Thermal (local Lambertian) emitters, PAPER.md:606-612 (Sec. 5.9: "local sources [are handled] in the same way
 * ... thermal emission as Lambertian", recoil 2/3 of a collimated beam); R22.
 * facet_power DEVICE float[sumT] in watts, ORIGINAL triangle order of all designs back to back (tri_offsets of
 * srp_designs_info); sign = emitting side (+: the side of normalize((v1-v0) x (v2-v0)), -: the other side); zero =
 * no emission.  Every emitting facet launches rays_per_facet photons (uniform origin on the triangle,
 * cosine-weighted direction, Philox counter (ray, facet, design, 0x80000000 | depth)) which are followed for up to
 * max_bounces reflections like sun photons.  out_forces DEVICE float[D,3]: net recoil force per design in newtons
 * (emission recoil plus what the emitted photons deposit on the design itself).  srp_options.deposit applies;
 * srp_get_stats counts the emitted photons.  Enqueues only. */
srp_status srp_thermal_forces(srp_context *ctx, const srp_designs *designs, const float *facet_power,
                              long long rays_per_facet, int max_bounces, unsigned long long seed,
                              float *out_forces);

/* Host-buffer convenience (the end-to-end call): theta-independent; sun_dirs_host HOST float[S,3],
 * out_forces_host HOST float[D,S,3].  Copies in, runs srp_forces, copies out, syncs. */
srp_status srp_forces_host(srp_context *ctx, const srp_designs *designs, const float *sun_dirs_host,
                           int S, long long rays_per_dir, int max_bounces, unsigned long long seed,
                           float *out_forces_host);

/* The paper's own workload shape: a batch of M records, each with
 * its OWN design theta_m and its OWN light direction omega_m -- "every ray effectively intersects a different world"
 * -- and only rays_per_record photons, so no hierarchy is built: the closest hit is that of the paper's test of every
 * ray against all triangles of its record's mesh (found with fewer tests: primaries rasterised into the emitter grid,
 * bounce rays through boxes around clusters of 32 triangles).  theta DEVICE float[M, n_params], sun_dirs DEVICE float[M,3] (body->sun),
 * out_forces DEVICE float[M,3] newtons.  Record m is design m with direction m: its mesh, materials and photons are
 * those of srp_build_designs + srp_forces_pairs with the pair (m, m), except that the direction index in the Philox
 * counter is 0 (counter (ray, 0, m, depth)); M is not limited to 65535.  The family's meshes must have at most 3970
 * triangles (one record's triangles live in a thread block's shared memory); srp_options.sampler and .deposit
 * apply; torque, glossy lobes and escape masks do not.  The meshes are generated chunk by chunk on the way and not
 * kept.  srp_get_stats covers the whole batch.  Enqueues only. */
srp_status srp_forces_per_sample(srp_context *ctx, srp_family family, const float *theta, int n_params,
                                 const float *sun_dirs, long long M, long long rays_per_record, int max_bounces,
                                 unsigned long long seed, unsigned long long mesh_seed, float *out_forces);

/* Debug: primary-hit triangle (ORIGINAL index, -1 = miss) of every ray of the listed pairs:
 * out_prim DEVICE int[n_pairs, rays_per_dir].  method 0 = BVH traversal, 1 = brute force. */
srp_status srp_first_hits(srp_context *ctx, const srp_designs *designs, const float *sun_dirs, int S,
                          const int *pairs, long long n_pairs, long long rays_per_dir,
                          unsigned long long seed, int method, int *out_prim);

/* Debug: path signature of every photon of the listed pairs: out_sig DEVICE unsigned long long
 * [n_pairs, rays_per_dir]; sig = 0, then sig = sig * 1000003 + (ORIGINAL triangle index + 1) at every
 * hit (mod 2^64).  Two tracers took the same path through the mesh iff the signatures agree, so the
 * harness counts divergent rays with it.  Runs the instrumented kernel.  Enqueues only. */
srp_status srp_path_signatures(srp_context *ctx, const srp_designs *designs, const float *sun_dirs, int S,
                               const int *pairs, long long n_pairs, long long rays_per_dir,
                               int max_bounces, unsigned long long seed, unsigned long long *out_sig);

/* srp_forces for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): same arguments, same results (S2-S7), but this call allocates nothing and
 * frees nothing -- no cudaMalloc / cudaFree, no stream-ordered pool, no escape-mask build (masks that an earlier
 * call built with these designs are used).  Its scratch (device counters and the int64 accumulators, 24 bytes per
 * (design, direction) pair) is a static device array of SRP_NOALLOC_MAX_PAIRS pairs = 1.5 MiB that every GPU which
 * loads the library holds until the process exits.  Limits: designs x directions <= SRP_NOALLOC_MAX_PAIRS, else
 * SRP_ERR_INVALID; calls that srp_forces would trace as beams through a ray queue (designs with more than 64
 * triangles and rays_per_dir >= 8 x the largest triangle count, unless srp_options.primary_mode = 1) and the
 * instrumented kernels give SRP_ERR_UNSUPPORTED.  All contexts and streams of a process on one GPU share the array:
 * calls that overlap on the GPU race (enqueue them on one stream, or order them with events); the array keeps the
 * last call's contents and every call clears what it uses.  srp_get_stats does not cover this call.  sun_dirs and
 * out_forces are DEVICE pointers as in srp_forces.  Enqueues only. */
#define SRP_NOALLOC_MAX_PAIRS 65536
srp_status srp_forces_noalloc(srp_context *ctx, const srp_designs *designs, const float *sun_dirs, int S,
                              long long rays_per_dir, int max_bounces, unsigned long long seed, float *out_forces);

/* Counters of the last srp_forces* call on this context.  Syncs. */
srp_status srp_get_stats(srp_context *ctx, srp_stats *host_out);

/* Kernels of this library that this context has run since srp_create (builds, mask builds, trace kernels, loop
 * rounds as counted on the device, finalisation; not CUB's sort kernels, not the probes).  Syncs. */
srp_status srp_launch_count(srp_context *ctx, unsigned long long *n_kernels);

/* Workspace from the caller (PyTorch stays the only allocator): `bytes` of DEVICE memory at `ptr` (256-byte aligned)
 * that the library uses for the ray queue between the beam kernel and the bounce kernel instead of allocating one
 * itself (36 bytes per queued ray, 44 in the instrumented build).  The memory must stay valid until the next srp_set_workspace or srp_destroy;
 * (NULL, 0) hands the choice back to the library.  A workspace smaller than srp_workspace_bytes_min(ctx) is refused
 * with SRP_ERR_INVALID; a larger one means fewer rounds of the beam / bounce loop.  Syncs. */
srp_status srp_set_workspace(srp_context *ctx, void *ptr, unsigned long long bytes);
unsigned long long srp_workspace_bytes_min(const srp_context *ctx);

/* Micro-benchmarks for the roofline denominators: register-resident FP32
 * FMA chains, and an L2-resident 16-byte-load sweep.  Syncs; results in TFLOP/s and GB/s. */
srp_status srp_probe_peaks(srp_context *ctx, double *fp32_tflops, double *l2_read_gbs);

#ifdef __cplusplus
}
#endif
#endif /* SRP_B200_H */
