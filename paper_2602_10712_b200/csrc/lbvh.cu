// lbvh.cu -- S1 of the hot path: per-design linear BVH (Morton order + Karras-style hierarchy,
// the structure the paper builds for Fig. 8; PAPER.md:64,148 discuss why the paper
// itself does not trace with one).  All designs of a batch are built together:
//   design AABB -> 48-bit Morton code of each centroid, keyed (design << 48 | code) -> one radix
//   sort (CUB) -> hierarchy (one thread per internal node) -> bottom-up refit (atomic arrival
//   flags) -> emit 64-byte BVH2 nodes holding both child boxes, small subtrees collapsed to leaves
//   -> pack triangles in sorted order as 3 x float4 with the material in the w lanes.
// Designs with T <= SRP_BRUTE_MAX_TRIS in a batch whose largest design is that small get no
// hierarchy: the tracer tests all their triangles (the paper's own method).
#include <cub/device/device_radix_sort.cuh>
#include <cfloat>
#include "srp_internal.cuh"

namespace {

typedef unsigned long long u64;

__device__ inline int find_design(const long long *off, int D, long long g)
{
    int lo = 0, hi = D;            // off[lo] <= g < off[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (off[mid] <= g) lo = mid; else hi = mid;
    }
    return lo;
}

// ---- design AABB: one block per design ----
__global__ void __launch_bounds__(256)
design_box_kernel(const float *verts, const long long *off, float4 *box)
{
    const int k = blockIdx.x;
    const long long v_begin = off[k] * 3, v_end = off[k + 1] * 3;   // vertex index range
    float lo[3] = { FLT_MAX, FLT_MAX, FLT_MAX }, hi[3] = { -FLT_MAX, -FLT_MAX, -FLT_MAX };
    for (long long v = v_begin + threadIdx.x; v < v_end; v += blockDim.x) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            float x = verts[v * 3 + c];
            lo[c] = fminf(lo[c], x); hi[c] = fmaxf(hi[c], x);
        }
    }
    __shared__ float s_lo[3][8], s_hi[3][8];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        for (int o = 16; o > 0; o >>= 1) {
            lo[c] = fminf(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], o));
            hi[c] = fmaxf(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], o));
        }
        if ((threadIdx.x & 31) == 0) { s_lo[c][threadIdx.x >> 5] = lo[c]; s_hi[c][threadIdx.x >> 5] = hi[c]; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int c = 0; c < 3; ++c)
            for (int w = 1; w < 8; ++w) { s_lo[c][0] = fminf(s_lo[c][0], s_lo[c][w]); s_hi[c][0] = fmaxf(s_hi[c][0], s_hi[c][w]); }
        box[2 * k] = make_float4(s_lo[0][0], s_lo[1][0], s_lo[2][0], 0.f);
        box[2 * k + 1] = make_float4(s_hi[0][0], s_hi[1][0], s_hi[2][0], 0.f);
    }
}

__device__ inline u64 spread16(unsigned v)       // 16 bits -> every third bit of 48
{
    u64 x = v & 0xFFFFu;
    x = (x | (x << 16)) & 0x0000FF0000FFull;
    x = (x | (x << 8)) & 0x00F00F00F00Full;
    x = (x | (x << 4)) & 0x0C30C30C30C3ull;
    x = (x | (x << 2)) & 0x249249249249ull;
    return x;
}

__global__ void __launch_bounds__(256)
morton_kernel(const float *verts, const long long *off, int D, long long sumT, const float4 *box,
              u64 *keys, unsigned *vals)
{
    long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= sumT) return;
    const int k = find_design(off, D, g);
    const float4 lo = box[2 * k], hi = box[2 * k + 1];
    const float *v = verts + g * 9;
    float c[3], l[3] = { lo.x, lo.y, lo.z }, h[3] = { hi.x, hi.y, hi.z };
    unsigned q[3];
    // one scale for all axes (cubic cells): an elongated design (19 m of wings, 1.6 m wide) is then
    // split along its long axis first instead of alternating x, y, z halves of a flat box
    const float ext = fmaxf(h[0] - l[0], fmaxf(h[1] - l[1], h[2] - l[2]));
    const float s = ext > 0.f ? 65535.0f / ext : 0.f;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        c[a] = (v[a] + v[3 + a] + v[6 + a]) * (1.0f / 3.0f);
        q[a] = (unsigned)fminf(fmaxf((c[a] - l[a]) * s, 0.f), 65535.f);
    }
    u64 code = (spread16(q[0]) << 2) | (spread16(q[1]) << 1) | spread16(q[2]);
    keys[g] = ((u64)k << 48) | code;
    vals[g] = (unsigned)g;
}

// ---- pack triangles in sorted order; perm = sorted position -> original index in the design ----
__global__ void __launch_bounds__(256)
pack_kernel(const float *verts, const float *mats, const long long *off, int D, long long sumT,
            const unsigned *vals /* nullptr = identity */, float4 *tri, int *perm)
{
    long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= sumT) return;
    const long long src = vals ? (long long)vals[g] : g;
    const int k = find_design(off, D, g);
    const float *v = verts + src * 9;
    const float *m = mats + src * 3;
    tri[3 * g + 0] = make_float4(v[0], v[1], v[2], m[0]);
    tri[3 * g + 1] = make_float4(v[3] - v[0], v[4] - v[1], v[5] - v[2], m[1]);
    tri[3 * g + 2] = make_float4(v[6] - v[0], v[7] - v[1], v[8] - v[2], m[2]);
    perm[g] = (int)(src - off[k]);
}

// ---- Karras hierarchy ----
__device__ inline int delta(const u64 *keys, int n, int i, int j)
{
    if (j < 0 || j >= n) return -1;
    u64 a = keys[i], b = keys[j];
    if (a == b) return 64 + __clz(i ^ j);
    return __clzll((long long)(a ^ b));
}

// child encoding in the temporary arrays: >= 0 internal node (local), < 0 leaf ~pos (local sorted position)
__global__ void __launch_bounds__(256)
hierarchy_kernel(const u64 *keys_all, const long long *off, int D, long long sumT, int *left,
                 int *right, int *parent_node, int *parent_leaf, int *range_first, int *range_count)
{
    long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= sumT) return;
    const int k = (int)(keys_all[g] >> 48);
    const long long base = off[k];
    const int n = (int)(off[k + 1] - base);
    const int i = (int)(g - base);
    if (i >= n - 1) return;
    const u64 *keys = keys_all + base;
    const int d = (delta(keys, n, i, i + 1) - delta(keys, n, i, i - 1)) >= 0 ? 1 : -1;
    const int dmin = delta(keys, n, i, i - d);
    int lmax = 2;
    while (delta(keys, n, i, i + lmax * d) > dmin) lmax <<= 1;
    int l = 0;
    for (int t = lmax >> 1; t >= 1; t >>= 1)
        if (delta(keys, n, i, i + (l + t) * d) > dmin) l += t;
    const int j = i + l * d;
    const int dnode = delta(keys, n, i, j);
    int s = 0, t = l;
    do {
        t = (t + 1) >> 1;
        if (delta(keys, n, i, i + (s + t) * d) > dnode) s += t;
    } while (t > 1);
    const int gamma = i + s * d + min(d, 0);
    const int first = min(i, j), last = max(i, j);
    int L, R;
    if (first == gamma) { L = ~gamma; parent_leaf[base + gamma] = i; }
    else { L = gamma; parent_node[base + gamma] = i; }
    if (last == gamma + 1) { R = ~(gamma + 1); parent_leaf[base + gamma + 1] = i; }
    else { R = gamma + 1; parent_node[base + gamma + 1] = i; }
    left[g] = L; right[g] = R;
    range_first[g] = first; range_count[g] = last - first + 1;
    if (i == 0) parent_node[base] = -1;
}

// ---- bottom-up refit: the second thread to arrive at a node merges its children's boxes ----
__global__ void __launch_bounds__(256)
refit_kernel(const float4 *tri, const long long *off, int D, long long sumT, const int *left,
             const int *right, const int *parent_node, const int *parent_leaf, int *flags,
             float4 *lbox, float4 *nbox)
{
    long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= sumT) return;
    const float4 a = tri[3 * g], e1 = tri[3 * g + 1], e2 = tri[3 * g + 2];
    float3 lo = make_float3(a.x, a.y, a.z), hi = lo;
    const float3 p1 = make_float3(a.x + e1.x, a.y + e1.y, a.z + e1.z);
    const float3 p2 = make_float3(a.x + e2.x, a.y + e2.y, a.z + e2.z);
    lo.x = fminf(lo.x, fminf(p1.x, p2.x)); hi.x = fmaxf(hi.x, fmaxf(p1.x, p2.x));
    lo.y = fminf(lo.y, fminf(p1.y, p2.y)); hi.y = fmaxf(hi.y, fmaxf(p1.y, p2.y));
    lo.z = fminf(lo.z, fminf(p1.z, p2.z)); hi.z = fmaxf(hi.z, fmaxf(p1.z, p2.z));
    lbox[2 * g] = make_float4(lo.x, lo.y, lo.z, 0.f);
    lbox[2 * g + 1] = make_float4(hi.x, hi.y, hi.z, 0.f);
    const int k = find_design(off, D, g);
    const long long base = off[k];
    if (off[k + 1] - base < 2) return;
    int cur = parent_leaf[g];
    for (;;) {
        __threadfence();
        if (atomicAdd(&flags[base + cur], 1) == 0) return;
        float4 blo, bhi;
#pragma unroll
        for (int side = 0; side < 2; ++side) {
            const int c = side ? right[base + cur] : left[base + cur];
            const float4 *src = c < 0 ? lbox + 2 * (base + ~c) : nbox + 2 * (base + c);
            const float4 clo = __ldcg(src), chi = __ldcg(src + 1);
            if (side == 0) { blo = clo; bhi = chi; }
            else {
                blo.x = fminf(blo.x, clo.x); blo.y = fminf(blo.y, clo.y); blo.z = fminf(blo.z, clo.z);
                bhi.x = fmaxf(bhi.x, chi.x); bhi.y = fmaxf(bhi.y, chi.y); bhi.z = fmaxf(bhi.z, chi.z);
            }
        }
        nbox[2 * (base + cur)] = blo;
        nbox[2 * (base + cur) + 1] = bhi;
        cur = parent_node[base + cur];
        if (cur < 0) return;
    }
}

// ---- emit the traversal layout ----
__global__ void __launch_bounds__(256)
emit_kernel(const unsigned long long *keys_all, const long long *off, long long sumT, const int *left,
            const int *right, const int *range_first, const int *range_count, const float4 *lbox,
            const float4 *nbox, float4 *nodes, int leaf_max)
{
    long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= sumT) return;
    const int k = (int)(keys_all[g] >> 48);
    const long long base = off[k];
    const int n = (int)(off[k + 1] - base);
    const int i = (int)(g - base);
    float4 lo[2], hi[2];
    int link[2];
    if (n == 1) {                       // single triangle: root with one real leaf and one empty box
        lo[0] = lbox[2 * g]; hi[0] = lbox[2 * g + 1]; link[0] = ~0;
        lo[1] = make_float4(FLT_MAX, FLT_MAX, FLT_MAX, 0.f);
        hi[1] = make_float4(-FLT_MAX, -FLT_MAX, -FLT_MAX, 0.f); link[1] = ~0;
    } else {
        if (i >= n - 1) return;
#pragma unroll
        for (int side = 0; side < 2; ++side) {
            const int c = side ? right[g] : left[g];
            if (c < 0) {
                const long long p = base + ~c;
                lo[side] = lbox[2 * p]; hi[side] = lbox[2 * p + 1];
                link[side] = ~((~c) << 3);
            } else {
                lo[side] = nbox[2 * (base + c)]; hi[side] = nbox[2 * (base + c) + 1];
                const int cnt = range_count[base + c];
                link[side] = cnt <= leaf_max ? ~((range_first[base + c] << 3) | (cnt - 1)) : c;
            }
        }
    }
    nodes[4 * g + 0] = make_float4(lo[0].x, lo[0].y, lo[0].z, hi[0].x);
    nodes[4 * g + 1] = make_float4(hi[0].y, hi[0].z, lo[1].x, lo[1].y);
    nodes[4 * g + 2] = make_float4(lo[1].z, hi[1].x, hi[1].y, hi[1].z);
    // spare words: the node's own sorted triangle range (first, count) -- read by node_plane_kernel
    nodes[4 * g + 3] = make_float4(__int_as_float(link[0]), __int_as_float(link[1]),
                                   __int_as_float(n == 1 ? 0 : range_first[g]), __int_as_float(n == 1 ? 1 : range_count[g]));
}

// ---- per-node plane slab (for the escape masks): the tightest slab dmin <= n . x <= dmax that holds all vertices
// of the node's triangles, along n = the normalised sum of their area normals.  A flat patch gives dmax - dmin ~ 1e-6;
// escape_mask.cu uses it to tell "this whole subtree lies in my plane" where the axis-aligned box of a tilted patch
// cannot.  One thread per internal node, two passes over its (contiguous, sorted) triangle range.
__global__ void __launch_bounds__(256)
node_plane_kernel(const DesignsDev dz, long long sumT, float4 *nplane)
{
    // one warp per node: the top nodes span the whole design, so the lanes share a node's triangle range
    const long long g = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (g >= sumT) return;
    const int k = find_design(dz.tri_off, dz.D, g);
    const long long base = dz.tri_off[k];
    const int n = (int)(dz.tri_off[k + 1] - base);
    const int i = (int)(g - base);
    if (i >= n - 1 && !(n == 1 && i == 0)) return;
    const float4 rec = dz.nodes[4 * g + 3];
    const int first = __float_as_int(rec.z), cnt = __float_as_int(rec.w);
    const float4 *t = dz.tri + 3 * (base + first);
    float sx = 0.f, sy = 0.f, sz = 0.f;
    for (int f = lane; f < cnt; f += 32) {
        const float4 e1 = t[3 * f + 1], e2 = t[3 * f + 2];
        sx += e1.y * e2.z - e1.z * e2.y; sy += e1.z * e2.x - e1.x * e2.z; sz += e1.x * e2.y - e1.y * e2.x;
    }
    for (int off = 16; off > 0; off >>= 1) {               // xor tree: every lane ends with the same sums
        sx += __shfl_xor_sync(0xffffffffu, sx, off); sy += __shfl_xor_sync(0xffffffffu, sy, off);
        sz += __shfl_xor_sync(0xffffffffu, sz, off);
    }
    const float len = sqrtf(sx * sx + sy * sy + sz * sz);
    if (!(len > 0.f)) {                                   // normals cancel: no usable plane
        if (lane == 0) {
            nplane[2 * g] = make_float4(0.f, 0.f, 0.f, -FLT_MAX); nplane[2 * g + 1] = make_float4(FLT_MAX, 0.f, 0.f, 0.f);
        }
        return;
    }
    sx /= len; sy /= len; sz /= len;
    float dmin = FLT_MAX, dmax = -FLT_MAX;
    for (int f = lane; f < cnt; f += 32) {
        const float4 a = t[3 * f], e1 = t[3 * f + 1], e2 = t[3 * f + 2];
        const float d0 = sx * a.x + sy * a.y + sz * a.z;
        const float d1 = sx * (a.x + e1.x) + sy * (a.y + e1.y) + sz * (a.z + e1.z);
        const float d2 = sx * (a.x + e2.x) + sy * (a.y + e2.y) + sz * (a.z + e2.z);
        dmin = fminf(dmin, fminf(d0, fminf(d1, d2))); dmax = fmaxf(dmax, fmaxf(d0, fmaxf(d1, d2)));
    }
    for (int off = 16; off > 0; off >>= 1) {
        dmin = fminf(dmin, __shfl_xor_sync(0xffffffffu, dmin, off)); dmax = fmaxf(dmax, __shfl_xor_sync(0xffffffffu, dmax, off));
    }
    if (lane == 0) {
        nplane[2 * g] = make_float4(sx, sy, sz, dmin);
        nplane[2 * g + 1] = make_float4(dmax, 0.f, 0.f, 0.f);
    }
}

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return e_; } while (0)

} // namespace

// Builds box / tri / perm (and nodes when the batch has a design above the brute-force limit) from
// verts_orig / mats_orig.  All device arrays of `dz` are already allocated.
cudaError_t srp_launch_build(srp_designs *dz, int leaf_max, int builder, cudaMemPool_t pool, cudaStream_t stream, int *launches)
{
    const long long sumT = dz->sumT;
    const int D = dz->D;
    const unsigned blocks = (unsigned)((sumT + 255) / 256);
    design_box_kernel<<<D, 256, 0, stream>>>(dz->verts_orig, dz->tri_off_dev, dz->box);
    if (!dz->has_bvh) {
        pack_kernel<<<blocks, 256, 0, stream>>>(dz->verts_orig, dz->mats_orig, dz->tri_off_dev, D, sumT,
                                                nullptr, dz->tri, dz->perm);
        *launches = 2;
        return cudaGetLastError();
    }
    // scratch of the build, from the context's pool; freed (stream-ordered) whether or not the build succeeds
    u64 *keys = nullptr, *keys_out = nullptr;
    unsigned *vals = nullptr, *vals_out = nullptr;
    int *ibuf = nullptr;          // left, right, parent_node, parent_leaf, range_first, range_count, flags
    float4 *lbox = nullptr, *nbox = nullptr;
    void *tmp = nullptr; size_t tmp_bytes = 0;
    if (leaf_max < 1 || leaf_max > 8) leaf_max = SRP_LEAF_MAX;       // srp_options.leaf_max; 0 = default
    auto build = [&]() -> cudaError_t {
        CK(cudaMallocFromPoolAsync((void **)&keys, sizeof(u64) * sumT, pool, stream));
        CK(cudaMallocFromPoolAsync((void **)&keys_out, sizeof(u64) * sumT, pool, stream));
        CK(cudaMallocFromPoolAsync((void **)&vals, sizeof(unsigned) * sumT, pool, stream));
        CK(cudaMallocFromPoolAsync((void **)&vals_out, sizeof(unsigned) * sumT, pool, stream));
        if (builder == 1) {
            CK(cudaMallocFromPoolAsync((void **)&ibuf, sizeof(int) * 7 * sumT, pool, stream));
            CK(cudaMallocFromPoolAsync((void **)&lbox, sizeof(float4) * 2 * sumT, pool, stream));
            CK(cudaMallocFromPoolAsync((void **)&nbox, sizeof(float4) * 2 * sumT, pool, stream));
        }
        int end_bit = 48;
        while ((1LL << (end_bit - 48)) < D) ++end_bit;
        CK(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys, keys_out, vals, vals_out, (int)sumT, 0,
                                           end_bit, stream));
        CK(cudaMallocFromPoolAsync(&tmp, tmp_bytes, pool, stream));
        morton_kernel<<<blocks, 256, 0, stream>>>(dz->verts_orig, dz->tri_off_dev, D, sumT, dz->box, keys, vals);
        CK(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, keys, keys_out, vals, vals_out, (int)sumT, 0,
                                           end_bit, stream));
        *launches = 2 + 4;                     // box, codes; the sort: histogram, exclusive sum, 2 onesweep passes or more
        if (builder != 1) {                    // binned SAH over the Morton order (bvh_sah.cu); `vals` is free again
            int n = 0;
            CK(srp_launch_sah_build(dz, vals_out, vals, leaf_max, pool, stream, &n));
            pack_kernel<<<blocks, 256, 0, stream>>>(dz->verts_orig, dz->mats_orig, dz->tri_off_dev, D, sumT,
                                                    vals, dz->tri, dz->perm);
            *launches += n + 1;
            return cudaGetLastError();
        }
        pack_kernel<<<blocks, 256, 0, stream>>>(dz->verts_orig, dz->mats_orig, dz->tri_off_dev, D, sumT,
                                                vals_out, dz->tri, dz->perm);
        *launches += 5;
        int *left = ibuf, *right = ibuf + sumT, *pnode = ibuf + 2 * sumT, *pleaf = ibuf + 3 * sumT,
            *rfirst = ibuf + 4 * sumT, *rcount = ibuf + 5 * sumT, *flags = ibuf + 6 * sumT;
        CK(cudaMemsetAsync(flags, 0, sizeof(int) * sumT, stream));
        hierarchy_kernel<<<blocks, 256, 0, stream>>>(keys_out, dz->tri_off_dev, D, sumT, left, right, pnode,
                                                     pleaf, rfirst, rcount);
        refit_kernel<<<blocks, 256, 0, stream>>>(dz->tri, dz->tri_off_dev, D, sumT, left, right, pnode, pleaf,
                                                 flags, lbox, nbox);
        emit_kernel<<<blocks, 256, 0, stream>>>(keys_out, dz->tri_off_dev, sumT, left, right, rfirst, rcount,
                                                lbox, nbox, dz->nodes, leaf_max);
        return cudaGetLastError();
    };
    const cudaError_t e = build();
    void *scratch[8] = { keys, keys_out, vals, vals_out, ibuf, lbox, nbox, tmp };
    for (void *q : scratch)
        if (q) cudaFreeAsync(q, stream);
    return e;
}

// Shininess (R23) comes in the caller's triangle order; the trace kernels index triangles by sorted position.
__global__ void __launch_bounds__(256)
gather_shininess_kernel(const DesignsDev dz, long long sumT, const float *__restrict__ shin_orig, float *__restrict__ shin_sorted)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= sumT) return;
    const int k = find_design(dz.tri_off, dz.D, g);
    shin_sorted[g] = shin_orig[dz.tri_off[k] + dz.perm[g]];
}

cudaError_t srp_launch_gather_shininess(const DesignsDev &dz, long long sumT, const float *shin_orig, float *shin_sorted,
                                        cudaStream_t stream)
{
    gather_shininess_kernel<<<(unsigned)((sumT + 255) / 256), 256, 0, stream>>>(dz, sumT, shin_orig, shin_sorted);
    return cudaGetLastError();
}

// Per-node plane slabs for the escape masks (built lazily with them, srp_api.cu).
cudaError_t srp_launch_node_planes(const DesignsDev &dz, long long sumT, float4 *nplane, cudaStream_t stream)
{
    node_plane_kernel<<<(unsigned)((sumT + 7) / 8), 256, 0, stream>>>(dz, sumT, nplane);
    return cudaGetLastError();
}
