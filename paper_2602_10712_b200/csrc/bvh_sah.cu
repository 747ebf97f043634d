// bvh_sah.cu -- S1 of the hot path, default builder: a top-down binned surface-area-heuristic BVH2 over the
// Morton-sorted triangles of every design of a batch, built level by level on the device (PAPER.md:366 builds a
// linear BVH; per-ray traversal of bounce rays costs 27 % fewer node steps in this hierarchy).
//
// A node is a contiguous range of positions [head, head + count) of its design's triangle order; the order starts as
// the Morton order and every level partitions each range in place (stably), so the final order is a depth-first order
// of the leaves and every node's triangles stay contiguous -- the layout lbvh.cu emits and every trace kernel reads.
// One level =
//   bin      every triangle of an open node adds its box to 3 axes x 16 bins of its node (integer atomics on
//            order-preserving codes of the floats: the result does not depend on the order of arrival)
//   split    one warp per open node: 45 candidate planes, cost = area(L) n(L) + area(R) n(R); the node takes its
//            number (head + n(L) - 1: the position it splits after, unique like Karras's), links itself to its parent,
//            opens its children or writes them as leaves (<= leaf_max triangles)
//   flag / scan / scatter   stable partition by an exclusive sum over "goes right"
// A node whose centroids coincide (duplicate triangles), and every node below level `sah_levels`, is halved by
// position instead; `levels` bounds the depth (the traversal stacks hold 92 entries).
// Afterwards the boxes are fitted bottom-up (second arrival at a node merges its children) straight into the 64-byte
// traversal nodes.  Everything is enqueued on the stream; nothing is read back.
#include <cub/device/device_scan.cuh>
#include <cfloat>
#include "srp_internal.cuh"

namespace {

#ifndef SAH_BINS_DEF
#define SAH_BINS_DEF 16
#endif
constexpr int NB = SAH_BINS_DEF;        // bins per axis
constexpr int BIN_WORDS = 3 * NB * 7;   // per open node: [axis][bin]{lo.xyz, hi.xyz as codes, count}
constexpr unsigned FULL = 0xffffffffu;

// order-preserving code of a float: a < b  <=>  code(a) < code(b) as unsigned
__device__ __forceinline__ unsigned f2o(float f)
{
    const unsigned b = __float_as_uint(f);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float o2f(unsigned u)
{
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
}

__device__ inline int find_design(const long long *off, int D, long long g)
{
    int lo = 0, hi = D;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (off[mid] <= g) lo = mid; else hi = mid;
    }
    return lo;
}

struct Sah {                 // scratch of one build; `cur` / `nxt` index the ping-pong halves
    long long sumT;
    int D, leaf_max;
    const long long *off;
    const float4 *lbox;      // [2 sumT] triangle boxes in Morton order
    unsigned *idx[2];        // [sumT] position -> Morton position
    int *head[2];            // [sumT] position -> head position of its open node, -1 = in a finished leaf
    int *count[2];           // per open node, at its head position
    int *parent[2];          //   2 * (global id of the parent) + side, -1 = root
    unsigned *cb[2];         //   [6 sumT] bounds of the centroid sums lo + hi (codes): min xyz, max xyz
    int4 *dec;               //   decision of this level: axis, last left bin, n(L), 1 = by position
    unsigned *bins;          // [slots * BIN_WORDS], slot = head / (leaf_max + 1)
    int *flag, *scan;        // [sumT]
    int *rootnat;            // [D] the number the root would have taken
    int *parent_of;          // [sumT] per node id: 2 * parent id + side (global ids), -1 = root
    int *arrived;            // [sumT] refit flags
    float4 *nodes;           // output
};

__device__ __forceinline__ long long slot_of(const Sah &s, int head) { return head / (s.leaf_max + 1); }

__device__ __forceinline__ int bin_of(float c, float cmin, float cmax)
{
    const float ext = cmax - cmin;
    if (!(ext > 0.f)) return 0;
    const int b = (int)((c - cmin) * ((float)NB / ext));
    return b < 0 ? 0 : (b > NB - 1 ? NB - 1 : b);
}

// lanes with the same key add their (lo, hi) to one set of 6 codes with one atomic per word
__device__ __forceinline__ void grouped_minmax(unsigned *dst, bool active, int key, const float lo[3], const float hi[3],
                                               int *count_dst)
{
    const int lane = threadIdx.x & 31;
    const unsigned m = __match_any_sync(FULL, active ? key : -1);
    unsigned v[6];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        v[c] = __reduce_min_sync(m, f2o(lo[c]));
        v[3 + c] = __reduce_max_sync(m, f2o(hi[c]));
    }
    if (active && (__ffs(m) - 1) == lane) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { atomicMin(dst + c, v[c]); atomicMax(dst + 3 + c, v[3 + c]); }
        if (count_dst) atomicAdd(count_dst, __popc(m));
    }
}

__device__ __forceinline__ void open_node(const Sah &s, int nx, int head, int count, int parent)
{
    s.count[nx][head] = count; s.parent[nx][head] = parent;
#pragma unroll
    for (int c = 0; c < 3; ++c) { s.cb[nx][6LL * head + c] = 0xffffffffu; s.cb[nx][6LL * head + 3 + c] = 0u; }
}

__device__ __forceinline__ void clear_bins(const Sah &s, int head, int lane)
{
    unsigned *b = s.bins + slot_of(s, head) * BIN_WORDS;
    for (int w = lane; w < BIN_WORDS; w += 32) {
        const int j = w % 7;
        b[w] = j < 3 ? 0xffffffffu : 0u;
    }
}

// ---- triangle boxes in Morton order ----
__global__ void __launch_bounds__(256)
tri_box_kernel(const float *verts, const unsigned *vals, long long sumT, float4 *lbox)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= sumT) return;
    const float *v = verts + (long long)vals[g] * 9;
    float lo[3], hi[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        lo[c] = fminf(v[c], fminf(v[3 + c], v[6 + c]));
        hi[c] = fmaxf(v[c], fmaxf(v[3 + c], v[6 + c]));
    }
    lbox[2 * g] = make_float4(lo[0], lo[1], lo[2], 0.f);
    lbox[2 * g + 1] = make_float4(hi[0], hi[1], hi[2], 0.f);
}

// ---- level 0: every design with two or more triangles opens its root ----
__global__ void __launch_bounds__(256)
sah_init_kernel(Sah s)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool in = g < s.sumT;
    int head = -1;
    if (in) {
        const int k = find_design(s.off, s.D, g);
        const long long base = s.off[k];
        if (s.off[k + 1] - base >= 2) head = (int)base;
        s.idx[0][g] = (unsigned)g;
        s.head[0][g] = head;
        s.arrived[g] = 0; s.parent_of[g] = -1;
        s.nodes[4 * g + 0] = s.nodes[4 * g + 1] = s.nodes[4 * g + 2] = s.nodes[4 * g + 3] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (head == (int)g) open_node(s, 0, head, (int)(s.off[k + 1] - base), -1);
    }
    const unsigned heads = __ballot_sync(FULL, in && head == (int)g);
    for (unsigned m = heads; m; m &= m - 1) {
        const int h = (int)(g - lane) + (__ffs(m) - 1);
        clear_bins(s, h, lane);
    }
}

__global__ void __launch_bounds__(256)
sah_root_centroids_kernel(Sah s)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool in = g < s.sumT;
    const int head = in ? s.head[0][g] : -1;
    float c[3] = { 0.f, 0.f, 0.f };
    if (head >= 0) {
        const float4 lo = s.lbox[2 * g], hi = s.lbox[2 * g + 1];
        c[0] = lo.x + hi.x; c[1] = lo.y + hi.y; c[2] = lo.z + hi.z;
    }
    grouped_minmax(s.cb[0] + 6LL * (head < 0 ? 0 : head), head >= 0, head, c, c, nullptr);
}

// ---- bin ----
__global__ void __launch_bounds__(256)
sah_bin_kernel(Sah s, int cur)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool in = g < s.sumT;
    const int head = in ? s.head[cur][g] : -1;
    if (__ballot_sync(FULL, head >= 0) == 0u) return;
    float lo[3] = { 0.f, 0.f, 0.f }, hi[3] = { 0.f, 0.f, 0.f };
    int bin[3] = { 0, 0, 0 };
    if (head >= 0) {
        const unsigned t = s.idx[cur][g];
        const float4 l = s.lbox[2LL * t], h = s.lbox[2LL * t + 1];
        lo[0] = l.x; lo[1] = l.y; lo[2] = l.z; hi[0] = h.x; hi[1] = h.y; hi[2] = h.z;
        const unsigned *cb = s.cb[cur] + 6LL * head;
#pragma unroll
        for (int a = 0; a < 3; ++a) bin[a] = bin_of(lo[a] + hi[a], o2f(cb[a]), o2f(cb[3 + a]));
    }
    unsigned *b = s.bins + (head < 0 ? 0 : slot_of(s, head)) * BIN_WORDS;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        unsigned *d = b + (a * NB + bin[a]) * 7;
        grouped_minmax(d, head >= 0, head * NB + bin[a], lo, hi, (int *)(d + 6));
    }
}

__device__ __forceinline__ float half_area(const float lo[3], const float hi[3])
{
    const float dx = hi[0] - lo[0], dy = hi[1] - lo[1], dz = hi[2] - lo[2];
    return dx * dy + dy * dz + dx * dz;
}

// ---- split: one warp per 32 positions, the open nodes whose head lies among them one after the other ----
__global__ void __launch_bounds__(256)
sah_split_kernel(Sah s, int cur, int by_position)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool in = g < s.sumT;
    const unsigned heads = __ballot_sync(FULL, in && s.head[cur][g] == (int)g);
    const int nx = cur ^ 1;
    for (unsigned m = heads; m; m &= m - 1) {
        const int h = (int)(g - lane) + (__ffs(m) - 1);
        const int count = s.count[cur][h];
        const unsigned *b = s.bins + slot_of(s, h) * BIN_WORDS;
        float best = FLT_MAX;                        // this lane's cheapest candidate plane, then the warp's
        int who = 3 * (NB - 1), nl_best = 0;
        for (int cand = lane; cand < 3 * (NB - 1) && !by_position; cand += 32) {
            const int a = cand / (NB - 1), sp = cand % (NB - 1);       // left = bins 0..sp of axis a
            float llo[3] = { FLT_MAX, FLT_MAX, FLT_MAX }, lhi[3] = { -FLT_MAX, -FLT_MAX, -FLT_MAX };
            float rlo[3] = { FLT_MAX, FLT_MAX, FLT_MAX }, rhi[3] = { -FLT_MAX, -FLT_MAX, -FLT_MAX };
            int nl = 0, nr = 0;
            for (int i = 0; i < NB; ++i) {
                const unsigned *w = b + (a * NB + i) * 7;
                const int n = (int)w[6];
                if (n == 0) continue;
                if (i <= sp) {
                    nl += n;
#pragma unroll
                    for (int c = 0; c < 3; ++c) { llo[c] = fminf(llo[c], o2f(w[c])); lhi[c] = fmaxf(lhi[c], o2f(w[3 + c])); }
                } else {
                    nr += n;
#pragma unroll
                    for (int c = 0; c < 3; ++c) { rlo[c] = fminf(rlo[c], o2f(w[c])); rhi[c] = fmaxf(rhi[c], o2f(w[3 + c])); }
                }
            }
            if (nl > 0 && nr > 0) {
                const float cost = half_area(llo, lhi) * (float)nl + half_area(rlo, rhi) * (float)nr;
                if (cost < best) { best = cost; who = cand; nl_best = nl; }
            }
        }
        // the cheapest candidate of the warp, the lowest-numbered among equals
        for (int o = 16; o > 0; o >>= 1) {
            const float oc = __shfl_xor_sync(FULL, best, o);
            const int ow = __shfl_xor_sync(FULL, who, o);
            const int on = __shfl_xor_sync(FULL, nl_best, o);
            if (oc < best || (oc == best && ow < who)) { best = oc; who = ow; nl_best = on; }
        }
        const bool positional = !(best < FLT_MAX);
        const int n_left = positional ? count / 2 : nl_best;
        __syncwarp();
        if (lane == 0) {
            const int k = find_design(s.off, s.D, h);
            const int base = (int)s.off[k];
            const int par = s.parent[cur][h];
            const int nat = (h - base) + n_left - 1;
            int id;
            if (par < 0) { id = 0; s.rootnat[k] = nat; }
            else id = nat == 0 ? s.rootnat[k] : nat;
            const long long gid = (long long)base + id;
            s.dec[h] = make_int4(positional ? 0 : who / (NB - 1), positional ? 0 : who % (NB - 1), n_left, positional ? 1 : 0);
            s.parent_of[gid] = par;
            int *rec = (int *)(s.nodes + 4 * gid + 3);
            rec[2] = h - base; rec[3] = count;
            if (par >= 0) ((int *)(s.nodes + 4 * (long long)(par >> 1) + 3))[par & 1] = id;
            const int ch[2] = { h, h + n_left }, cn[2] = { n_left, count - n_left };
#pragma unroll
            for (int side = 0; side < 2; ++side) {
                if (cn[side] <= s.leaf_max) rec[side] = ~(((ch[side] - base) << 3) | (cn[side] - 1));
                else open_node(s, nx, ch[side], cn[side], (int)(gid * 2 + side));
            }
        }
        __syncwarp();
        // the bins of the children that stay open, for the next level (this node's own are read above)
        if (n_left > s.leaf_max) clear_bins(s, h, lane);
        if (count - n_left > s.leaf_max) clear_bins(s, h + n_left, lane);
    }
}

__device__ __forceinline__ int goes_right(const Sah &s, int cur, long long g, int head)
{
    const int4 d = s.dec[head];
    if (d.w) return (int)(g - head) >= d.z;
    const unsigned t = s.idx[cur][g];
    const float4 l = s.lbox[2LL * t], h = s.lbox[2LL * t + 1];
    const float c = d.x == 0 ? l.x + h.x : (d.x == 1 ? l.y + h.y : l.z + h.z);
    const unsigned *cb = s.cb[cur] + 6LL * head;
    return bin_of(c, o2f(cb[d.x]), o2f(cb[3 + d.x])) > d.y;
}

__global__ void __launch_bounds__(256)
sah_flag_kernel(Sah s, int cur)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= s.sumT) return;
    const int head = s.head[cur][g];
    s.flag[g] = head >= 0 ? goes_right(s, cur, g, head) : 0;
}

// ---- scatter: stable partition of every open node; the children's centroid bounds for the next level ----
__global__ void __launch_bounds__(256)
sah_scatter_kernel(Sah s, int cur)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool in = g < s.sumT;
    const int nx = cur ^ 1;
    const int head = in ? s.head[cur][g] : -1;
    int child = -1;
    float c[3] = { 0.f, 0.f, 0.f };
    if (in && head < 0) { s.idx[nx][g] = s.idx[cur][g]; s.head[nx][g] = -1; }
    if (head >= 0) {
        const int4 d = s.dec[head];
        const int right = s.flag[g];
        const int rb = s.scan[g] - s.scan[head];                  // right-goers before this one in its node
        const int count = s.count[cur][head];
        const int pos = right ? head + d.z + rb : head + ((int)(g - head) - rb);
        const unsigned t = s.idx[cur][g];
        s.idx[nx][pos] = t;
        const int cc = right ? count - d.z : d.z;
        child = cc > s.leaf_max ? (right ? head + d.z : head) : -1;
        s.head[nx][pos] = child;
        if (child >= 0) {
            const float4 l = s.lbox[2LL * t], h = s.lbox[2LL * t + 1];
            c[0] = l.x + h.x; c[1] = l.y + h.y; c[2] = l.z + h.z;
        }
    }
    if (__ballot_sync(FULL, child >= 0) == 0u) return;
    grouped_minmax(s.cb[nx] + 6LL * (child < 0 ? 0 : child), child >= 0, child, c, c, nullptr);
}

// ---- after the last level: Morton position -> original index, composed with the final order ----
__global__ void __launch_bounds__(256)
sah_compose_kernel(const unsigned *idx, const unsigned *vals, long long sumT, unsigned *vals_final)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g < sumT) vals_final[g] = vals[idx[g]];
}

// ---- fit the boxes bottom-up into the traversal nodes.  One thread per (node, side) that is a leaf. ----
__device__ __forceinline__ void store_child_box(float4 *nodes, long long gid, int side, const float lo[3], const float hi[3])
{
    float *f = (float *)(nodes + 4 * gid) + 6 * side;
#pragma unroll
    for (int c = 0; c < 3; ++c) { __stcg(f + c, lo[c]); __stcg(f + 3 + c, hi[c]); }
}

__global__ void __launch_bounds__(256)
sah_fit_kernel(Sah s, const unsigned *idx)
{
    const long long gt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long gid0 = gt >> 1;
    const int side0 = (int)(gt & 1);
    if (gid0 >= s.sumT) return;
    const int k = find_design(s.off, s.D, gid0);
    const long long base = s.off[k];
    const int n = (int)(s.off[k + 1] - base);
    if (n == 1) {                        // single triangle: root with one real leaf and one empty box
        float lo[3], hi[3];
        if (side0 == 0) {
            const float4 l = s.lbox[2 * base], h = s.lbox[2 * base + 1];
            lo[0] = l.x; lo[1] = l.y; lo[2] = l.z; hi[0] = h.x; hi[1] = h.y; hi[2] = h.z;
        } else {
            lo[0] = lo[1] = lo[2] = FLT_MAX; hi[0] = hi[1] = hi[2] = -FLT_MAX;
        }
        store_child_box(s.nodes, base, side0, lo, hi);
        int *rec = (int *)(s.nodes + 4 * base + 3);
        rec[side0] = ~0;
        if (side0 == 0) { rec[2] = 0; rec[3] = 1; }
        return;
    }
    const int *rec0 = (const int *)(s.nodes + 4 * gid0 + 3);
    if (rec0[3] == 0) return;            // a number no node took
    const int link = rec0[side0];
    if (link >= 0) return;               // an inner child: its own leaves will come up through it
    const int first = (~link) >> 3, cnt = ((~link) & 7) + 1;
    float lo[3] = { FLT_MAX, FLT_MAX, FLT_MAX }, hi[3] = { -FLT_MAX, -FLT_MAX, -FLT_MAX };
    for (int f = 0; f < cnt; ++f) {
        const unsigned t = idx[base + first + f];
        const float4 l = s.lbox[2LL * t], h = s.lbox[2LL * t + 1];
        lo[0] = fminf(lo[0], l.x); lo[1] = fminf(lo[1], l.y); lo[2] = fminf(lo[2], l.z);
        hi[0] = fmaxf(hi[0], h.x); hi[1] = fmaxf(hi[1], h.y); hi[2] = fmaxf(hi[2], h.z);
    }
    long long gid = gid0;
    int side = side0;
    for (;;) {
        store_child_box(s.nodes, gid, side, lo, hi);
        __threadfence();
        if (atomicAdd(&s.arrived[gid], 1) == 0) return;          // the other child is still on its way
        const float *f = (const float *)(s.nodes + 4 * gid);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            lo[c] = fminf(__ldcg(f + c), __ldcg(f + 6 + c));
            hi[c] = fmaxf(__ldcg(f + 3 + c), __ldcg(f + 9 + c));
        }
        const int par = s.parent_of[gid];
        if (par < 0) return;
        gid = par >> 1; side = par & 1;
    }
}

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return e_; } while (0)

int ceil_log2(long long n) { int l = 0; while ((1LL << l) < n) ++l; return l; }

} // namespace

// `vals`: Morton position -> original global triangle index (the sorted values of lbvh.cu's radix sort).
// Writes dz->nodes and `vals_final` (final position -> original global index); the caller packs the triangles.
cudaError_t srp_launch_sah_build(srp_designs *dz, const unsigned *vals, unsigned *vals_final, int leaf_max,
                                 cudaMemPool_t pool, cudaStream_t stream, int *launches)
{
    const long long sumT = dz->sumT;
    const unsigned blocks = (unsigned)((sumT + 255) / 256);
    Sah s;
    s.sumT = sumT; s.D = dz->D; s.leaf_max = leaf_max; s.off = dz->tri_off_dev; s.nodes = dz->nodes;
    const long long slots = sumT / (leaf_max + 1) + 1;
    void *mem[8] = { nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr };
    int n_launch = 0;
    auto build = [&]() -> cudaError_t {
        float4 *lbox; unsigned *words; void *tmp = nullptr; size_t tmp_bytes = 0;
        CK(cudaMallocFromPoolAsync(&mem[0], sizeof(float4) * 2 * sumT, pool, stream));
        lbox = (float4 *)mem[0];
        // 4-byte arrays: idx 2, head 2, count 2, parent 2, cb 12, flag, scan, parent_of, arrived = 24 sumT, + rootnat
        CK(cudaMallocFromPoolAsync(&mem[1], sizeof(unsigned) * (24 * sumT + dz->D), pool, stream));
        words = (unsigned *)mem[1];
        CK(cudaMallocFromPoolAsync(&mem[2], sizeof(int4) * sumT, pool, stream));
        CK(cudaMallocFromPoolAsync(&mem[3], sizeof(unsigned) * BIN_WORDS * slots, pool, stream));
        for (int h = 0; h < 2; ++h) {
            s.idx[h] = words + (0 + h) * sumT; s.head[h] = (int *)(words + (2 + h) * sumT);
            s.count[h] = (int *)(words + (4 + h) * sumT); s.parent[h] = (int *)(words + (6 + h) * sumT);
            s.cb[h] = words + (8 + 6 * h) * sumT;
        }
        s.flag = (int *)(words + 20 * sumT); s.scan = (int *)(words + 21 * sumT);
        s.parent_of = (int *)(words + 22 * sumT); s.arrived = (int *)(words + 23 * sumT);
        s.rootnat = (int *)(words + 24 * sumT);
        s.dec = (int4 *)mem[2]; s.bins = (unsigned *)mem[3]; s.lbox = lbox;
        CK(cub::DeviceScan::ExclusiveSum(nullptr, tmp_bytes, s.flag, s.scan, (int)sumT, stream));
        CK(cudaMallocFromPoolAsync(&mem[4], tmp_bytes, pool, stream));
        tmp = mem[4];
        tri_box_kernel<<<blocks, 256, 0, stream>>>(dz->verts_orig, vals, sumT, lbox);
        sah_init_kernel<<<blocks, 256, 0, stream>>>(s);
        sah_root_centroids_kernel<<<blocks, 256, 0, stream>>>(s);
        n_launch += 3;
        // depth: planes chosen by cost for 2 log2(n) + 8 levels, then halving by position (log2(n) levels at most)
        const int lg = ceil_log2(dz->maxT > 1 ? dz->maxT : 2);
        const int sah_levels = 2 * lg + 8, levels = sah_levels + lg;
        int cur = 0;
        for (int level = 0; level < levels; ++level) {
            const int by_position = level >= sah_levels;
            if (!by_position) sah_bin_kernel<<<blocks, 256, 0, stream>>>(s, cur);
            sah_split_kernel<<<blocks, 256, 0, stream>>>(s, cur, by_position);
            sah_flag_kernel<<<blocks, 256, 0, stream>>>(s, cur);
            CK(cub::DeviceScan::ExclusiveSum(tmp, tmp_bytes, s.flag, s.scan, (int)sumT, stream));
            sah_scatter_kernel<<<blocks, 256, 0, stream>>>(s, cur);
            n_launch += by_position ? 5 : 6;
            cur ^= 1;
        }
        sah_compose_kernel<<<blocks, 256, 0, stream>>>(s.idx[cur], vals, sumT, vals_final);
        sah_fit_kernel<<<(unsigned)((2 * sumT + 255) / 256), 256, 0, stream>>>(s, s.idx[cur]);
        n_launch += 2;
        return cudaGetLastError();
    };
    const cudaError_t e = build();
    for (void *q : mem)
        if (q) cudaFreeAsync(q, stream);
    if (launches) *launches = n_launch;
    return e;
}
