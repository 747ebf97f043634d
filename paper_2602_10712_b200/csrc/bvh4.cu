// bvh4.cu -- S1, after the BVH2 is built: 4-wide nodes for per-ray traversal, folded from the BVH2 (every node takes
// its grandchildren, or a child that is a leaf, as its up to four children).  A wide node keeps the number of its
// BVH2 node, so links need no translation; slots of numbers that no traversal reaches from the root stay unused.
// Record = 8 x float4 = 128 B: 4 child boxes (lo.xyz, hi.xyz) in words 0..23, 4 links in words 24..27 (link as in the
// BVH2: >= 0 node, < 0 leaf), unused children have an empty box (lo = FLT_MAX, hi = -FLT_MAX) that no ray meets.
#include <cfloat>
#include "srp_internal.cuh"

namespace {

__device__ inline int find_design4(const long long *off, int D, long long g)
{
    int lo = 0, hi = D;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (off[mid] <= g) lo = mid; else hi = mid;
    }
    return lo;
}

struct Child { float b[6]; int link; };

__device__ inline void children_of(const float4 *nodes, long long g, Child c[2])
{
    const float4 n0 = nodes[4 * g], n1 = nodes[4 * g + 1], n2 = nodes[4 * g + 2], n3 = nodes[4 * g + 3];
    c[0].b[0] = n0.x; c[0].b[1] = n0.y; c[0].b[2] = n0.z; c[0].b[3] = n0.w; c[0].b[4] = n1.x; c[0].b[5] = n1.y;
    c[1].b[0] = n1.z; c[1].b[1] = n1.w; c[1].b[2] = n2.x; c[1].b[3] = n2.y; c[1].b[4] = n2.z; c[1].b[5] = n2.w;
    c[0].link = __float_as_int(n3.x); c[1].link = __float_as_int(n3.y);
}

__global__ void __launch_bounds__(256)
collapse4_kernel(const float4 *nodes, const long long *off, int D, long long sumT, float4 *nodes4)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= sumT) return;
    const int k = find_design4(off, D, g);
    const long long base = off[k];
    const int n = (int)(off[k + 1] - base);
    const int i = (int)(g - base);
    if (i >= n - 1 && !(n == 1 && i == 0)) return;
    if (__float_as_int(nodes[4 * g + 3].w) == 0) return;          // a number no node took (count = 0)
    Child two[2], out[4];
    int m = 0;
    children_of(nodes, g, two);
    for (int side = 0; side < 2; ++side) {
        const bool empty = two[side].b[3] < two[side].b[0];
        if (two[side].link < 0 || empty) { if (!empty) out[m++] = two[side]; }
        else {
            Child gc[2];
            children_of(nodes, base + two[side].link, gc);
            for (int s2 = 0; s2 < 2; ++s2)
                if (!(gc[s2].b[3] < gc[s2].b[0])) out[m++] = gc[s2];
        }
    }
    for (; m < 4; ++m) {
        out[m].b[0] = out[m].b[1] = out[m].b[2] = FLT_MAX; out[m].b[3] = out[m].b[4] = out[m].b[5] = -FLT_MAX;
        out[m].link = ~0;
    }
    float w[32];
    for (int c = 0; c < 4; ++c) {
        for (int x = 0; x < 6; ++x) w[6 * c + x] = out[c].b[x];
        w[24 + c] = __int_as_float(out[c].link);
    }
    for (int x = 28; x < 32; ++x) w[x] = 0.f;
    for (int q = 0; q < 8; ++q) nodes4[8 * g + q] = make_float4(w[4 * q], w[4 * q + 1], w[4 * q + 2], w[4 * q + 3]);
}

} // namespace

cudaError_t srp_launch_collapse4(const srp_designs *dz, cudaStream_t stream)
{
    collapse4_kernel<<<(unsigned)((dz->sumT + 255) / 256), 256, 0, stream>>>(dz->nodes, dz->tri_off_dev, dz->D, dz->sumT, dz->nodes4);
    return cudaGetLastError();
}
