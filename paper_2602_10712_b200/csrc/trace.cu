// trace.cu -- which trace kernel runs (S2-S7), and the roofline probes.
//   beam_trace_kernel   (trace_beam.cu)    designs with a BVH, stratified sampler, many rays per triangle
//   small_beam_kernel   (trace_small.cu)   designs without a hierarchy (T <= 64), stratified sampler
//   bvh_trace_kernel    (trace_perray.cu)  designs with a BVH otherwise (about one ray per triangle, i.i.d. sampler)
//   trace_kernel        (trace_perray.cu)  all triangles for every segment: T <= 64 with the i.i.d. sampler, force_brute
#include "srp_internal.cuh"

int srp_perray_blocks_per_sm(bool brute);
int srp_beam_blocks_per_sm();
int srp_small_blocks_per_sm();
cudaError_t srp_launch_perray(const TraceArgs &a, int mode, bool instrumented, int num_sms, cudaStream_t stream);
cudaError_t srp_launch_beam(const TraceArgs &a, bool instrumented, int num_sms, cudaStream_t stream);
cudaError_t srp_launch_small(const TraceArgs &a, bool instrumented, int num_sms, cudaStream_t stream);

// resident warps per SM of the kernel that will run (tile sizing in srp_api.cu)
int srp_trace_blocks_per_sm(bool brute, bool beam)
{
    const int per_sm = brute ? (beam ? srp_small_blocks_per_sm() : srp_perray_blocks_per_sm(true))
                             : (beam ? srp_beam_blocks_per_sm() : srp_perray_blocks_per_sm(false));
    return per_sm * 4;
}

cudaError_t srp_launch_trace(const TraceArgs &a, bool brute, bool instrumented, int num_sms, cudaStream_t stream)
{
    if (brute) {
        if (a.dz.has_bvh)       // forced brute force over a design that also has a hierarchy (test use)
            return srp_launch_perray(a, 2, instrumented, num_sms, stream);
        if (a.sampler == 0 && a.primary_mode != 1) return srp_launch_small(a, instrumented, num_sms, stream);
        return srp_launch_perray(a, 0, instrumented, num_sms, stream);
    }
    if (a.sampler == 0 && a.rq != nullptr)          // beams chosen by the caller (srp_api.cu, want_beams)
        return srp_launch_beam(a, instrumented, num_sms, stream);
    return srp_launch_perray(a, 1, instrumented, num_sms, stream);
}

// ---- roofline probes ----
namespace {
__global__ void __launch_bounds__(256) fma_probe_kernel(float *out, int iters, float a, float b)
{
    float x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
            x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
        }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}
__global__ void __launch_bounds__(256) l2_probe_kernel(const float4 *buf, size_t n_vec, int passes, float *out)
{
    float s = 0.f;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int p = 0; p < passes; ++p)
        for (size_t x = (size_t)blockIdx.x * blockDim.x + threadIdx.x; x < n_vec; x += stride) {
            const float4 v = __ldcg(buf + x);
            s += v.x + v.y + v.z + v.w;
        }
    if (s == 12345.678f) out[0] = s;
}
} // namespace

cudaError_t srp_run_probes(int num_sms, cudaStream_t stream, double *fp32_tflops, double *l2_gbs)
{
    float *out = nullptr; float4 *buf = nullptr;
    const int blocks = num_sms * 8, iters = 4096;
    const size_t n_vec = (size_t)32 << 20 >> 4;           // 32 MiB, well inside L2
    cudaError_t e = cudaMalloc(&out, sizeof(float) * blocks * 256);
    if (e != cudaSuccess) return e;
    e = cudaMalloc(&buf, n_vec * sizeof(float4));
    if (e != cudaSuccess) { cudaFree(out); return e; }
    cudaMemsetAsync(buf, 0, n_vec * sizeof(float4), stream);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best_f = 0, best_l = 0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0, stream);
        fma_probe_kernel<<<blocks, 256, 0, stream>>>(out, iters, 0.999f, 0.001f);
        cudaEventRecord(e1, stream);
        cudaEventSynchronize(e1);
        float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
        double tf = 2.0 * 64.0 * iters * blocks * 256.0 / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best_f) best_f = tf;
        const int passes = 20;
        cudaEventRecord(e0, stream);
        l2_probe_kernel<<<num_sms * 8, 256, 0, stream>>>(buf, n_vec, passes, out);
        cudaEventRecord(e1, stream);
        cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        double gb = (double)passes * n_vec * 16.0 / (ms * 1e-3) / 1e9;
        if (rep > 0 && gb > best_l) best_l = gb;
    }
    e = cudaGetLastError();
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out); cudaFree(buf);
    *fp32_tflops = best_f; *l2_gbs = best_l;
    return e;
}
