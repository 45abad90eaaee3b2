// Measured denominators for the rooflines bench.py reports ("builder must measure fp32-FMA
// and L2 peaks"): three small kernels, timed with CUDA events on the system's stream.
//   fp32_tflops  eight independent FFMA chains per thread, every SM full of warps
//   l2_gbs       a 32 MB buffer (resident in the 126 MB L2 after the first pass) read again and again, 16 B per load
//   smem_gbs     conflict-free 16-byte shared-memory loads, four independent address streams per thread: the crossbar
//                the force kernel's neighbor gathers go through
#include "hb_internal.cuh"

constexpr int PK_THREADS = 256;

__global__ void __launch_bounds__(PK_THREADS) peak_fma_kernel(float *out, float b, float c, int iters)
{
    float a0 = threadIdx.x * 1e-3f, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f, a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f, a7 = a0 + 7.f;
#pragma unroll 1
    for (int k = 0; k < iters; k++) {
#pragma unroll
        for (int u = 0; u < 8; u++) {
            a0 = __fmaf_rn(a0, b, c); a1 = __fmaf_rn(a1, b, c); a2 = __fmaf_rn(a2, b, c); a3 = __fmaf_rn(a3, b, c);
            a4 = __fmaf_rn(a4, b, c); a5 = __fmaf_rn(a5, b, c); a6 = __fmaf_rn(a6, b, c); a7 = __fmaf_rn(a7, b, c);
        }
    }
    const float r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (r == 12345.678f) out[0] = r;   // never true in practice: keeps the chains alive
}

__global__ void __launch_bounds__(PK_THREADS) peak_l2_kernel(const float4 *__restrict__ buf, int64_t n4, int passes, float *out)
{
    float acc = 0.f;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int p = 0; p < passes; p++) {
        int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
        for (; i + 3 * stride < n4; i += 4 * stride) {
            const float4 a = __ldcg(buf + i), b = __ldcg(buf + i + stride), c = __ldcg(buf + i + 2 * stride), d = __ldcg(buf + i + 3 * stride);
            acc += (a.x + b.y) + (c.z + d.w);
        }
        for (; i < n4; i += stride) acc += __ldcg(buf + i).x;
    }
    if (acc == 12345.678f) out[0] = acc;
}

// Four address streams per thread, none of which depends on a loaded value (the index advances by a kernel argument,
// so the loads can neither be hoisted nor chained): the loads of one thread are independent and the pipe, not the
// load latency, is what limits the rate.  Consecutive lanes read consecutive 16-byte words: no bank conflict, four
// 128-byte wavefronts per warp instruction.
__global__ void __launch_bounds__(PK_THREADS) peak_smem_kernel(float *out, int iters, int step)
{
    __shared__ int4 tile[PK_THREADS * 4];
    for (int k = threadIdx.x; k < PK_THREADS * 4; k += PK_THREADS) tile[k] = make_int4(k, 1, 0, 3);
    __syncthreads();
    constexpr int MASK = PK_THREADS * 4 - 1;
    int acc0 = 0, acc1 = 0, acc2 = 0, acc3 = 0;
    int i0 = threadIdx.x, i1 = threadIdx.x + PK_THREADS, i2 = threadIdx.x + 2 * PK_THREADS, i3 = threadIdx.x + 3 * PK_THREADS;
#pragma unroll 1
    for (int k = 0; k < iters; k++) {
#pragma unroll
        for (int u = 0; u < 2; u++) {
            const int4 v0 = tile[i0], v1 = tile[i1], v2 = tile[i2], v3 = tile[i3];
            acc0 += (v0.x ^ v0.y) + (v0.z ^ v0.w);
            acc1 += (v1.x ^ v1.y) + (v1.z ^ v1.w);
            acc2 += (v2.x ^ v2.y) + (v2.z ^ v2.w);
            acc3 += (v3.x ^ v3.y) + (v3.z ^ v3.w);
            i0 = (i0 + step) & MASK; i1 = (i1 + step) & MASK; i2 = (i2 + step) & MASK; i3 = (i3 + step) & MASK;
        }
    }
    const int acc = (acc0 + acc1) + (acc2 + acc3);
    if (acc == 123456789) out[0] = (float)acc;
}

// value: TFLOP/s (fp32_tflops) or GB/s (l2_gbs, smem_gbs); best of 5 timed launches after a warm-up
int measure_peak(hb_system *h, const char *which, double *value)
{
    cudaStream_t st = h->stream;
    cudaEvent_t e0, e1;
    HB_CK(cudaEventCreate(&e0));
    HB_CK(cudaEventCreate(&e1));
    float *out = nullptr;
    float4 *buf = nullptr;
    const int64_t n4 = (32 << 20) / 16;
    int rc = HB_OK;
    cudaError_t e = cudaMalloc((void **)&out, 256);
    const int mode = !strcmp(which, "fp32_tflops") ? 0 : !strcmp(which, "l2_gbs") ? 1 : !strcmp(which, "smem_gbs") ? 2 : -1;
    if (mode < 0) { h->err = std::string("unknown peak ") + which; rc = HB_EINVAL; }
    if (rc == HB_OK && e == cudaSuccess && mode == 1) {
        e = cudaMalloc((void **)&buf, (size_t)n4 * 16);
        if (e == cudaSuccess) e = cudaMemsetAsync(buf, 0, (size_t)n4 * 16, st);
    }
    const int grid = h->sm_count * 8;       // 2048 threads per SM
    const int iters = 2048, passes = 100;
    double best = 0.0;
    for (int rep = 0; rep < 6 && rc == HB_OK && e == cudaSuccess; rep++) {
        cudaEventRecord(e0, st);
        double work = 0.0;
        if (mode == 0) {
            peak_fma_kernel<<<grid, PK_THREADS, 0, st>>>(out, 1.0000001f, 1e-7f, iters);
            work = (double)grid * PK_THREADS * iters * 64.0 * 2.0 / 1e12;           // TFLOP
        } else if (mode == 1) {
            peak_l2_kernel<<<grid, PK_THREADS, 0, st>>>(buf, n4, passes, out);
            work = (double)n4 * 16.0 * passes / 1e9;                                  // GB
        } else {
            peak_smem_kernel<<<grid, PK_THREADS, 0, st>>>(out, iters, PK_THREADS);
            work = (double)grid * PK_THREADS * iters * 8.0 * 16.0 / 1e9;              // GB
        }
        cudaEventRecord(e1, st);
        e = cudaStreamSynchronize(st);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess && rep > 0 && ms > 0.f) best = std::max(best, work / (ms * 1e-3));
    }
    if (rc == HB_OK && e != cudaSuccess) { h->err = std::string("hb_measure_peak: ") + cudaGetErrorString(e); rc = HB_ECUDA; }
    cudaFree(out);
    cudaFree(buf);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (rc == HB_OK) *value = best;
    return rc;
}
