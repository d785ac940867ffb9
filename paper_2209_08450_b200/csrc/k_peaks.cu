// k_peaks.cu -- issue-rate micro-benchmarks behind tcp_measure_rates: the denominators bench.py uses for the
// arithmetic roofs of this GPU are MEASURED here, at the clocks of the moment, instead of derived from unit counts:
//   fp32: 16 independent FFMA chains per thread, 8 CTAs of 256 threads per SM;
//   hmma: 8 independent mma.sync.m16n8k16 (fp16 in, fp32 accumulate) chains per warp, the instruction the
//         tensor-core transforms of mmafft.cuh are built on.
#include <stdint.h>

#include <algorithm>

#include "tcp_internal.h"

namespace tcpk {

__global__ void __launch_bounds__(256) peak_ffma_kernel(float* out, int iters) {
    float c[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = (float)i;
    const float a = 1.f + 1e-6f * (float)threadIdx.x, b = 0.5f;
    for (int it = 0; it < iters; ++it)
#pragma unroll
        for (int i = 0; i < 16; ++i) c[i] = fmaf(c[i], a, b);
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i];
    if (s == 123.456f) out[0] = s;                     // keeps the chains alive; never true in practice
}

__global__ void __launch_bounds__(256) peak_hmma_kernel(float* out, int iters) {
    float c[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) c[i][j] = 0.f;
    const uint32_t a0 = threadIdx.x, a1 = threadIdx.x * 3u, a2 = 7u, a3 = 9u, b0 = 0x3c003c00u, b1 = 0x3c003c00u;
    for (int it = 0; it < iters; ++it)
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                         : "+f"(c[i][0]), "+f"(c[i][1]), "+f"(c[i][2]), "+f"(c[i][3])
                         : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) s += c[i][j];
    if (s == 123.456f) out[0] = s;
}

}  // namespace tcpk

using namespace tcpk;

extern "C" int tcp_measure_rates(double* fp32_tflops, double* hmma_tflops) {
    if (!fp32_tflops || !hmma_tflops) return set_error(TCP_EINVAL, "NULL argument");
    int dev = 0, nsm = 0;
    TCP_CUDA_CHECK(cudaGetDevice(&dev));
    TCP_CUDA_CHECK(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    float* out = nullptr;
    TCP_CUDA_CHECK(cudaMalloc((void**)&out, 4));
    cudaEvent_t e0, e1;
    TCP_CUDA_CHECK(cudaEventCreate(&e0));
    TCP_CUDA_CHECK(cudaEventCreate(&e1));
    const int iters = 8192, ctas = nsm * 8;
    double best[2] = {0.0, 0.0};
    for (int rep = 0; rep < 4; ++rep)               // first repetition warms up; best of the others
        for (int which = 0; which < 2; ++which) {
            cudaEventRecord(e0, 0);
            if (which == 0) peak_ffma_kernel<<<ctas, 256>>>(out, iters);
            else peak_hmma_kernel<<<ctas, 256>>>(out, iters);
            cudaEventRecord(e1, 0);
            cudaEventSynchronize(e1);
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            const double flop = which == 0 ? (double)ctas * 256.0 * iters * 16.0 * 2.0 : (double)ctas * 8.0 * iters * 8.0 * 4096.0;
            if (rep > 0 && ms > 0.f) best[which] = std::max(best[which], flop / (ms * 1e-3) / 1e12);
        }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    TCP_CUDA_CHECK(cudaGetLastError());
    *fp32_tflops = best[0];
    *hmma_tflops = best[1];
    return TCP_OK;
}
