// bb_probe.cu -- device micro-benchmarks for the roofline denominators that
// MEASURED_PEAKS.json does not hold: L2 bandwidth over a resident buffer
// and the FP32 rates of the scalar (FFMA) and packed (FFMA2, sm_100) pipes.  Measurement
// support only; nothing on the BPM path calls these.
#include "../../include/bb.h"
#include <cuda_runtime.h>

namespace {

__global__ void l2_copy_kernel(const float4 *__restrict__ src, float4 *__restrict__ dst, size_t n, int iters) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int it = 0; it < iters; ++it)
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
            __stcg(dst + i, __ldcg(src + i));
}

__global__ void l2_read_kernel(const float4 *__restrict__ src, float *__restrict__ sink, size_t n, int iters) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    float acc = 0.f;
    for (int it = 0; it < iters; ++it)
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
            float4 v = __ldcg(src + i);
            acc += v.x + v.y + v.z + v.w;
        }
    if (acc == 123.456f) sink[0] = acc;
}

template <int PACKED>
__global__ void fma_kernel(float *__restrict__ sink, int iters, float a, float b) {
    float2 x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = make_float2(threadIdx.x * 1e-3f + i, blockIdx.x * 1e-3f - i);
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (PACKED) {
                unsigned long long xi = *reinterpret_cast<unsigned long long *>(&x[i]);
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(xi)
                             : "l"(*reinterpret_cast<const unsigned long long *>(&a2)),
                               "l"(*reinterpret_cast<const unsigned long long *>(&b2)));
                x[i] = *reinterpret_cast<float2 *>(&xi);
            } else {
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[i].x) : "f"(a), "f"(b));
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[i].y) : "f"(a), "f"(b));
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i].x + x[i].y;
    if (s == 123.456f) sink[0] = s;
}

int timed(cudaEvent_t e0, cudaEvent_t e1, float *ms) {
    if (cudaEventSynchronize(e1) != cudaSuccess) return BB_ERR_CUDA;
    if (cudaEventElapsedTime(ms, e0, e1) != cudaSuccess) return BB_ERR_CUDA;
    return BB_OK;
}

}  // namespace

extern "C" {

// mode 0: copy (read + write), mode 1: read only.  bytes = size of the resident working set.
int bb_probe_l2_bandwidth(unsigned long long bytes, int iters, int mode, double *gb_per_s) {
    if (!gb_per_s || bytes < (1u << 20) || iters < 1) return BB_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return BB_ERR_CUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    void *buf = nullptr;
    float *sink = nullptr;
    if (cudaMalloc(&buf, bytes) != cudaSuccess) return BB_ERR_OOM;
    if (cudaMalloc(&sink, 256) != cudaSuccess) { cudaFree(buf); return BB_ERR_OOM; }
    cudaMemset(buf, 0, bytes);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const size_t n4 = bytes / 16;
    float ms = 0.f;
    int rc = BB_OK;
    for (int rep = 0; rep < 2; ++rep) {        // first pass warms L2
        cudaEventRecord(e0);
        if (mode == 0)
            l2_copy_kernel<<<sms * 4, 512>>>((const float4 *)buf, (float4 *)buf + n4 / 2, n4 / 2, iters);
        else
            l2_read_kernel<<<sms * 4, 512>>>((const float4 *)buf, sink, n4, iters);
        cudaEventRecord(e1);
        rc = timed(e0, e1, &ms);
    }
    double moved = (double)(n4 * 16) * iters;   // copy: half read + half written = the whole buffer once per iteration
    *gb_per_s = moved / (ms * 1e-3) / 1e9;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    cudaFree(sink);
    return cudaGetLastError() == cudaSuccess ? rc : BB_ERR_CUDA;
}

// packed 0: scalar FFMA, 1: FFMA2 (fma.rn.f32x2).  Result in TFLOP/s (2 flop per fused multiply-add lane).
int bb_probe_fp32(int iters, int packed, double *tflops) {
    if (!tflops || iters < 1) return BB_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return BB_ERR_CUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    float *sink = nullptr;
    if (cudaMalloc(&sink, 256) != cudaSuccess) return BB_ERR_OOM;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float ms = 0.f;
    int rc = BB_OK;
    const int grid = sms * 8, block = 256;
    for (int rep = 0; rep < 2; ++rep) {
        cudaEventRecord(e0);
        if (packed) fma_kernel<1><<<grid, block>>>(sink, iters, 1.0000001f, 1e-9f);
        else fma_kernel<0><<<grid, block>>>(sink, iters, 1.0000001f, 1e-9f);
        cudaEventRecord(e1);
        rc = timed(e0, e1, &ms);
    }
    double flop = 2.0 * 16.0 * (double)iters * (double)grid * block;
    *tflops = flop / (ms * 1e-3) / 1e12;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    return cudaGetLastError() == cudaSuccess ? rc : BB_ERR_CUDA;
}

}  // extern "C"
