// bb_probe.cu -- device micro-benchmarks for the roofline denominators that
// MEASURED_PEAKS.json does not hold: L2 bandwidth over a resident buffer
// and the FP32 rates of the scalar (FFMA) and packed (FFMA2, sm_100) pipes.  Measurement
// support only; nothing on the BPM path calls these.
#include "../../include/bb.h"
#include "bb_fft16.cuh"
#include <cuda_runtime.h>

namespace {

// The arithmetic of one phase of the 16-point-thread kernel on a 1024-point line, per thread (16 points), with
// every operand in registers and no memory access at all: forward line transform (radix-16, 15 twiddles,
// radix-16, radix-4 class butterflies, 12 class twiddles), 16 pointwise multiplies, inverse transform --
// the library's own butterflies (packed FADD2 / FFMA2).  512 threads per CTA, one CTA per SM: the occupancy
// of bpm16_kernel.  What it reaches, in the flop count of SURVEY 8d (120 per point and phase at 1024^2), is
// the ceiling of this instruction mix: most of a butterfly is additions, which earn one flop per lane where
// the nominal peak counts two.
__global__ void __launch_bounds__(512, 1) butterfly_mix_kernel(float *__restrict__ sink, int iters) {
    using bb::cf;
    cf v[16], tw[15], ct[3];
    const float a = 1e-3f * (float)(threadIdx.x + 1);
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = make_float2(a + i, a - i);
#pragma unroll
    for (int i = 0; i < 15; ++i) { float s, c; __sincosf(a * (i + 1), &s, &c); tw[i] = make_float2(c, s); }
#pragma unroll
    for (int i = 0; i < 3; ++i) { float s, c; __sincosf(-a * (i + 1), &s, &c); ct[i] = make_float2(c, s); }
    const cf pw = make_float2(9.765625e-4f * tw[0].x, 9.765625e-4f * tw[0].y);      // 2^-10: keeps the values finite
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            bb::Dft<16, -1>::run(v);
#pragma unroll
            for (int k = 1; k < 16; ++k) v[k] = half ? bb::cmulc(v[k], tw[k - 1]) : bb::cmul(v[k], tw[k - 1]);
            bb::Dft<16, -1>::run(v);
#pragma unroll
            for (int g = 0; g < 4; ++g) {
#pragma unroll
                for (int c = 1; c < 4; ++c) v[4 * g + c] = bb::cmul(v[4 * g + c], ct[c - 1]);
                bb::class_dft<4, -1>(v + 4 * g);
            }
            if (half == 0) {
#pragma unroll
                for (int i = 0; i < 16; ++i) v[i] = bb::cmul(v[i], pw);
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += v[i].x + v[i].y;
    if (s == 123.456f) sink[0] = s;
}

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
// packed 2: the butterfly mix of a 1024-point phase from registers (butterfly_mix_kernel), in SURVEY 8d's flop count.
int bb_probe_fp32(int iters, int packed, double *tflops) {
    if (!tflops || iters < 1 || packed < 0 || packed > 2) return BB_ERR_INVALID_ARG;
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
    const int grid = packed == 2 ? sms : sms * 8, block = packed == 2 ? 512 : 256;
    for (int rep = 0; rep < 2; ++rep) {
        cudaEventRecord(e0);
        if (packed == 2) butterfly_mix_kernel<<<grid, block>>>(sink, iters);
        else if (packed) fma_kernel<1><<<grid, block>>>(sink, iters, 1.0000001f, 1e-9f);
        else fma_kernel<0><<<grid, block>>>(sink, iters, 1.0000001f, 1e-9f);
        cudaEventRecord(e1);
        rc = timed(e0, e1, &ms);
    }
    // mix: 16 points x 120 flop per point and phase ((10 (log2 Nx + log2 Ny) + 40) / 2 at 1024^2)
    double flop = (packed == 2 ? 16.0 * 120.0 : 2.0 * 16.0) * (double)iters * (double)grid * block;
    *tflops = flop / (ms * 1e-3) / 1e12;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    return cudaGetLastError() == cudaSuccess ? rc : BB_ERR_CUDA;
}

}  // extern "C"
