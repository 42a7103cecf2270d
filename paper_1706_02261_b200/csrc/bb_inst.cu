// bb_inst.cu -- instantiates bpm_kernel<TX, TY, 8> for one TX (= -DBB_TX) and every TY.
#include "bb_launch.h"

#ifndef BB_TX
#error "compile with -DBB_TX=<Nx/32>"
#endif

namespace bb {
namespace {

constexpr int kCW = 8;   // columns per tile: 64-byte row segments

template <int TY>
cudaError_t prepare_t() {
    return cudaFuncSetAttribute(bpm_kernel<BB_TX, TY, kCW>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)SmemLayout<BB_TX, TY, kCW>::bytes);
}
template <int TY>
int blocks_t() {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, bpm_kernel<BB_TX, TY, kCW>, kThreads,
                                                      SmemLayout<BB_TX, TY, kCW>::bytes) != cudaSuccess)
        return 0;
    return n;
}
template <int TY>
cudaError_t launch_t(const KParams &P, int grid, bool coop, cudaStream_t s) {
    constexpr size_t smem = SmemLayout<BB_TX, TY, kCW>::bytes;
    if (coop) {
        void *args[] = {(void *)&P};
        return cudaLaunchCooperativeKernel((const void *)bpm_kernel<BB_TX, TY, kCW>, dim3(grid), dim3(kThreads),
                                           args, smem, s);
    }
    bpm_kernel<BB_TX, TY, kCW><<<grid, kThreads, smem, s>>>(P);
    return cudaGetLastError();
}

}  // namespace

#define BB_CAT2(a, b, c) a##b##c
#define BB_CAT(a, b, c) BB_CAT2(a, b, c)
#define BB_SWITCH_TY(expr_prefix, ...)            \
    switch (TY) {                                 \
        case 1: return expr_prefix<1>(__VA_ARGS__);  \
        case 2: return expr_prefix<2>(__VA_ARGS__);  \
        case 4: return expr_prefix<4>(__VA_ARGS__);  \
        case 8: return expr_prefix<8>(__VA_ARGS__);  \
        case 16: return expr_prefix<16>(__VA_ARGS__); \
        case 32: return expr_prefix<32>(__VA_ARGS__); \
    }

cudaError_t BB_CAT(inst, BB_TX, _prepare)(int TY) {
    BB_SWITCH_TY(prepare_t)
    return cudaErrorInvalidValue;
}
int BB_CAT(inst, BB_TX, _blocks_per_sm)(int TY) {
    BB_SWITCH_TY(blocks_t)
    return 0;
}
cudaError_t BB_CAT(inst, BB_TX, _launch)(int TY, const KParams &P, int grid, bool coop, cudaStream_t s) {
    BB_SWITCH_TY(launch_t, P, grid, coop, s)
    return cudaErrorInvalidValue;
}

}  // namespace bb
