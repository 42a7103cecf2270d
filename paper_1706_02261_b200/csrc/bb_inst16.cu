// bb_inst16.cu -- instantiates bpm16_kernel<PX, PY, CW> for one PX (= -DBB_PX), one column tile width
// CW (= -DBB_CW), single-field or batch (= -DBB_BATCH) and every PY.
#include "bb_launch.h"
#include "bb_kernels16.cuh"

#if !defined(BB_PX) || !defined(BB_CW) || !defined(BB_BATCH)
#error "compile with -DBB_PX=<Nx/256> -DBB_CW=<columns per column tile: 4 or 8> -DBB_BATCH=<0 or 1>"
#endif

namespace bb {
namespace {

// a tile of 8 columns of a 2048-row grid would need a team of 1024 threads: such grids use tiles of 4
template <int PY> constexpr bool valid16() { return 16 * PY * BB_CW <= kThreads16; }

template <int PY>
cudaError_t prepare_t() {
    if constexpr (valid16<PY>())
        return cudaFuncSetAttribute(bpm16_kernel<BB_PX, PY, BB_CW, BB_BATCH != 0>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)Smem16<BB_PX, PY>::bytes);
    else
        return cudaSuccess;
}
template <int PY>
int blocks_t() {
    int n = 1;
    if constexpr (valid16<PY>()) {
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, bpm16_kernel<BB_PX, PY, BB_CW, BB_BATCH != 0>, kThreads16,
                                                          Smem16<BB_PX, PY>::bytes) != cudaSuccess)
            return 0;
    }
    return n;
}
template <int PY>
cudaError_t launch_t(const KParams &P, int grid, bool coop, cudaStream_t s) {
    if constexpr (valid16<PY>()) {
        constexpr size_t smem = Smem16<BB_PX, PY>::bytes;
        if (coop) {
            void *args[] = {(void *)&P};
            return cudaLaunchCooperativeKernel((const void *)bpm16_kernel<BB_PX, PY, BB_CW, BB_BATCH != 0>, dim3(grid), dim3(kThreads16),
                                               args, smem, s);
        }
        bpm16_kernel<BB_PX, PY, BB_CW, BB_BATCH != 0><<<grid, kThreads16, smem, s>>>(P);
        return cudaGetLastError();
    } else {
        return cudaErrorInvalidValue;
    }
}

}  // namespace

#define BB_CAT2(a, b, c, d, e, f, g) a##b##c##d##e##f##g
#define BB_CAT(a, b, c, d, e, f, g) BB_CAT2(a, b, c, d, e, f, g)
#define BB_SWITCH_PY(expr_prefix, ...)               \
    switch (PY) {                                    \
        case 1: return expr_prefix<1>(__VA_ARGS__);  \
        case 2: return expr_prefix<2>(__VA_ARGS__);  \
        case 4: return expr_prefix<4>(__VA_ARGS__);  \
        case 8: return expr_prefix<8>(__VA_ARGS__);  \
    }

cudaError_t BB_CAT(inst16_, BB_PX, _cw, BB_CW, _b, BB_BATCH, _prepare)(int PY) {
    BB_SWITCH_PY(prepare_t)
    return cudaErrorInvalidValue;
}
int BB_CAT(inst16_, BB_PX, _cw, BB_CW, _b, BB_BATCH, _blocks_per_sm)(int PY) {
    BB_SWITCH_PY(blocks_t)
    return 0;
}
cudaError_t BB_CAT(inst16_, BB_PX, _cw, BB_CW, _b, BB_BATCH, _launch)(int PY, const KParams &P, int grid, bool coop, cudaStream_t s) {
    BB_SWITCH_PY(launch_t, P, grid, coop, s)
    return cudaErrorInvalidValue;
}

}  // namespace bb
