// bb_instc.cu -- instantiates the cluster kernel bpmc_kernel<NX, NY, CS, MODE, PT> (bb_kernelsc.cuh) for
// Nx, Ny in {128, 256} and clusters of 8 and 16 CTAs, and launches it with the cluster attribute.
#include "bb_launch.h"
#include "bb_kernelsc.cuh"

namespace bb {
namespace {

template <int NX, int NY, int CS, int ST, int PT>
cudaError_t prepare_c() {
    if constexpr (SmemC<NX, NY, CS, PT>::fits) {
        auto *k = bpmc_kernel<NX, NY, CS, ST, PT>;
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SmemC<NX, NY, CS, PT>::bytes);
        if (e != cudaSuccess) return e;
        if (CS > 8) e = cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        return e;
    } else {
        return cudaErrorInvalidValue;
    }
}

template <int NX, int NY, int CS, int PT>
void fill_config(cudaLaunchConfig_t &cfg, cudaLaunchAttribute &attr, int nclusters, cudaStream_t s) {
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = dim3(CS * nclusters);
    cfg.blockDim = dim3(SmemC<NX, NY, CS, PT>::NT);
    cfg.dynamicSmemBytes = SmemC<NX, NY, CS, PT>::bytes;
    cfg.stream = s;
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = CS;
    attr.val.clusterDim.y = 1;
    attr.val.clusterDim.z = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
}

// how many clusters the device can hold at once (0: this cluster size cannot be scheduled)
template <int NX, int NY, int CS, int ST, int PT>
int clusters_c() {
    if constexpr (SmemC<NX, NY, CS, PT>::fits) {
        cudaLaunchConfig_t cfg;
        cudaLaunchAttribute attr;
        fill_config<NX, NY, CS, PT>(cfg, attr, 1, nullptr);
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, bpmc_kernel<NX, NY, CS, ST, PT>, &cfg) != cudaSuccess) {
            (void)cudaGetLastError();
            return 0;
        }
        return n;
    } else {
        return 0;
    }
}

template <int NX, int NY, int CS, int ST, int PT>
cudaError_t launch_c(const KParams &P, int nclusters, cudaStream_t s) {
    if constexpr (SmemC<NX, NY, CS, PT>::fits) {
        cudaLaunchConfig_t cfg;
        cudaLaunchAttribute attr;
        fill_config<NX, NY, CS, PT>(cfg, attr, nclusters, s);
        return cudaLaunchKernelEx(&cfg, bpmc_kernel<NX, NY, CS, ST, PT>, P);
    } else {
        return cudaErrorInvalidValue;
    }
}

// (shape, cluster size, exchange mode, points per thread): 16-point threads exist for 256 x 256 on 16 CTAs only
#define BB_C_SHAPE(fn, NXv, NYv, ...)                                                                                   \
    if (Nx == NXv && Ny == NYv && pt == 8) {                                                                            \
        if (cs == 16) return mode == 1 ? fn<NXv, NYv, 16, 1, 8>(__VA_ARGS__) : fn<NXv, NYv, 16, 0, 8>(__VA_ARGS__);     \
        if (cs == 8) return mode == 1 ? fn<NXv, NYv, 8, 1, 8>(__VA_ARGS__) : fn<NXv, NYv, 8, 0, 8>(__VA_ARGS__);        \
    }
#define BB_C_DISPATCH(fn, ...)                                                                                          \
    BB_C_SHAPE(fn, 128, 128, __VA_ARGS__)                                                                               \
    BB_C_SHAPE(fn, 256, 128, __VA_ARGS__)                                                                               \
    BB_C_SHAPE(fn, 128, 256, __VA_ARGS__)                                                                               \
    BB_C_SHAPE(fn, 256, 256, __VA_ARGS__)                                                                               \
    if (Nx == 256 && Ny == 256 && pt == 16 && cs == 16)                                                                 \
        return mode == 1 ? fn<256, 256, 16, 1, 16>(__VA_ARGS__) : fn<256, 256, 16, 0, 16>(__VA_ARGS__);

}  // namespace

bool kernelc_supports(int Nx, int Ny) { return (Nx == 128 || Nx == 256) && (Ny == 128 || Ny == 256); }

int kernelc_prepare(int Nx, int Ny, int cs, int mode, int pt) {
    BB_C_DISPATCH(prepare_c)
    return (int)cudaErrorInvalidValue;
}
int kernelc_max_clusters(int Nx, int Ny, int cs, int mode, int pt) {
    BB_C_DISPATCH(clusters_c)
    return 0;
}
cudaError_t kernelc_launch(int Nx, int Ny, int cs, int mode, int pt, const KParams &P, int nclusters, cudaStream_t s) {
    BB_C_DISPATCH(launch_c, P, nclusters, s)
    return cudaErrorInvalidValue;
}

}  // namespace bb
