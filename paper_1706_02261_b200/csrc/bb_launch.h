// bb_launch.h -- host-side entry points of the per-shape kernel instantiations (bb_inst.cu is
// compiled once per TX = Nx/32; each object holds the kernels for every TY = Ny/32).
#pragma once
#include "bb_kernels.cuh"

namespace bb {

// One set per TX in {1, 2, 4, 8, 16, 32}.
#define BB_DECLARE_INST(TX)                                                                     \
    cudaError_t inst##TX##_prepare(int TY);                                                     \
    int inst##TX##_blocks_per_sm(int TY);                                                       \
    cudaError_t inst##TX##_launch(int TY, const KParams &P, int grid, bool coop, cudaStream_t s);
BB_DECLARE_INST(1)
BB_DECLARE_INST(2)
BB_DECLARE_INST(4)
BB_DECLARE_INST(8)
BB_DECLARE_INST(16)
BB_DECLARE_INST(32)
#undef BB_DECLARE_INST

// 16-point-thread kernel (bb_kernels16.cuh), one set per PX = Nx/256 in {1, 2, 4, 8} and column
// tile width in {4, 8}; bb_inst16.cu.
#define BB_DECLARE_INST16(PX, CW, BT)                                                                              \
    cudaError_t inst16_##PX##_cw##CW##_b##BT##_prepare(int PY);                                                     \
    int inst16_##PX##_cw##CW##_b##BT##_blocks_per_sm(int PY);                                                       \
    cudaError_t inst16_##PX##_cw##CW##_b##BT##_launch(int PY, const KParams &P, int grid, bool coop, cudaStream_t s);
BB_DECLARE_INST16(1, 4, 0) BB_DECLARE_INST16(2, 4, 0) BB_DECLARE_INST16(4, 4, 0) BB_DECLARE_INST16(8, 4, 0)
BB_DECLARE_INST16(1, 8, 0) BB_DECLARE_INST16(2, 8, 0) BB_DECLARE_INST16(4, 8, 0) BB_DECLARE_INST16(8, 8, 0)
BB_DECLARE_INST16(1, 4, 1) BB_DECLARE_INST16(2, 4, 1) BB_DECLARE_INST16(4, 4, 1) BB_DECLARE_INST16(8, 4, 1)
BB_DECLARE_INST16(1, 8, 1) BB_DECLARE_INST16(2, 8, 1) BB_DECLARE_INST16(4, 8, 1) BB_DECLARE_INST16(8, 8, 1)
#undef BB_DECLARE_INST16

// 8-point-thread kernel (bb_kernels8.cuh), one set per PX = Nx/256 in {1, 2, 4, 8} and column tile width in
// {4, 8}; bb_inst8.cu.
#define BB_DECLARE_INST8(PX, CW, BT)                                                                              \
    cudaError_t inst8_##PX##_cw##CW##_b##BT##_prepare(int PY);                                                     \
    int inst8_##PX##_cw##CW##_b##BT##_blocks_per_sm(int PY);                                                       \
    cudaError_t inst8_##PX##_cw##CW##_b##BT##_launch(int PY, const KParams &P, int grid, bool coop, cudaStream_t s);
BB_DECLARE_INST8(1, 4, 0) BB_DECLARE_INST8(2, 4, 0) BB_DECLARE_INST8(4, 4, 0) BB_DECLARE_INST8(8, 4, 0)
BB_DECLARE_INST8(1, 8, 0) BB_DECLARE_INST8(2, 8, 0) BB_DECLARE_INST8(4, 8, 0) BB_DECLARE_INST8(8, 8, 0)
BB_DECLARE_INST8(1, 4, 1) BB_DECLARE_INST8(2, 4, 1) BB_DECLARE_INST8(4, 4, 1) BB_DECLARE_INST8(8, 4, 1)
BB_DECLARE_INST8(1, 8, 1) BB_DECLARE_INST8(2, 8, 1) BB_DECLARE_INST8(4, 8, 1) BB_DECLARE_INST8(8, 8, 1)
#undef BB_DECLARE_INST8

// Dispatch on (Nx, Ny); defined in bb_api.cu.
int kernel_prepare(int Nx, int Ny);           // returns a cudaError_t value
int kernel_blocks_per_sm(int Nx, int Ny);
cudaError_t kernel_launch(int Nx, int Ny, const KParams &P, int grid, bool coop, cudaStream_t s);
bool kernel16_supports(int Nx, int Ny);
int kernel16_prepare(int Nx, int Ny);
int kernel16_blocks_per_sm(int Nx, int Ny);
cudaError_t kernel16_launch(int Nx, int Ny, const KParams &P, int grid, bool coop, cudaStream_t s);
bool kernel8_supports(int Nx, int Ny);
int kernel8_prepare(int Nx, int Ny);
int kernel8_blocks_per_sm(int Nx, int Ny);
cudaError_t kernel8_launch(int Nx, int Ny, const KParams &P, int grid, bool coop, cudaStream_t s);

// Cluster kernel for small grids (bb_kernelsc.cuh; bb_instc.cu): one cluster of `cs` CTAs per field.
bool kernelc_supports(int Nx, int Ny);
int kernelc_prepare(int Nx, int Ny, int cs, int mode, int pt);        // returns a cudaError_t value
int kernelc_max_clusters(int Nx, int Ny, int cs, int mode, int pt);   // clusters the device holds at once; 0: cannot be scheduled
cudaError_t kernelc_launch(int Nx, int Ny, int cs, int mode, int pt, const KParams &P, int nclusters, cudaStream_t s);

}  // namespace bb
