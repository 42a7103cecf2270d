// bb_noalloc.cu -- bb_nref_from_dn_static (include/bb.h): the locally adapted reference index n_ref[j]
// (reading A3) computed without a single allocation, on the device or on the host.
//
// Who this is for.  bb_nref_from_dn keeps its per-slice partial sums in a workspace that it grows with
// cudaFree + cudaMalloc, and it copies them to a std::vector.  Two kinds of users of this library
// cannot live with that:
//   * a pipeline that computes n_ref of the NEXT sample volume while a propagation of the current one
//     is running on another stream: cudaMalloc and cudaFree wait for the whole device, so the
//     allocation stalls the propagation it was meant to overlap with;
//   * a process whose framework allocator already holds nearly all of the 180 GB (a 1024 x 2048 x 1024
//     volume with its intensity stack and a batch of fields is most of it): a raw cudaMalloc from
//     inside the library can then fail although the caller has memory of its own to give.
// Here the partial sums live in a file-scope __device__ array of fixed size instead.  The price: every
// CUDA context that loads this library carries the array (512 KiB) until the process exits, and the
// volume depth is capped at BB_STATIC_MAX_NZ slices.
//
// The arithmetic is the one of bb_nref_from_dn: slice_sum_static_kernel is slice_sum_kernel
// (bb_aux_kernels.cuh) with the same grid and summation order; the slab means, which that entry point
// forms on the host, are formed here by slab_mean_kernel in the same order with a compensated
// (two-double) sum, so both entry points agree to the last float32 bit except on a rounding tie.
#include "../../include/bb.h"
#include "bb_hooks.h"

#include <cuda_runtime.h>
#include <cstdio>
#include <mutex>

namespace {

constexpr int kParts = 16;                           // partial sums per slice, as in bb_nref_from_dn
constexpr int kMaxDevices = 64;

// The scratch.  In HOST code this name is only a handle for the runtime's symbol table, not a device
// address: the address a kernel may use comes from cudaGetSymbolAddress (static_scratch below).
static __device__ __align__(256) double g_nref_partial[(size_t)BB_STATIC_MAX_NZ * kParts];

// partial[j][b] = sum of the b-th of gridDim.x contiguous pieces of slice j, in double, fixed order.
__global__ void __launch_bounds__(256) slice_sum_static_kernel(const float *__restrict__ dn, size_t npx,
                                                               double *__restrict__ partial) {
    __shared__ double sm[256];
    const float *p = dn + (size_t)blockIdx.y * npx;
    const size_t chunk = (npx + gridDim.x - 1) / gridDim.x;
    const size_t i0 = (size_t)blockIdx.x * chunk, i1 = i0 + chunk < npx ? i0 + chunk : npx;
    double s = 0.0;
    for (size_t i = i0 + threadIdx.x; i < i1; i += blockDim.x) s += (double)p[i];
    sm[threadIdx.x] = s;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w) sm[threadIdx.x] += sm[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = sm[0];
}

// One thread per slab: n_ref = float(n0 + mean of dn over the slab), written to every slice of the slab.
// The slab sum is carried as hi + lo (Knuth's two-sum), which holds more bits than the host's long double.
__global__ void slab_mean_kernel(const double *__restrict__ partial, size_t npx, int Nz, int slab, double n0,
                                 float *__restrict__ nref_out) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long j0 = t * slab;
    if (j0 >= Nz) return;
    const int j1 = (int)(j0 + slab < Nz ? j0 + slab : Nz);
    double hi = 0.0, lo = 0.0;
    for (int j = (int)j0; j < j1; ++j) {
        double sj = 0.0;
        for (int q = 0; q < kParts; ++q) sj = __dadd_rn(sj, partial[(size_t)j * kParts + q]);
        const double s = __dadd_rn(hi, sj);
        const double bv = __dsub_rn(s, hi);
        const double err = __dadd_rn(__dsub_rn(hi, __dsub_rn(s, bv)), __dsub_rn(sj, bv));
        hi = s;
        lo = __dadd_rn(lo, err);
    }
    const double denom = __dmul_rn((double)npx, (double)(j1 - (int)j0));      // exact: < 2^53
    const double mean = __ddiv_rn(__dadd_rn(hi, lo), denom);
    const float v = (float)__dadd_rn(n0, mean);
    for (int j = (int)j0; j < j1; ++j) nref_out[j] = v;
}

std::mutex g_setup_mu;
double *g_scratch_addr[kMaxDevices] = {};            // device address of g_nref_partial, per device ordinal

// Set-up, once per device, with that device current: ask the runtime where this device's copy of the
// array lives.  (Passing g_nref_partial itself to a kernel from host code would hand it the host-side
// handle.)  cudaGetSymbolAddress allocates nothing: the array came with the module.
int static_scratch(int dev, double **out) {
    std::lock_guard<std::mutex> lk(g_setup_mu);
    if (!g_scratch_addr[dev]) {
        double *ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_nref_partial);
        if (e != cudaSuccess || !ptr) {
            char msg[256];
            snprintf(msg, sizeof msg, "cudaGetSymbolAddress(g_nref_partial) failed on device %d: %s", dev,
                     cudaGetErrorString(e));
            return bb::report_error(BB_ERR_CUDA, msg);
        }
        g_scratch_addr[dev] = ptr;
    }
    *out = g_scratch_addr[dev];
    return BB_OK;
}

}  // namespace

extern "C" {

int bb_static_max_nz(void) { return BB_STATIC_MAX_NZ; }

int bb_nref_from_dn_static(const float *dn, int Nx, int Ny, int Nz, float n0, int slab, float *nref_out,
                           void *stream) {
    if (!dn || !nref_out) return bb::report_error(BB_ERR_INVALID_ARG, "dn_volume or nref_out is NULL");
    if (Nx < 1 || Ny < 1 || Nz < 1 || slab < 1) return bb::report_error(BB_ERR_INVALID_ARG, "Nx, Ny, Nz, slab must be >= 1");
    if (Nz > BB_STATIC_MAX_NZ) {
        char msg[256];
        snprintf(msg, sizeof msg,
                 "bb_nref_from_dn_static: Nz = %d exceeds the static scratch (BB_STATIC_MAX_NZ = %d slices); "
                 "split the volume or call bb_nref_from_dn", Nz, BB_STATIC_MAX_NZ);
        return bb::report_error(BB_ERR_INVALID_ARG, msg);
    }
    int dev = 0, major = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) {
        char msg[256];
        snprintf(msg, sizeof msg, "no usable CUDA device: %s", cudaGetErrorString(e));
        return bb::report_error(BB_ERR_CUDA, msg);
    }
    if (major != 10) return bb::report_error(BB_ERR_ARCH, "this library is sm_100a only");
    if (dev >= kMaxDevices) return bb::report_error(BB_ERR_INVALID_ARG, "device ordinal beyond the static table (64)");
    double *partial = nullptr;
    int rc = static_scratch(dev, &partial);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t npx = (size_t)Nx * Ny;
    // Every partial sum the second kernel reads (j < Nz, all kParts of it) is written by the first one in
    // this same call, so what an earlier call left in the array is never seen and nothing needs clearing.
    slice_sum_static_kernel<<<dim3(kParts, Nz), 256, 0, s>>>(dn, npx, partial);
    const int nslabs = (Nz + slab - 1) / slab;
    slab_mean_kernel<<<(nslabs + 127) / 128, 128, 0, s>>>(partial, npx, Nz, slab, (double)n0, nref_out);
    bb::count_launches(2);
    e = cudaGetLastError();
    if (e != cudaSuccess) {
        char msg[256];
        snprintf(msg, sizeof msg, "bb_nref_from_dn_static: launch failed: %s", cudaGetErrorString(e));
        return bb::report_error(BB_ERR_CUDA, msg);
    }
    return BB_OK;
}

}  // extern "C"
