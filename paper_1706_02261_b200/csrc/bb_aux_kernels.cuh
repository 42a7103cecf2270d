// bb_aux_kernels.cuh -- kernels off the per-slice loop: propagator table (fp64), multiplexed
// point-source spectrum, per-slice sums of dn for the adapted reference index.
#pragma once
#include <cuda_runtime.h>

namespace bb {

// DFT bin -> signed frequency index (bb.h: kx[p] = 2 pi (p < N/2 ? p : p - N) / (N d)).
__device__ __forceinline__ int freq_index(int p, int n) { return (p < n / 2) ? p : p - n; }

// H[q][p] = (s > 0) ? exp(i dz sqrt(s)) * inv_norm : 0,  s = k^2 - kx^2 - ky^2   (bb.h; reading A2).
// Everything in double, no fused multiply-adds in s (the cut-off test is a decision).
// perm > 1: column p holds DFT bin perm * (p mod Nx/perm) + p / (Nx/perm), the kx-class-major order in
// which the 16-point-thread kernel keeps the field between its phases (bb_kernels16.cuh).
__global__ void propagator_table_kernel(float2 *__restrict__ H, int Nx, int Ny, double dx, double dz,
                                        double k, double inv_norm, int perm) {
    const double two_pi = 6.283185307179586476925286766559;
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    int q = blockIdx.y;
    if (p >= Nx) return;
    const int Lc = Nx / perm;
    const int bin = perm * (p % Lc) + p / Lc;
    double kx = __ddiv_rn(__dmul_rn(two_pi, (double)freq_index(bin, Nx)), __dmul_rn((double)Nx, dx));
    double ky = __ddiv_rn(__dmul_rn(two_pi, (double)freq_index(q, Ny)), __dmul_rn((double)Ny, dx));
    double s = __dsub_rn(__dsub_rn(__dmul_rn(k, k), __dmul_rn(kx, kx)), __dmul_rn(ky, ky));
    float2 h = make_float2(0.f, 0.f);
    if (s > 0.0) {
        double sn, cs;
        sincos(__dmul_rn(dz, sqrt(s)), &sn, &cs);
        h.x = (float)(cs * inv_norm);
        h.y = (float)(sn * inv_norm);
    }
    H[(size_t)q * Nx + p] = h;
}

// Emitter data prepared for the spectrum kernel: fractional positions in units of the
// field width (double, so that the phase ramp can be range-reduced exactly), phase, amplitude.
struct EmitterPrep { double ax, ay; float phase, amp; };

__global__ void emitter_prep_kernel(const float *__restrict__ pos, const float *__restrict__ phase,
                                    const float *__restrict__ amp, int M, int Nx, int Ny, double dx,
                                    EmitterPrep *__restrict__ out) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= M) return;
    double X = (double)pos[2 * e] + (double)(Nx / 2) * dx;
    double Y = (double)pos[2 * e + 1] + (double)(Ny / 2) * dx;
    EmitterPrep r;
    r.ax = X / ((double)Nx * dx);
    r.ay = Y / ((double)Ny * dx);
    r.phase = phase ? phase[e] : 0.f;
    r.amp = amp ? amp[e] : 1.f;
    out[e] = r;
}

// U0[q][p] = P * sum_e a_e exp(i (phi_e - kx X_e - ky Y_e))   (bb.h bb_multiplex_psf; readings A12-A14).
// kx X_e = 2 pi f_p (X_e / (Nx dx)): the product f_p * ax is reduced mod 1 in double, the
// remaining angle (|.| <= pi + |phi|) goes through single-precision sincos.
__global__ void multiplex_spectrum_kernel(float2 *__restrict__ U0, int Nx, int Ny, double dx, double kc2,
                                          const EmitterPrep *__restrict__ em, int M) {
    const double two_pi = 6.283185307179586476925286766559;
    extern __shared__ EmitterPrep sm_em[];
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    int q = blockIdx.y;
    int fp = freq_index(p < Nx ? p : 0, Nx), fq = freq_index(q, Ny);
    double kx = __ddiv_rn(__dmul_rn(two_pi, (double)fp), __dmul_rn((double)Nx, dx));
    double ky = __ddiv_rn(__dmul_rn(two_pi, (double)fq), __dmul_rn((double)Ny, dx));
    bool inside = (p < Nx) && (__dadd_rn(__dmul_rn(kx, kx), __dmul_rn(ky, ky)) <= kc2);
    float sr = 0.f, si = 0.f;
    // whole blocks outside the pupil skip the emitter loop
    if (__syncthreads_or(inside ? 1 : 0)) {
        for (int e0 = 0; e0 < M; e0 += blockDim.x) {
            int n = min((int)blockDim.x, M - e0);
            __syncthreads();
            if ((int)threadIdx.x < n) sm_em[threadIdx.x] = em[e0 + threadIdx.x];
            __syncthreads();
            if (inside) {
                for (int e = 0; e < n; ++e) {
                    double tt = (double)fp * sm_em[e].ax + (double)fq * sm_em[e].ay;
                    float r = (float)(tt - rint(tt));
                    float s, c;
                    sincosf(fmaf(-6.283185307179586f, r, sm_em[e].phase), &s, &c);
                    sr = fmaf(sm_em[e].amp, c, sr);
                    si = fmaf(sm_em[e].amp, s, si);
                }
            }
        }
    }
    if (p < Nx) U0[(size_t)q * Nx + p] = inside ? make_float2(sr, si) : make_float2(0.f, 0.f);
}

// Per-slice partial sums of dn in double: partial[j][blockIdx.x] (fixed summation order,
// so the result is reproducible).  Used by bb_nref_from_dn.
__global__ void slice_sum_kernel(const float *__restrict__ dn, size_t npx, double *__restrict__ partial) {
    __shared__ double sm[256];
    const float *p = dn + (size_t)blockIdx.y * npx;
    size_t chunk = (npx + gridDim.x - 1) / gridDim.x;
    size_t i0 = (size_t)blockIdx.x * chunk, i1 = i0 + chunk < npx ? i0 + chunk : npx;
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

}  // namespace bb
