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
// kx X_e = 2 pi f_p (X_e / (Nx dx)): the product f_p * ax is reduced mod 1 in double, the remaining
// angle (|.| <= pi + |phi|) goes through single-precision sincos.  Separable form:
// the phase ramp factorises,
//   a_e exp(i (phi_e - kx X_e - ky Y_e)) = [a_e exp(i (phi_e - kx X_e))] [exp(-i ky Y_e)] = EX[e][p] EY[e][q],
// so the sum over emitters is a complex matrix product over the bounding box of the pupil,
//   U0[q][p] = P[q][p] sum_e EY[e][q] EX[e][p]      (M x Wy)^T (M x Wx),
// instead of one sincos per (pixel, emitter).
// Bins f = i - Fx (i < Wx) along x, f = i - Fy (i < Wy) along y: [-F, F] clipped to [-N/2, N/2 - 1].
__global__ void emitter_axis_kernel(const EmitterPrep *__restrict__ em, int M, int Fx, int Wx, int Fy, int Wy,
                                    float2 *__restrict__ EX, float2 *__restrict__ EY) {
    const int e = blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= M) return;
    const EmitterPrep E = em[e];
    if (i < Wx) {
        const double tt = (double)(i - Fx) * E.ax;
        const float r = (float)(tt - rint(tt));
        float s, c;
        sincosf(fmaf(-6.283185307179586f, r, E.phase), &s, &c);
        EX[(size_t)e * Wx + i] = make_float2(E.amp * c, E.amp * s);
    }
    if (i < Wy) {
        const double tt = (double)(i - Fy) * E.ay;
        const float r = (float)(tt - rint(tt));
        float s, c;
        sincosf(-6.283185307179586f * r, &s, &c);
        EY[(size_t)e * Wy + i] = make_float2(c, s);
    }
}

// U0 over the pupil's bounding box: 32 x 32 outputs per CTA (256 threads, 2 x 2 each), emitters in
// chunks of 32 through shared memory.  U0 must have been zeroed (pixels outside the box stay zero).
__global__ void __launch_bounds__(256) multiplex_gemm_kernel(float2 *__restrict__ U0, int Nx, int Ny, double dx, double ki2, double kc2,
                                                             const float2 *__restrict__ EX, const float2 *__restrict__ EY,
                                                             int M, int Fx, int Wx, int Fy, int Wy) {
    const double two_pi = 6.283185307179586476925286766559;
    constexpr int TK = 32;
    __shared__ float2 sx[TK][32], sy[TK][32];
    const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;           // outputs (ty + 16 a, tx + 16 b), a, b < 2
    const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
    float2 acc[2][2] = {};
    for (int e0 = 0; e0 < M; e0 += TK) {
        __syncthreads();
        for (int l = threadIdx.x; l < TK * 32; l += 256) {
            const int k = l / 32, c = l % 32, e = e0 + k;
            sx[k][c] = (e < M && i0 + c < Wx) ? EX[(size_t)e * Wx + i0 + c] : make_float2(0.f, 0.f);
            sy[k][c] = (e < M && j0 + c < Wy) ? EY[(size_t)e * Wy + j0 + c] : make_float2(0.f, 0.f);
        }
        __syncthreads();
#pragma unroll 8
        for (int k = 0; k < TK; ++k) {
            const float2 x0 = sx[k][tx], x1 = sx[k][tx + 16], y0 = sy[k][ty], y1 = sy[k][ty + 16];
            acc[0][0].x = fmaf(y0.x, x0.x, fmaf(-y0.y, x0.y, acc[0][0].x)); acc[0][0].y = fmaf(y0.x, x0.y, fmaf(y0.y, x0.x, acc[0][0].y));
            acc[0][1].x = fmaf(y0.x, x1.x, fmaf(-y0.y, x1.y, acc[0][1].x)); acc[0][1].y = fmaf(y0.x, x1.y, fmaf(y0.y, x1.x, acc[0][1].y));
            acc[1][0].x = fmaf(y1.x, x0.x, fmaf(-y1.y, x0.y, acc[1][0].x)); acc[1][0].y = fmaf(y1.x, x0.y, fmaf(y1.y, x0.x, acc[1][0].y));
            acc[1][1].x = fmaf(y1.x, x1.x, fmaf(-y1.y, x1.y, acc[1][1].x)); acc[1][1].y = fmaf(y1.x, x1.y, fmaf(y1.y, x1.x, acc[1][1].y));
        }
    }
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const int j = j0 + ty + 16 * a, i = i0 + tx + 16 * b;
            if (j >= Wy || i >= Wx) continue;
            const int fq = j - Fy, fp = i - Fx;
            const double kx = __ddiv_rn(__dmul_rn(two_pi, (double)fp), __dmul_rn((double)Nx, dx));
            const double ky = __ddiv_rn(__dmul_rn(two_pi, (double)fq), __dmul_rn((double)Ny, dx));
            const double k2 = __dadd_rn(__dmul_rn(kx, kx), __dmul_rn(ky, ky));
            if (!(k2 <= kc2 && k2 >= ki2)) continue;                  // pupil: disk, or annulus (bb_multiplex_annular)
            const int p = fp >= 0 ? fp : fp + Nx, q = fq >= 0 ? fq : fq + Ny;
            U0[(size_t)q * Nx + p] = acc[a][b];
        }
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

// T x T windows around the emitters of every plane of a stack (bb_extract_tiles): out[e][z][ty][tx] =
// src[z][(cy - T/2 + ty) mod Ny][(cx - T/2 + tx) mod Nx], (cx, cy) = nearest pixel of emitter e; ELEM floats per pixel.
template <int ELEM>
__global__ void extract_tiles_kernel(const float *__restrict__ src, int Nx, int Ny, int Np, const float *__restrict__ pos,
                                     int M, double dx, int T, float *__restrict__ out) {
    const int e = blockIdx.z, z = blockIdx.y;
    const long long cx = (long long)floor(__ddiv_rn((double)pos[2 * e], dx) + 0.5) + Nx / 2;
    const long long cy = (long long)floor(__ddiv_rn((double)pos[2 * e + 1], dx) + 0.5) + Ny / 2;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < T * T; i += gridDim.x * blockDim.x) {
        const int ty = i / T, tx = i - ty * T;
        const long long x = ((cx - T / 2 + tx) % Nx + Nx) % Nx, y = ((cy - T / 2 + ty) % Ny + Ny) % Ny;
        const float *sp = src + (((size_t)z * Ny + y) * Nx + x) * ELEM;
        float *op = out + ((((size_t)e * Np + z) * T + ty) * T + tx) * ELEM;
#pragma unroll
        for (int c = 0; c < ELEM; ++c) op[c] = sp[c];
    }
}

// Waist profile of the cylindrical light sheet (bb_lightsheet): u[y][x] = exp(-y^2 / w0^2), y = (i - Ny/2) dx.
__global__ void gaussian_sheet_kernel(float2 *__restrict__ u, int Nx, int Ny, double dx, double w0) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x, yi = blockIdx.y;
    if (x >= Nx) return;
    const double y = (double)(yi - Ny / 2) * dx;
    u[(size_t)yi * Nx + x] = make_float2((float)exp(-(y * y) / (w0 * w0)), 0.f);
}

// Image formation (bb_image_formation), step 1: the emitter nearest to every pixel (periodic distance, lowest
// index on ties; double, no fused multiply-adds: the comparison is a decision).
__global__ void nearest_emitter_kernel(int Nx, int Ny, const float *__restrict__ pos, int M, double dx, int *__restrict__ owner) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (x >= Nx) return;
    const double px = __dmul_rn((double)(x - Nx / 2), dx), py = __dmul_rn((double)(y - Ny / 2), dx);
    const double Lx = __dmul_rn((double)Nx, dx), Ly = __dmul_rn((double)Ny, dx);
    int best = 0;
    double bd = 0.0;
    for (int e = 0; e < M; ++e) {
        double ddx = __dsub_rn(px, (double)pos[2 * e]), ddy = __dsub_rn(py, (double)pos[2 * e + 1]);
        ddx = __dsub_rn(ddx, __dmul_rn(Lx, floor(__dadd_rn(__ddiv_rn(ddx, Lx), 0.5))));
        ddy = __dsub_rn(ddy, __dmul_rn(Ly, floor(__dadd_rn(__ddiv_rn(ddy, Ly), 0.5))));
        const double d2 = __dadd_rn(__dmul_rn(ddx, ddx), __dmul_rn(ddy, ddy));
        if (e == 0 || d2 < bd) { bd = d2; best = e; }
    }
    owner[(size_t)y * Nx + x] = best;
}

// Step 2: image[r] = sum over the T x T taps t of S[r - (t - T/2)] psf[owner[r - (t - T/2)]][t] (periodic).
// A CTA computes a 32 x 8 patch; the (32 + T - 1) x (8 + T - 1) halo of S and owner sits in shared memory.
__global__ void __launch_bounds__(256) image_formation_kernel(const float *__restrict__ S, const int *__restrict__ owner, int Nx, int Ny,
                                                              const float *__restrict__ psf, int T, float *__restrict__ image) {
    extern __shared__ float sm_if[];
    const int HW = 32 + T - 1, HH = 8 + T - 1;
    float *sS = sm_if;
    int *sO = reinterpret_cast<int *>(sm_if + HW * HH);
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 8;
    // halo origin: source pixel r' = r - (t - T/2) ranges over [r - (T - 1 - T/2), r + T/2]
    const int hx0 = x0 - (T - 1 - T / 2), hy0 = y0 - (T - 1 - T / 2);
    for (int i = threadIdx.x; i < HW * HH; i += 256) {
        const int hy = i / HW, hx = i - hy * HW;
        const int sx = ((hx0 + hx) % Nx + Nx) % Nx, sy = ((hy0 + hy) % Ny + Ny) % Ny;
        sS[i] = S[(size_t)sy * Nx + sx];
        sO[i] = owner[(size_t)sy * Nx + sx];
    }
    __syncthreads();
    const int lx = threadIdx.x % 32, ly = threadIdx.x / 32;
    const int x = x0 + lx, y = y0 + ly;
    if (x >= Nx || y >= Ny) return;
    float acc = 0.f;
    for (int ty = 0; ty < T; ++ty)
        for (int tx = 0; tx < T; ++tx) {
            // r' = r - (t - T/2)  ->  halo index r' - h0 = l + (T - 1 - T/2) - (t - T/2) = l + T - 1 - t
            const int hi = (ly + T - 1 - ty) * HW + (lx + T - 1 - tx);
            acc = fmaf(sS[hi], __ldg(psf + ((size_t)sO[hi] * T + ty) * T + tx), acc);
        }
    image[(size_t)y * Nx + x] = acc;
}

}  // namespace bb
